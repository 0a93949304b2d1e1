"""Event-by-event helicity and colour selection and running alpha_s -- ORACLE SIDE (test infrastructure, not product).

The paper's ME engine "also receives other inputs, such as: an event-by-event running coupling alpha_s ...; two
event-by-event random numbers for the selection of one specific helicity and leading color in the generated event (which
are also returned as outputs)", and Table 1 has the line "Randomly select a color and a helicity for event
ievt / selcol[ievt] = ...; selhel[ievt] = ... // extra output (from extra input random numbers)".  The
paper prints no formula for the selection; reading A15 fixes it the way event generators unweight a discrete
choice: inverse-CDF sampling with the contributions as weights, written out plainly here:

    helicity: weights me_h (the per-helicity, colour-summed contribution) over the good helicities in increasing h;
    colour:   weights w_sigma = sum_{good h} |A_h(sigma)|^2 over the colour flows sigma in lexicographic order
              (A_h(sigma) = the colour-ordered partial amplitudes of the Berends-Giele recursion, oracle/me_oracle.c);
    choice:   the first index k with  rnd * sum_j w_j < sum_{j <= k} w_j   (rnd in [0, 1)).

Running alpha_s: the matrix element is simply evaluated with that event's alpha_s (gs = sqrt(4 pi alpha_s)).
Pure Python loops over events and helicities: for small samples only.
"""
from __future__ import annotations

import math

import numpy as np

from . import me_oracle


def inverse_cdf(weights, rnd):
    """first k with rnd * sum(w) < w_0 + ... + w_k (the last index if rounding leaves none)"""
    total = 0.0
    for w in weights:
        total += w
    target = rnd * total
    cum = 0.0
    for k, w in enumerate(weights):
        cum += w
        if target < cum:
            return k
    return len(weights) - 1


def good_helicities(mh):
    """reading A5: h good iff max over the events of me_h / sum_h' me_h' > 1e-8"""
    frac = mh / mh.sum(axis=1, keepdims=True)
    return np.nonzero(frac.max(axis=0) > 1e-8)[0]


def color_weights(process, mom, params, good):
    """w[e][sigma] = sum over the good helicities of |A_h(sigma)|^2"""
    n = me_oracle.NGLUONS[process]
    npar = n + 2
    gs = math.sqrt(4.0 * math.pi * params["aS"])
    w = np.zeros((mom.shape[0], math.factorial(n)))
    for e in range(mom.shape[0]):
        for h in good:
            hel = [1 if (h >> (npar - 1 - i)) & 1 else -1 for i in range(npar)]
            A = me_oracle.partial_amplitudes(n, mom[e], hel, params["mT"], params["wT"], gs)
            w[e] += (A * A.conj()).real
    return w


def select(process, mom, params, rndhel, rndcol, alphas=None, good=None):
    """(me[nevt], selhel[nevt], selcol[nevt]) for the events `mom` [nevt][npar][4]; alphas[nevt] optional running alpha_s;
    good = the good-helicity list (default: derived from these very events, reading A5)"""
    nevt = mom.shape[0]
    me = np.zeros(nevt)
    mh = None
    if alphas is None:
        me, mh = me_oracle.matrix_elements(process, mom, params, per_helicity=True)
    else:
        mh = np.zeros((nevt, 1 << mom.shape[1]))
        for e in range(nevt):
            pe = dict(params, aS=float(alphas[e]))
            m1, h1 = me_oracle.matrix_elements(process, mom[e:e + 1], pe, per_helicity=True)
            me[e], mh[e] = m1[0], h1[0]
    if good is None:
        good = good_helicities(mh)
    selhel = np.array([good[inverse_cdf(mh[e][good], rndhel[e])] for e in range(nevt)], dtype=np.int32)
    if process == "epem_mupmum":
        selcol = np.zeros(nevt, dtype=np.int32)            # one colour flow
    else:
        w = color_weights(process, mom, params, good)      # the common factor alpha_s^n drops out of the choice
        selcol = np.array([inverse_cdf(w[e], rndcol[e]) for e in range(nevt)], dtype=np.int32)
    return me, selhel, selcol
