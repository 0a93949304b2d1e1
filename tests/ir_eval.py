"""numpy evaluator of the generator's diagram program (IR) -- CPU TEST HELPER, not product, not oracle.

It restates what each IR op means with plain 4x4 chiral-representation gamma matrices, so that the
host-side generator (diagram enumeration, centroid lowering, colour polynomials) can be checked against
the oracle on CPU, before any kernel runs.  The CUDA kernels implement the same ops in
paper_2510_05392_b200/csrc/helas.cuh; nothing here is imported by the package.
"""
import math

import numpy as np

_s0 = np.eye(2, dtype=complex)
_sig = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], dtype=complex)]
_Z2 = np.zeros((2, 2), dtype=complex)
GAM = [np.block([[_Z2, _s0], [_s0, _Z2]])] + [np.block([[_Z2, s], [-s, _Z2]]) for s in _sig]
G = np.array([1.0, -1.0, -1.0, -1.0])


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def slash(a):
    return a[0] * GAM[0] - a[1] * GAM[1] - a[2] * GAM[2] - a[3] * GAM[3]


def chi(p, lam):
    pp = math.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    if pp + p[3] <= 1e-14 * pp:
        return np.array([0, 1], dtype=complex) if lam > 0 else np.array([-1, 0], dtype=complex)
    nrm = 1 / math.sqrt(2 * pp * (pp + p[3]))
    if lam > 0:
        return np.array([pp + p[3], p[1] + 1j * p[2]]) * nrm
    return np.array([-p[1] + 1j * p[2], pp + p[3]]) * nrm


def _roots(p, m):
    pp = math.sqrt(p[1] ** 2 + p[2] ** 2 + p[3] ** 2)
    sp = math.sqrt(p[0] + pp)
    sm = m / sp if m > 0 else 0.0          # sqrt(E - |p|) = m / sqrt(E + |p|)
    return sp, sm


def u_spinor(p, m, lam):
    """u(p, lam) = (sqrt(E - lam|p|) chi_lam, sqrt(E + lam|p|) chi_lam) in the chiral representation"""
    sp, sm = _roots(p, m)
    x = chi(p, lam)
    return np.concatenate([sm * x, sp * x]) if lam > 0 else np.concatenate([sp * x, sm * x])


def v_spinor(p, m, lam):
    """v(p, lam) = (sqrt(E + lam|p|) chi_{-lam}, -sqrt(E - lam|p|) chi_{-lam}), lam = physical helicity"""
    sp, sm = _roots(p, m)
    x = chi(p, -lam)
    return np.concatenate([sp * x, -sm * x]) if lam > 0 else np.concatenate([sm * x, -sp * x])


def polvec(p, lam):
    pt = math.hypot(p[1], p[2])
    pp = math.sqrt(pt * pt + p[3] ** 2)
    if pt > 1e-14 * pp:
        ct, st, cf, sf = p[3] / pp, pt / pp, p[1] / pt, p[2] / pt
    else:
        ct, st, cf, sf = (1.0 if p[3] > 0 else -1.0), 0.0, 1.0, 0.0
    e1 = np.array([ct * cf, ct * sf, -st])
    e2 = np.array([-sf, cf, 0.0])
    return np.concatenate([[0.0], (-lam * e1 - 1j * e2) / math.sqrt(2)])


def evaluate(proc, mom, hel, mt, wt):
    """jamps [ncolor] (without the g^n factor) for one event mom[npar][4] and helicities hel[npar] (+-1)"""
    npar = proc.npar
    k = [mom[i] * (1 if i < 2 else -1) for i in range(npar)]

    def K(legs):
        return sum(k[i] for i in legs)

    w = [None] * len(proc.currents)
    for c in proc.currents:
        a = c.args
        if c.op == "ext_v":
            ip = a[0]
            e = polvec(mom[ip], hel[ip])
            w[c.id] = e if ip < 2 else e.conj()
        elif c.op == "ext_ql":
            u = u_spinor(mom[2], mt, hel[2])
            w[c.id] = u.conj() @ GAM[0]
        elif c.op == "ext_qr":
            w[c.id] = v_spinor(mom[3], mt, hel[3])
        elif c.op == "v3":
            A, B = w[a[0]], w[a[1]]
            kA, kB = K(proc.currents[a[0]].legs), K(proc.currents[a[1]].legs)
            Kt = kA + kB
            w[c.id] = (mdot(A, B) * (kA - kB) + mdot(2 * kB + kA, A) * B - mdot(2 * kA + kB, B) * A) / mdot(Kt, Kt)
        elif c.op == "v4":
            X, Y, Z = w[a[0]], w[a[1]], w[a[2]]
            Kt = K(c.legs)
            w[c.id] = (mdot(X, Z) * Y - mdot(Y, Z) * X) / mdot(Kt, Kt)
        elif c.op == "ffv_l":
            q = -K(c.legs)
            w[c.id] = w[a[0]] @ slash(w[a[1]]) @ (slash(q) + mt * np.eye(4)) / (mdot(q, q) - mt * mt + 1j * mt * wt)
        elif c.op == "ffv_r":
            q = K(c.legs)
            w[c.id] = (slash(q) + mt * np.eye(4)) @ slash(w[a[0]]) @ w[a[1]] / (mdot(q, q) - mt * mt + 1j * mt * wt)
        elif c.op == "ffv_p":
            Kt = K(c.legs)
            w[c.id] = np.array([w[a[0]] @ GAM[mu] @ w[a[1]] for mu in range(4)]) / mdot(Kt, Kt)
        else:
            raise ValueError(c.op)
    jamp = np.zeros(proc.ncolor, dtype=complex)
    for am in proc.amps:
        a = am.args
        if am.op == "ffv":
            val = w[a[0]] @ slash(w[a[1]]) @ w[a[2]]
        elif am.op == "vvv":
            A, B, C = w[a[0]], w[a[1]], w[a[2]]
            kA, kB, kC = (K(proc.currents[i].legs) for i in a)
            val = mdot(A, B) * mdot(kA - kB, C) + mdot(B, C) * mdot(kB - kC, A) + mdot(C, A) * mdot(kC - kA, B)
        elif am.op == "vvvv":
            X, Y, Z, W = (w[i] for i in a)
            val = mdot(X, Z) * mdot(Y, W) - mdot(X, W) * mdot(Y, Z)
        else:
            raise ValueError(am.op)
        for ci, coef in am.jamps:
            jamp[ci] += coef * val
    return jamp


def matrix_element(proc, C, denom, mom, mt, wt, gs, per_helicity=False):
    npar = proc.npar
    tot = 0.0
    mh = np.zeros(1 << npar)
    for h in range(1 << npar):
        hel = [1 if (h >> (npar - 1 - i)) & 1 else -1 for i in range(npar)]
        j = evaluate(proc, mom, hel, mt, wt)
        mh[h] = (j.conj() @ C @ j).real * gs ** (2 * proc.n) / denom
        tot += mh[h]
    return (tot, mh) if per_helicity else tot
