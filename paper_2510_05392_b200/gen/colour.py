"""Exact colour algebra for one quark line + n gluons (build-time only, pure Python integers/Fractions).

Colour factors are polynomials in words over the gluon labels 0..n-1: a word (a, b, c) stands for the
string (T^a T^b T^c)_{i jbar}, first generator next to the top quark.  The n! full-length words are the
leading colour flows of PAPER.md:124, 241 ("dual amplitudes for a given color flow (jamps)", Table 2
row 4: 2/6/24/120), indexed by the lexicographic rank of the permutation.

A gluon-type current that contains the quark line carries words with one hole STAR: the place where the
generator T^c of its open adjoint index c sits.

Every structure constant is rewritten with  f^{abc} T^c = -i [T^a, T^b]  (cyclic in abc).  The factors of
-i, i and g are the same for every diagram of a process ("Phases"), so only the bare
commutators are kept here: `c3(P1, P2)` is the colour of the third leg of f^{123}.
"""
from __future__ import annotations

from fractions import Fraction
from functools import lru_cache
from itertools import permutations

STAR = -1


def poly_add(p, q, sign=1):
    out = dict(p)
    for w, c in q.items():
        v = out.get(w, 0) + sign * c
        if v:
            out[w] = v
        else:
            out.pop(w, None)
    return out


def poly_scale(p, s):
    return {w: c * s for w, c in p.items()} if s else {}


def concat(*polys):
    out = {(): 1}
    for p in polys:
        nxt = {}
        for w1, c1 in out.items():
            for w2, c2 in p.items():
                w = w1 + w2
                v = nxt.get(w, 0) + c1 * c2
                if v:
                    nxt[w] = v
                else:
                    nxt.pop(w, None)
        out = nxt
    return out


def comm(p, q):
    return poly_add(concat(p, q), concat(q, p), -1)


def has_star(p):
    return any(STAR in w for w in p)


def subst(x, p):
    """replace the hole of every word of x by the polynomial p"""
    out = {}
    for w, c in x.items():
        i = w.index(STAR)
        for w2, c2 in p.items():
            ww = w[:i] + w2 + w[i + 1:]
            v = out.get(ww, 0) + c * c2
            if v:
                out[ww] = v
            else:
                out.pop(ww, None)
    return out


STAR_POLY = {(STAR,): 1}


def c3(p1, p2):
    """colour carried by leg 3 of f^{123} when legs 1, 2 carry p1, p2 (at most one of them holds the quark line)."""
    s1, s2 = has_star(p1), has_star(p2)
    assert not (s1 and s2)
    if s1:      # T^x f^{x2c} = f^{2cx} T^x  ->  [P2, T^c]
        return subst(p1, comm(p2, STAR_POLY))
    if s2:      # f^{1xc} T^x = f^{c1x} T^x  ->  [T^c, P1]
        return subst(p2, comm(STAR_POLY, p1))
    return comm(p1, p2)


def c3amp(p1, p2, p3):
    """colour of the closed vertex f^{123}; exactly one leg holds the quark line (has the hole)."""
    s = [has_star(p) for p in (p1, p2, p3)]
    assert sum(s) == 1
    if s[2]:
        return subst(p3, comm(p1, p2))
    if s[0]:
        return subst(p1, comm(p2, p3))
    return subst(p2, comm(p3, p1))


def perm_rank_table(n):
    return {p: i for i, p in enumerate(permutations(range(n)))}


# ------------------------------------------------------------------------------------------------
# colour matrix  C_{s s'} = sum_{colours} (T^{s1}..T^{sn})_{ij} conj((T^{s'1}..T^{s'n})_{ij})
#              = Tr(T^{s1} ... T^{sn} T^{s'n} ... T^{s'1})   summed over all adjoint indices,
# reduced exactly with the SU(N) Fierz identity  T^a_{ij} T^a_{kl} = 1/2 (d_il d_jk - d_ij d_kl / N).
NC = 3


@lru_cache(maxsize=None)
def _trace_product(traces):
    """sum over all repeated letters of a product of traces of words; `traces` = tuple of tuples."""
    traces = tuple(t for t in traces)
    # find a letter
    for ti, t in enumerate(traces):
        if len(t) == 0:
            continue
        a = t[0]
        rest = t[1:]
        others = traces[:ti] + traces[ti + 1:]
        if a in rest:
            j = rest.index(a)
            X, Y = rest[:j], rest[j + 1:]
            # Tr(a X a Y) = 1/2 Tr(X) Tr(Y) - 1/(2N) Tr(X Y)
            return (Fraction(1, 2) * _trace_product(_canon(others + (X, Y)))
                    - Fraction(1, 2 * NC) * _trace_product(_canon(others + (X + Y,))))
        for tj, u in enumerate(others):
            if a in u:
                k = u.index(a)
                U = u[k + 1:] + u[:k]            # rotate so that u = (a, U)
                oth2 = others[:tj] + others[tj + 1:]
                # Tr(a X) Tr(a U) = 1/2 Tr(X U) - 1/(2N) Tr(X) Tr(U)
                return (Fraction(1, 2) * _trace_product(_canon(oth2 + (rest + U,)))
                        - Fraction(1, 2 * NC) * _trace_product(_canon(oth2 + (rest, U))))
        raise AssertionError("unpaired colour index")
    # only empty traces left: Tr(1) = N each
    return Fraction(NC) ** len(traces)


def _canon(traces):
    """canonical form of a product of cyclic words (rotate each to its minimum, sort)."""
    out = []
    for t in traces:
        if len(t) > 1:
            m = min(range(len(t)), key=lambda i: t[i:] + t[:i])
            t = t[m:] + t[:m]
        out.append(t)
    return tuple(sorted(out))


def colour_matrix(n):
    """exact C as a list of lists of Fractions, permutations in lexicographic order."""
    perms = list(permutations(range(n)))
    idx = {p: i for i, p in enumerate(perms)}
    # C depends only on the relative permutation: C[s][s'] = c(s^-1 o s')
    base = perms[0]
    row = []
    for sp in perms:
        word = base + tuple(reversed(sp))
        row.append(_trace_product(_canon((word,))))
    C = [[None] * len(perms) for _ in perms]
    for s in perms:
        inv = [0] * n
        for pos, g in enumerate(s):
            inv[g] = pos
        for sp in perms:
            rel = tuple(inv[g] for g in sp)     # relabel gluons so that s becomes the identity
            C[idx[s]][idx[sp]] = row[idx[rel]]
    return C


def common_denominator(C):
    from math import lcm
    d = 1
    for r in C:
        for x in r:
            d = lcm(d, x.denominator)
    return d
