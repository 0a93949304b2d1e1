"""Feynman-diagram enumeration for g g -> t tbar + (n-2) g and its lowering to a HELAS-style program.

The paper's diagrams come from the MG5aMC code generator, which is not available
here; this module enumerates them from the QCD Feynman rules instead and reproduces Table 2 row 2
(PAPER.md:182): 3 / 16 / 123 / 1240 diagrams, a four-gluon vertex counting as ONE diagram.

A diagram is an ordered list of pure-gluon trees hanging off the quark line (top side first).  Each one
is turned into an unrooted tree graph, cut at its centroid vertex -- so that no branch holds more than
half of the external legs -- and evaluated the way the paper describes: wavefunctions of
external particles, wavefunctions of internal propagators (off-shell currents, shared between diagrams),
one amplitude per diagram term, `jamp[c] += coeff * amp`.  A four-gluon vertex expands into its three
colour/Lorentz terms (HELAS VVVV1/3/4).

Program (IR) produced by `build_process`:
  currents : list of Current(id, kind, op, args, legs, col)      kind in {'V','FO','FI'}
  amps     : list of Amp(op, args, jamps=[(colour index, integer coeff)], diagram)
Ops and their Lorentz meaning are defined in csrc/helas.cuh (device) and restated independently in
tests/ir_eval.py (numpy, CPU tests only).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from functools import lru_cache
from itertools import combinations, permutations

from . import colour as col

# ------------------------------------------------------------------------------------------------
# pure-gluon trees over a set of gluon labels: ('g', i) | ('v3', A, B) | ('v4', A, B, C)


def _partitions2(items):
    items = list(items)
    first, rest = items[0], items[1:]
    for r in range(0, len(rest)):
        for sub in combinations(rest, r):
            s1 = (first,) + sub
            s2 = tuple(x for x in rest if x not in sub)
            if s2:
                yield s1, s2


def _partitions3(items):
    items = list(items)
    first, rest = items[0], items[1:]
    for r in range(0, len(rest) - 1):
        for sub in combinations(rest, r):
            s1 = (first,) + sub
            rem = [x for x in rest if x not in sub]
            for s2, s3 in _partitions2(rem):
                yield s1, s2, s3


@lru_cache(maxsize=None)
def gluon_trees(leaves):
    """all off-shell gluon trees with the given (sorted tuple of) leaves"""
    if len(leaves) == 1:
        return (("g", leaves[0]),)
    out = []
    for s1, s2 in _partitions2(leaves):
        for a in gluon_trees(s1):
            for b in gluon_trees(s2):
                out.append(("v3", a, b))
    if len(leaves) >= 3:
        for s1, s2, s3 in _partitions3(leaves):
            for a in gluon_trees(s1):
                for b in gluon_trees(s2):
                    for c in gluon_trees(s3):
                        out.append(("v4", a, b, c))
    return tuple(out)


def _ordered_set_partitions(items):
    """ordered sequences of disjoint non-empty blocks covering items"""
    items = tuple(items)
    if not items:
        yield ()
        return
    n = len(items)
    for r in range(1, n + 1):
        for first in combinations(items, r):
            rest = tuple(x for x in items if x not in first)
            for tail in _ordered_set_partitions(rest):
                yield (first,) + tail


def enumerate_diagrams(n):
    """every tree diagram of q qbar + n gluons: a tuple of gluon trees along the quark line (top first)"""
    out = []
    for blocks in _ordered_set_partitions(range(n)):
        def rec(i, acc):
            if i == len(blocks):
                out.append(tuple(acc))
                return
            for t in gluon_trees(blocks[i]):
                rec(i + 1, acc + [t])
        rec(0, [])
    return out


# ------------------------------------------------------------------------------------------------
@dataclass
class Current:
    id: int
    kind: str            # 'V' vector (4 complex), 'FO' row spinor (ubar side), 'FI' column spinor (v side)
    op: str
    args: tuple          # ids of input currents (and small integers for op variants)
    legs: frozenset      # external particles contained
    col: dict = field(repr=False, default=None)
    level: int = 0


@dataclass
class Amp:
    op: str
    args: tuple
    jamps: list          # [(colour index, integer coefficient)]
    diagram: int


class Process:
    """IR of one g g -> t tbar + (n-2) g process"""

    def __init__(self, n):
        self.n = n
        self.npar = n + 2
        self.name = "gg_ttx" + "g" * (n - 2)
        self.currents: list[Current] = []
        self.amps: list[Amp] = []
        self._memo = {}
        self.ndiagrams = 0
        self.rank = col.perm_rank_table(n)
        self.ncolor = len(self.rank)

    # particle index of gluon label g; all-incoming momentum sign of a particle
    @staticmethod
    def particle_of_gluon(g):
        return g if g < 2 else g + 2

    @staticmethod
    def momentum_sign(ip):
        return 1 if ip < 2 else -1

    def _new(self, kind, op, args, legs, colr):
        key = (op, args)
        if key in self._memo:
            return self._memo[key]
        ids = self._arg_ids(op, args)
        lvl = 1 + max((self.currents[i].level for i in ids), default=-1)
        c = Current(len(self.currents), kind, op, args, frozenset(legs), colr, lvl)
        self.currents.append(c)
        self._memo[key] = c
        return c

    @staticmethod
    def _arg_ids(op, args):
        if op in ("ext_v", "ext_ql", "ext_qr"):
            return ()
        return tuple(args)

    # --- constructors (operands sorted into a canonical order; colour follows the same order) ---
    def ext_v(self, g):
        ip = self.particle_of_gluon(g)
        return self._new("V", "ext_v", (ip,), {ip}, {(g,): 1})

    def ext_ql(self):
        return self._new("FO", "ext_ql", (), {2}, {(): 1})

    def ext_qr(self):
        return self._new("FI", "ext_qr", (), {3}, {(): 1})

    def v3(self, a, b):
        if a.id > b.id:
            a, b = b, a
        return self._new("V", "v3", (a.id, b.id), a.legs | b.legs, col.c3(a.col, b.col))

    def v4(self, x, y, z):
        """term of the four-gluon vertex in which z is paired with the off-shell leg: (x y | z out)"""
        if x.id > y.id:
            x, y = y, x
        return self._new("V", "v4", (x.id, y.id, z.id), x.legs | y.legs | z.legs,
                         col.c3(col.c3(x.col, y.col), z.col))

    def ffv_l(self, ql, g):
        return self._new("FO", "ffv_l", (ql.id, g.id), ql.legs | g.legs, col.concat(ql.col, g.col))

    def ffv_r(self, g, qr):
        return self._new("FI", "ffv_r", (g.id, qr.id), g.legs | qr.legs, col.concat(g.col, qr.col))

    def ffv_p(self, ql, qr):
        return self._new("V", "ffv_p", (ql.id, qr.id), ql.legs | qr.legs,
                         col.concat(ql.col, col.STAR_POLY, qr.col))

    # --- amplitudes ---
    def _add_amp(self, op, args, colr, diagram):
        jl = []
        for w, c in sorted(colr.items()):
            assert col.STAR not in w and len(w) == self.n, (op, w)
            jl.append((self.rank[w], c))
        self.amps.append(Amp(op, tuple(args), jl, diagram))

    def amp_ffv(self, ql, g, qr, d):
        self._add_amp("ffv", (ql.id, g.id, qr.id), col.concat(ql.col, g.col, qr.col), d)

    def amp_vvv(self, a, b, c, d):
        # sort by id; an odd permutation flips both the Lorentz value (totally antisymmetric vertex
        # function) and the colour computed from the same order, so no sign needs tracking
        a, b, c = sorted((a, b, c), key=lambda x: x.id)
        self._add_amp("vvv", (a.id, b.id, c.id), col.c3amp(a.col, b.col, c.col), d)

    def amp_vvvv(self, legs4, d):
        a, b, c, e = sorted(legs4, key=lambda x: x.id)
        # three pairings (x y | z w): Lorentz (X.Z)(Y.W) - (X.W)(Y.Z), colour f^{xye} f^{zwe}
        for (x, y, z, w) in ((a, b, c, e), (a, c, b, e), (a, e, b, c)):
            h = col.c3(x.col, y.col)
            self._add_amp("vvvv", (x.id, y.id, z.id, w.id), col.c3amp(z.col, w.col, h), d)


# ------------------------------------------------------------------------------------------------
# unrooted tree graph of one diagram
class _Graph:
    def __init__(self):
        self.kind = []      # per node: ('ext', ip) | ('qqg',) | ('ggg',) | ('gggg',)
        self.adj = []       # per node: ordered neighbour list (qqg: [L, G, R]; ggg: cyclic; gggg: any)

    def add(self, kind):
        self.kind.append(kind)
        self.adj.append([])
        return len(self.kind) - 1


def _diagram_graph(proc, diagram):
    g = _Graph()
    top = g.add(("ext", 2))
    atop = g.add(("ext", 3))

    def tree(t, parent):
        if t[0] == "g":
            v = g.add(("ext", proc.particle_of_gluon(t[1])))
            g.adj[v] = [parent]
            return v
        v = g.add(("ggg",) if t[0] == "v3" else ("gggg",))
        g.adj[v] = [None] * (len(t) - 1) + [parent]
        for i, sub in enumerate(t[1:]):
            g.adj[v][i] = tree(sub, v)
        return v

    prev = top
    qv = []
    for t in diagram:
        v = g.add(("qqg",))
        g.adj[v] = [prev, None, None]
        if g.kind[prev][0] == "ext":
            g.adj[prev] = [v]
        else:
            g.adj[prev][2] = v
        g.adj[v][1] = tree(t, v)
        qv.append(v)
        prev = v
    g.adj[prev][2] = atop
    g.adj[atop] = [prev]
    return g


def _branch_sizes(g):
    """number of external legs in the branch seen from node u through neighbour w"""
    memo = {}

    def size(u, frm):           # legs in the subtree of u when entered from frm
        key = (u, frm)
        if key in memo:
            return memo[key]
        if g.kind[u][0] == "ext":
            r = 1
        else:
            r = sum(size(w, u) for w in g.adj[u] if w != frm)
        memo[key] = r
        return r
    return size


def _lower_diagram(proc, diagram, dindex, prefer):
    g = _diagram_graph(proc, diagram)
    size = _branch_sizes(g)
    best = None

    def legs_of(u, frm):
        if g.kind[u][0] == "ext":
            return {g.kind[u][1]}
        out = set()
        for w in g.adj[u]:
            if w != frm:
                out |= legs_of(w, u)
        return out

    for u in range(len(g.kind)):
        if g.kind[u][0] == "ext":
            continue
        worst = max(size(w, u) for w in g.adj[u])
        # 8 external legs: a propagator can split them 4 | 4 and both of its end vertices are centroids.  Take the end on
        # the top quark's side, whatever the vertices are: the set of diagrams cut at (vertex, leg sets) is then the full
        # product of the sub-diagrams of its branches, which the colour factorisation of gen/co_program.py needs.  (With
        # 6 legs the 3 | 3 tie is left to `prefer`, as the committed tables of g g -> t tbar g g were built.)
        tie = 0
        if proc.npar >= 8 and 2 * worst == proc.npar:
            big = next(w for w in g.adj[u] if size(w, u) == worst)
            tie = 1 if 2 in legs_of(big, u) else 0
        score = (worst, tie, prefer.get(g.kind[u][0], 0), u)
        if best is None or score < best[0]:
            best = (score, u)
    centre = best[1]

    def cur(u, frm):
        """list of alternative term-currents flowing out of u towards frm"""
        k = g.kind[u]
        if k[0] == "ext":
            ip = k[1]
            if ip == 2:
                return [proc.ext_ql()]
            if ip == 3:
                return [proc.ext_qr()]
            return [proc.ext_v(ip if ip < 2 else ip - 2)]
        nb = g.adj[u]
        if k[0] == "qqg":
            L, G, R = nb
            out = []
            if frm == R:
                for a in cur(L, u):
                    for b in cur(G, u):
                        out.append(proc.ffv_l(a, b))
            elif frm == L:
                for a in cur(G, u):
                    for b in cur(R, u):
                        out.append(proc.ffv_r(a, b))
            else:
                for a in cur(L, u):
                    for b in cur(R, u):
                        out.append(proc.ffv_p(a, b))
            return out
        if k[0] == "ggg":
            i = nb.index(frm)
            e1, e2 = nb[(i + 1) % 3], nb[(i + 2) % 3]
            return [proc.v3(a, b) for a in cur(e1, u) for b in cur(e2, u)]
        # gggg
        others = [w for w in nb if w != frm]
        out = []
        for a in cur(others[0], u):
            for b in cur(others[1], u):
                for c in cur(others[2], u):
                    out.append(proc.v4(a, b, c))
                    out.append(proc.v4(a, c, b))
                    out.append(proc.v4(b, c, a))
        return out

    k = g.kind[centre]
    nb = g.adj[centre]
    if k[0] == "qqg":
        for a in cur(nb[0], centre):
            for b in cur(nb[1], centre):
                for c in cur(nb[2], centre):
                    proc.amp_ffv(a, b, c, dindex)
    elif k[0] == "ggg":
        for a in cur(nb[0], centre):
            for b in cur(nb[1], centre):
                for c in cur(nb[2], centre):
                    proc.amp_vvv(a, b, c, dindex)
    else:
        for a in cur(nb[0], centre):
            for b in cur(nb[1], centre):
                for c in cur(nb[2], centre):
                    for e in cur(nb[3], centre):
                        proc.amp_vvvv((a, b, c, e), dindex)


@lru_cache(maxsize=None)
def build_process(n, prefer_qqg=True):
    proc = Process(n)
    # externals first, in particle order, so that their ids are stable
    proc.ext_v(0)
    proc.ext_v(1)
    proc.ext_ql()
    proc.ext_qr()
    for gl in range(2, n):
        proc.ext_v(gl)
    diagrams = enumerate_diagrams(n)
    proc.ndiagrams = len(diagrams)
    prefer = {"qqg": 0, "ggg": 1, "gggg": 2} if prefer_qqg else {"qqg": 2, "ggg": 1, "gggg": 0}
    for di, d in enumerate(diagrams):
        _lower_diagram(proc, d, di, prefer)
    return proc


def summary(proc):
    from collections import Counter
    ops = Counter(c.op for c in proc.currents)
    aops = Counter(a.op for a in proc.amps)
    return {
        "name": proc.name, "ndiagrams": proc.ndiagrams, "ncolor": proc.ncolor,
        "ncurrents": len(proc.currents), "current_ops": dict(ops),
        "namps": len(proc.amps), "amp_ops": dict(aops),
        "jamp_updates": sum(len(a.jamps) for a in proc.amps),
        "max_legs": max(len(c.legs) for c in proc.currents),
    }
