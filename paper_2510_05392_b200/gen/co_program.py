"""Helicity-shared program ("hs") of a g g -> t tbar + (n-2) g process: tables for csrc/hs_kernel.cu.

Starting point: the diagram program of gen/diagrams.py -- every Feynman diagram explicitly enumerated
(Table 2), cut at its centroid vertex into <= 4 off-shell currents with <= half of the
external legs each, one amplitude per diagram term, `jamp[sigma] += coeff * amp`.

Two exact rewritings of that sum (neither changes what is computed):

  (1) helicity sharing.  A current with legs L depends on the helicities of L only, so it has 2^|L| <= 8
      distinct values ("variants") per event, not ncomb = 2^npar.  They are computed once per event and
      kept in shared memory; the thread of helicity combination h reads variant pext(h, L).

  (2) factorised colour.  Within the amplitudes that share (vertex type, leg sets of the branches), the
      coefficient of flow sigma is a product of the branches' own colour polynomials evaluated on the
      sub-words of sigma (gen/colour.py: concat / commutator substitution), times a sign that depends on
      (sigma, leg sets) only.  The vertex functions are multilinear, hence
          sum_d coeff[sigma, d] * V(c1_d, c2_d, c3_d) = s * V(O1, O2, O3),   O_i = sum_c col_c[w_i(sigma)] c
      with O_i "colour-ordered objects": signed sums of the Feynman currents of one leg set.  The
      factorisation is verified term by term against the diagram program in `build` (`_check_expansion`).

  Every V(O1, O2, O3) is then split as X . Y with Y the branch with most legs (<= 3) and X = the vertex
  contracted with the other branches (a "pair object", 2^(npar-|Y|) variants, metric folded in), so that
  the per-helicity work of one jamp is a short sum of 4-component complex dot products and each jamp is
  complete when its loop ends -- no per-thread jamp array.

With 6 gluons a branch can hold 4 legs; such a colour-ordered object is itself factorised over the objects of its own
branches (`_factorised_terms`).  The program is lowered to device tables by gen/hs_streams.py (tuned kernel, <= 5 gluons)
and gen/hsg_tables.py (generic kernel).
"""
from __future__ import annotations

from collections import defaultdict
from dataclasses import dataclass, field

import numpy as np

from . import colour, diagrams

STAR = colour.STAR

# term opcodes (phase 1: currents with propagators; phase 2: raw vertices, output lowered for the plain dot)
OPS = {"ext_v": 0, "ext_ql": 1, "ext_qr": 2, "v3": 3, "v4": 4, "ffv_l": 5, "ffv_r": 6, "ffv_p": 7,
       "x_row": 8, "x_col": 9, "x_bil": 10, "x_v3": 11, "x_v4": 12, "x_v4s": 13}


def merge_v4_pairs(terms):
    """With x_v4(p, q, r) = (p.r) q - (q.r) p and S(m; a, b) = 2 (a.b) m - (m.b) a - (m.a) b =: x_v4s(a, m, b):
         x_v4(p, q, r) + x_v4(r, q, p) =  S(q; p, r)
         x_v4(p, q, r) - x_v4(q, r, p) =  S(q; p, r)
         x_v4(p, q, r) + x_v4(p, r, q) = -S(p; q, r)
    The two orderings of the four-gluon vertex that a colour-ordered amplitude takes together share their dot
    products: 3 dots + 12 complex multiply-adds instead of 4 + 16, and one pass over the arguments instead of two."""
    out, used = [], set()
    for i, t in enumerate(terms):
        if i in used:
            continue
        merged = None
        if t.op == "x_v4":
            p_, q_, r_ = t.args
            for j in range(i + 1, len(terms)):
                u = terms[j]
                if j in used or u.op != "x_v4":
                    continue
                if u.args == (r_, q_, p_) and u.sign == t.sign:
                    merged = Term(t.sign, "x_v4s", (p_, q_, r_), t.legs)
                elif u.args == (q_, r_, p_) and u.sign == -t.sign:
                    merged = Term(t.sign, "x_v4s", (p_, q_, r_), t.legs)
                elif u.args == (p_, r_, q_) and u.sign == t.sign:
                    merged = Term(-t.sign, "x_v4s", (q_, p_, r_), t.legs)
                if merged is not None:
                    used.add(j)
                    break
        out.append(merged if merged is not None else t)
    return out


def acc_swizzle(h):
    """index of helicity combination h in the per-warp jamp accumulator of csrc/hs_kernel.cu (phase 3): a GF(2)-linear
    map that XORs the bank-group bits (h & 7) with distinct non-zero 3-bit codes of the higher bits, so that the 8
    lanes of a quarter-warp (3 varying helicity bits) mostly hit 8 different 16-byte bank groups"""
    hi = h >> 3
    t = ((hi & 1) * 3) ^ (((hi >> 1) & 1) * 5) ^ (((hi >> 2) & 1) * 6) ^ (((hi >> 3) & 1) * 7)
    return h ^ t


@dataclass
class Term:
    sign: int
    op: str
    args: tuple            # object ids (ext ops: (particle,))
    legs: tuple            # legs of the result (sorted particles)


@dataclass
class Obj:
    id: int
    kind: str              # 'V' | 'FO' | 'FI'
    legs: tuple            # sorted particle indices
    terms: list = field(default_factory=list)
    off: int = 0           # offset in the object area, units of one complex number


def _gluons(legs):
    return frozenset((ip if ip < 2 else ip - 2) for ip in legs if ip not in (2, 3))


def _key_word(c, sigma):
    """sub-word of the colour flow sigma seen by current c (with the hole for a gluon-type current that
    contains the quark line)"""
    own = _gluons(c.legs)
    if c.kind == "V" and 2 in c.legs:
        w, done = [], False
        for g in sigma:
            if g in own:
                w.append(g)
            elif not done:
                w.append(STAR)
                done = True
        return tuple(w)
    return tuple(g for g in sigma if g in own)


class Program:
    def __init__(self, n, group_prefix=None):
        """group_prefix: number of leading letters of sigma shared by a group of colour flows, or "file": the partition
        of gen/flow_groups_n<n>.txt (gen/regroup.py)"""
        self.n = n
        self.proc = diagrams.build_process(n)
        self.npar = n + 2
        self.name = self.proc.name
        self.ncolor = self.proc.ncolor
        self.group_prefix = group_prefix if group_prefix is not None else max(0, n - 2)
        self.objs: list[Obj] = []
        self._fobj = {}          # Feynman current id -> object id (levels 1, 2)
        self._combo = {}         # canonical combination -> object id
        self._build_objects()
        self._build_evals()
        self._check_expansion()
        self._build_groups()

    # ---------------------------------------------------------------------------------------------
    def _new_obj(self, kind, legs):
        o = Obj(len(self.objs), kind, tuple(sorted(legs)))
        self.objs.append(o)
        return o

    def _term_of_current(self, c, sign):
        cur = self.proc.currents
        if c.op == "ext_v":
            return Term(sign, c.op, (c.args[0],), tuple(sorted(c.legs)))
        if c.op in ("ext_ql", "ext_qr"):
            return Term(sign, c.op, (2 if c.op == "ext_ql" else 3,), tuple(sorted(c.legs)))
        return Term(sign, c.op, tuple(self._fobj[i] for i in c.args), tuple(sorted(c.legs)))

    def _build_objects(self):
        cur = self.proc.currents
        for c in cur:                      # ids are topologically ordered
            if len(c.legs) <= 2:
                o = self._new_obj(c.kind, c.legs)
                o.terms.append(self._term_of_current(c, 1))
                self._fobj[c.id] = o.id
        self._by_legs = defaultdict(list)
        for c in cur:
            self._by_legs[(c.kind, c.legs)].append(c)

    def object_for(self, kind, legs, word):
        """(object id, sign) of the colour-ordered combination sum_c col_c[word] c over the currents of
        this kind and leg set"""
        combo = tuple(sorted((c.id, c.col[word]) for c in self._by_legs[(kind, legs)] if c.col.get(word, 0)))
        assert combo, (kind, legs, word)
        assert all(abs(s) == 1 for _, s in combo)
        if len(legs) <= 2:
            assert len(combo) == 1
            return self._fobj[combo[0][0]], combo[0][1]
        sign = combo[0][1]
        canon = tuple((i, s * sign) for i, s in combo)
        if canon not in self._combo:
            if len(legs) <= 3:
                o = self._new_obj(kind, legs)
                for i, s in canon:
                    o.terms.append(self._term_of_current(self.proc.currents[i], s))
            else:
                terms = self._factorised_terms(canon, word, sign, legs)      # creates the argument objects first
                o = self._new_obj(kind, legs)
                o.terms = terms
            self._combo[canon] = o.id
        return self._combo[canon], sign

    def _factorised_terms(self, canon, word, sign, legs):
        """terms of a colour-ordered object with more than 3 legs, sum_c s_c c with s_c = sign * col_c[word]: its Feynman
        currents c = V(a_1, .., a_k) have arguments with up to 3 legs, which are not objects themselves, so the sum is
        factorised the way the amplitudes are (module docstring, (2)): col_c[word] = t * prod_i col_{a_i}[w_i] with w_i
        the sub-word of `word` seen by a_i and t = +-1 fixed by (vertex, leg sets, word); V is multilinear, hence
            sum_c s_c c = sum over (vertex, leg sets) of  sign t V(O_1, .., O_k),  O_i = sum_a col_a[w_i] a.
        The currents sort their arguments by id (v3, and the first two of v4: vertex function and colour are both odd
        under that exchange); here they are put in the order of their leg sets, so that one (vertex, leg sets) class is one
        term.  `_check_expansion` expands the result back into Feynman currents."""
        cur = self.proc.currents
        found = {}
        for cid, s_c in canon:
            c = cur[cid]
            args = [cur[i] for i in c.args]
            flip = 1
            if c.op in ("v3", "v4") and min(args[0].legs) > min(args[1].legs):
                args[0], args[1] = args[1], args[0]
                flip = -1                                  # Lorentz part alone changes sign (the colour is read off c.col)
            words = [_key_word(a, word) for a in args]
            prod = 1
            for a, w in zip(args, words):
                prod *= a.col.get(w, 0)
            assert prod in (1, -1), "coefficient of a current does not factorise"
            objs = tuple(self.object_for(a.kind, a.legs, w) for a, w in zip(args, words))
            t = s_c * prod * flip
            for _, os_ in objs:
                t *= os_
            key = (c.op, tuple(o for o, _ in objs))
            assert found.setdefault(key, t) == t
        # expansion check: the terms, multiplied out over the Feynman currents of their argument objects, are exactly canon
        import itertools
        inv_combo = getattr(self, "_members", None)
        if inv_combo is None:
            inv_combo = self._members = {}
        for cn, oid in self._combo.items():
            inv_combo.setdefault(oid, list(cn))
        for fid, oid in self._fobj.items():
            inv_combo.setdefault(oid, [(fid, 1)])
        got = {}
        for (op, ids), t in found.items():
            for pick in itertools.product(*[inv_combo[o] for o in ids]):
                fids, co = [f for f, _ in pick], t
                for _, s_ in pick:
                    co *= s_
                if op in ("v3", "v4") and fids[0] > fids[1]:
                    fids[0], fids[1] = fids[1], fids[0]
                    co = -co
                c = self.proc._memo.get((op, tuple(fids)))
                assert c is not None, "factorised object holds a current that no diagram has"
                got[c.id] = got.get(c.id, 0) + co
        assert {k: v for k, v in got.items() if v} == dict(canon), "factorised object differs from its Feynman currents"
        return [Term(t, op, ids, tuple(sorted(legs))) for (op, ids), t in sorted(found.items())]

    # ---------------------------------------------------------------------------------------------
    def _build_evals(self):
        """per colour flow sigma: the distinct vertex evaluations (op, ((object, sign), ...)) -> sign"""
        proc = self.proc
        cur = proc.currents
        assert max(len(c.legs) for c in cur) <= 4, "centroid branches with more than 4 legs are not supported"
        inv = {v: k for k, v in proc.rank.items()}
        self.sigmas = [inv[j] for j in range(self.ncolor)]
        self.evals = [dict() for _ in range(self.ncolor)]
        self._raw = [dict() for _ in range(self.ncolor)]       # for the expansion check
        for a in proc.amps:
            for j, co in a.jamps:
                s = inv[j]
                words = [_key_word(cur[i], s) for i in a.args]
                prod = 1
                for i, w in zip(a.args, words):
                    prod *= cur[i].col.get(w, 0)
                assert prod in (1, -1), "coefficient does not factorise"
                sign = co // prod
                assert sign in (1, -1)
                objs = tuple(self.object_for(cur[i].kind, cur[i].legs, w) for i, w in zip(a.args, words))
                key = (a.op, objs)
                if key in self.evals[j]:
                    assert self.evals[j][key] == sign
                self.evals[j][key] = sign
                self._raw[j][(a.op, a.args)] = co

    def _check_expansion(self):
        """expanding every factorised evaluation back into Feynman currents must give exactly the diagram
        program's (amplitude, coefficient) list of that colour flow: no term lost, none invented"""
        import itertools
        members = {}
        for canon, oid in self._combo.items():
            members[oid] = list(canon)
        for cid, oid in self._fobj.items():
            members[oid] = [(cid, 1)]
        for j in range(self.ncolor):
            got = {}
            for (op, objs), sign in self.evals[j].items():
                for combo in itertools.product(*[members[o] for o, _ in objs]):
                    co = sign
                    for (_, osign), (_, csign) in zip(objs, combo):
                        co *= osign * csign
                    k = (op, tuple(c for c, _ in combo))
                    got[k] = got.get(k, 0) + co
            got = {k: v for k, v in got.items() if v}
            assert got == self._raw[j], f"factorised colour flow {j} differs from the diagram program"

    # ---------------------------------------------------------------------------------------------
    def _split_xy(self, op, objs):
        """V(objs) = X . Y: index of Y, the raw-vertex term that builds X, and the rearrangement sign"""
        nlegs = [len(self.objs[o].legs) for o, _ in objs]
        iy = max(range(len(objs)), key=lambda i: (nlegs[i], i))
        ids = [o for o, _ in objs]
        if op == "ffv":                                   # (fo, v, fi)
            xop, args, sg = {2: ("x_row", (ids[0], ids[1]), 1), 0: ("x_col", (ids[1], ids[2]), 1),
                             1: ("x_bil", (ids[0], ids[2]), 1)}[iy]
        elif op == "vvv":                                 # totally antisymmetric: cyclic rotations are even
            xop, sg = "x_v3", 1
            args = {2: (ids[0], ids[1]), 0: (ids[1], ids[2]), 1: (ids[2], ids[0])}[iy]
        elif op == "vvvv":                                # (x y | z w) = (x.z)(y.w) - (x.w)(y.z)
            x, y, z, w = ids
            xop = "x_v4"                                  # x_v4(p, q, r) = (p.r) q - (q.r) p
            args, sg = {3: ((x, y, z), 1), 2: ((x, y, w), -1), 0: ((w, z, y), 1), 1: ((z, w, x), 1)}[iy]
        else:
            raise ValueError(op)
        return iy, xop, args, sg

    def _build_groups(self, merge=True):
        """groups of colour flows (same first `group_prefix` letters, or the stored partition), their pair objects and
        dot entries"""
        gp = self.group_prefix
        order = defaultdict(list)
        if gp == "file":
            from . import regroup
            for k, members in enumerate(regroup.load(self.n, self.sigmas)):
                order[k] = members
        else:
            for j, s in enumerate(self.sigmas):
                order[s[:gp]].append(j)
        self.groups = []          # dicts: sigmas [j], xobjs [ {legs, terms:[Term]} ], entries {j: [(xslot, yobj, sign)]}
        for pre in sorted(order):
            xkey_to_slot, xobjs, entries = {}, [], {}
            for j in order[pre]:
                per_y = defaultdict(list)                 # (y object, x legs) -> [(sign, xop, args)]
                for (op, objs), sign in sorted(self.evals[j].items()):
                    iy, xop, args, sg = self._split_xy(op, objs)
                    total = sign * sg
                    for _, os_ in objs:
                        total *= os_
                    yo = objs[iy][0]
                    key = yo if merge else (yo, len(per_y))
                    per_y[key].append((total, xop, args))
                ents = []
                for key, terms in per_y.items():
                    yo = key if merge else key[0]
                    terms = sorted(terms, key=lambda t: (t[1], t[2]))
                    s0 = terms[0][0]
                    canon = tuple((t[0] * s0, t[1], t[2]) for t in terms)
                    if canon not in xkey_to_slot:
                        legs = set()
                        for _, _, args in canon:
                            for a in args:
                                legs |= set(self.objs[a].legs)
                        legs = tuple(sorted(legs))
                        assert set(legs) | set(self.objs[yo].legs) == set(range(self.npar))
                        assert not set(legs) & set(self.objs[yo].legs)
                        xkey_to_slot[canon] = len(xobjs)
                        xobjs.append({"legs": legs,
                                      "terms": merge_v4_pairs([Term(sg_, xop, args, legs) for sg_, xop, args in canon])})
                    ents.append((xkey_to_slot[canon], yo, s0))
                entries[j] = ents
            self.groups.append({"sigmas": order[pre], "xobjs": xobjs, "entries": entries})

    def stats(self):
        nx = [len(g["xobjs"]) for g in self.groups]
        xv = [sum(1 << len(x["legs"]) for x in g["xobjs"]) for g in self.groups]
        ne = sum(len(e) for g in self.groups for e in g["entries"].values())
        nt = sum(len(x["terms"]) * (1 << len(x["legs"])) for g in self.groups for x in g["xobjs"])
        ov = sum(1 << len(o.legs) for o in self.objs)
        return {"name": self.name, "objects": len(self.objs), "object_variants": ov, "groups": len(self.groups),
                "xobjs_per_group_max": max(nx), "x_variants_per_group_max": max(xv), "dot_entries": ne,
                "x_term_variants": nt, "obj_term_variants": sum(len(o.terms) << len(o.legs) for o in self.objs)}


_CACHE = {}


def build(n, group_prefix=None):
    key = (n, group_prefix)
    if key not in _CACHE:
        _CACHE[key] = Program(n, group_prefix)
    return _CACHE[key]
