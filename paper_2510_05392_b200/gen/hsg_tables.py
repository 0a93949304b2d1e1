"""Tables of the helicity-shared program (gen/co_program.py) for the GENERIC kernel csrc/hsg_kernel.cu.

The tuned kernel of g g -> t tbar g g (g) (csrc/hs_kernel.cu, gen/hs_streams.py) keeps every object of an event in shared
memory and runs straight-line code per record type; that does not carry over to g g -> t tbar g g g g (Table 2,
PAPER.md:180-187: 15 495 diagrams, 720 colour flows, 256 helicities): 5 984 object variants (383 KB) and 43 680 variants of
pair objects (2.8 MB) per event.  The generic kernel interprets the program from these tables and keeps the objects of the
event a CTA works on in a scratch area in global memory (L1/L2) -- the "diagram-group hand-off through global memory" of
PAPER.md:424-444, here inside one kernel.  One group of colour flows (every pair object once).

Scratch area of one CTA: four component planes, byte(c, slot) = c * 16 * nslot + 16 * slot; variant v of an object with
first slot s0 is slot s0 + v; the objects come first (slots [0, ns_obj)), then the pair objects.

Packing (int32; variant bit j <-> helicity of the j-th leg in DESCENDING particle order, 1 = +: phase 3 runs lane = the
helicities of the five highest-numbered particles, so the variants the lanes of a warp read are the LOWEST bits of the index --
one contiguous run of 16-byte words, one L1 wavefront instead of four; measured in profiles/r3_gg_ttxgggg.md):
  obj[i]     = { first slot, L | legset << 8, first term, number of terms }                      (sorted by L = number of legs)
  term[t]    = { op | negative << 8 | legset(arg0) << 16 | legset(arg1) << 24, word(arg0), word(arg1), word(arg2) }
               word(arg) = first slot of the argument object | code << 16, code = 4 x 3 bits: position in the parent's variant
               index of the argument's j-th leg (7 = none); external ops (0..2): word(arg0) = particle number
               ops as in csrc/hs_tables.h
  p1_items   = obj << 8 | variant, level by level (p1_level[l] .. p1_level[l + 1] = objects with l + 1 legs); inside a level
               objects with the same sequence of opcodes are neighbours
  legset_mask[s] = particles of leg set s (bit p)
  xitem[i]   = { first term | terms << 24, slot | variant << 20 | vector-valued << 28 }: one variant of a pair object; sorted
               by the sequence of opcodes.  Vector-valued (opcodes >= 10): components 1-3 are negated at the store, so that
               the contraction with Y is a plain sum over the four components
  entry[e]   = { first slot of X, first slot of Y, row of vtab, negative | (particles 0, 1, 2 that are legs of X) << 1 |
                 lx << 4 | ly << 7 }: lx (ly) = number of legs of X (Y) other than particles 0, 1, 2 -- those three are the
                 HIGHEST bits of the variant index, so the variants a thread of phase 3 needs are 2^lx (2^ly) slots apart
  flow[f]    = { colour index, first entry, entries, 0 }
  vtab[row][h] (uint16) = variant of X | variant of Y << 8 for helicity combination h (bit npar-1-p of h = particle p)
"""
from __future__ import annotations

import numpy as np

from . import co_program

OPS = co_program.OPS
# flops per term (real operations, as counted for the tuned kernel's records in gen/emit_hs.py)
FLOPS = {"ext_v": 40, "ext_ql": 60, "ext_qr": 60, "v3": 150, "v4": 90, "ffv_l": 190, "ffv_r": 190, "ffv_p": 110,
         "x_row": 72, "x_col": 72, "x_bil": 80, "x_v3": 134, "x_v4": 112, "x_v4s": 170}


def _desc(legs):
    return tuple(sorted(legs, reverse=True))


def _code(parent, child):
    parent, child = _desc(parent), _desc(child)
    pos = [parent.index(p) for p in child]
    assert len(pos) <= 4 and all(q < 7 for q in pos)
    pos += [7] * (4 - len(pos))
    return pos[0] | (pos[1] << 3) | (pos[2] << 6) | (pos[3] << 9)


def build(n):
    prog = co_program.build(n, 0)
    assert len(prog.groups) == 1
    npar = prog.npar
    order = sorted(range(len(prog.objs)), key=lambda i: (len(prog.objs[i].legs), tuple(t.op for t in prog.objs[i].terms), i))
    slot0, s = {}, 0
    for i in order:
        slot0[i] = s
        s += 1 << len(prog.objs[i].legs)
    ns_obj = s
    legsets, ls_id = [], {}

    def lsid(legs):
        legs = tuple(sorted(legs))
        if legs not in ls_id:
            ls_id[legs] = len(legsets)
            legsets.append(legs)
        return ls_id[legs]

    terms = []

    def add_terms(tl, parent_legs):
        first = len(terms)
        for t in tl:
            neg = (1 if t.sign < 0 else 0) << 8
            if t.op.startswith("ext"):
                terms.append([OPS[t.op] | neg, t.args[0], 0, 0])
                continue
            ls = [lsid(prog.objs[x].legs) for x in t.args]
            w = [OPS[t.op] | neg | (ls[0] << 16) | (ls[1] << 24), 0, 0, 0]
            for k, x in enumerate(t.args):
                assert slot0[x] < 65536
                w[1 + k] = slot0[x] | (_code(tuple(parent_legs), prog.objs[x].legs) << 16)
            terms.append(w)
        return first, len(tl)

    obj_tab, p1_items, p1_level = [], [], [0]
    flops_p1 = 0
    for oi, i in enumerate(order):
        o = prog.objs[i]
        t0, nt = add_terms(o.terms, o.legs)
        obj_tab.append([slot0[i], len(o.legs) | (lsid(o.legs) << 8), t0, nt])
        flops_p1 += sum(FLOPS[t.op] + 8 for t in o.terms) << len(o.legs)
    maxlegs = max(len(o.legs) for o in prog.objs)
    for lvl in range(1, maxlegs + 1):
        for oi, i in enumerate(order):
            if len(prog.objs[i].legs) == lvl:
                p1_items += [(oi << 8) | v for v in range(1 << lvl)]
        p1_level.append(len(p1_items))

    g = prog.groups[0]
    xslot, s = [], ns_obj
    for x in g["xobjs"]:
        xslot.append(s)
        s += 1 << len(x["legs"])
    nslot = s
    assert nslot < (1 << 20)
    xitems, flops_p2 = [], 0
    shape = lambda x: (tuple(t.op for t in x["terms"]), -len(x["legs"]))
    for k in sorted(range(len(g["xobjs"])), key=lambda k: (shape(g["xobjs"][k]), k)):
        x = g["xobjs"][k]
        t0, nt = add_terms(x["terms"], x["legs"])
        assert t0 < (1 << 24) and nt < 128 and len(x["legs"]) <= 7
        vec = 1 if OPS[x["terms"][0].op] >= 10 else 0
        assert all((OPS[t.op] >= 10) == bool(vec) for t in x["terms"])
        for v in range(1 << len(x["legs"])):
            xitems.append([t0 | (nt << 24), (xslot[k] + v) | (v << 20) | (vec << 28)])
        flops_p2 += sum(FLOPS[t.op] + 8 for t in x["terms"]) << len(x["legs"])
    assert len(legsets) < 256

    vrows, vrow_id = [], {}

    def vrow(xlegs):
        if xlegs not in vrow_id:
            ylegs = _desc(p for p in range(npar) if p not in xlegs)
            xlegs_d = _desc(xlegs)
            row = []
            for h in range(1 << npar):
                hb = [(h >> (npar - 1 - p)) & 1 for p in range(npar)]
                vx = sum(hb[p] << j for j, p in enumerate(xlegs_d))
                vy = sum(hb[p] << j for j, p in enumerate(ylegs))
                assert vx < 256 and vy < 256
                row.append(vx | (vy << 8))
            vrow_id[xlegs] = len(vrows)
            vrows.append(row)
        return vrow_id[xlegs]

    flows, entries = [], []
    for j in g["sigmas"]:
        e0 = len(entries)
        for xs, yo, sign in g["entries"][j]:
            x = g["xobjs"][xs]
            assert set(x["legs"]) | set(prog.objs[yo].legs) == set(range(npar))
            nfx = sum(1 for p in x["legs"] if p < 3)
            lx, ly = len(x["legs"]) - nfx, (npar - len(x["legs"])) - (3 - nfx)
            flags = (1 if sign < 0 else 0) | (sum(1 << p for p in x["legs"] if p < 3) << 1) | (lx << 4) | (ly << 7)
            entries.append([xslot[xs], slot0[yo], vrow(tuple(x["legs"])), flags])
        flows.append([j, e0, len(entries) - e0, 0])
    i32 = lambda a, w: np.asarray(a, dtype=np.int64).astype(np.int32).reshape(-1, w)
    return {
        "npar": npar, "ncolor": prog.ncolor, "ns_obj": ns_obj, "nslot": nslot, "nlegsets": len(legsets),
        "obj": i32(obj_tab, 4), "term": i32(terms, 4), "p1_items": np.asarray(p1_items, np.int32),
        "p1_level": np.asarray(p1_level, np.int32), "legset_mask": np.asarray([sum(1 << p for p in l) for l in legsets], np.int32),
        "xitem": i32(xitems, 2), "entry": i32(entries, 4), "flow": i32(flows, 4),
        "vtab": np.asarray(vrows, np.int64).astype(np.uint16).reshape(-1, 1 << npar),
        # per event (phases 1, 2) and per (event, helicity) (phase 3: 4 complex multiply-adds per entry + sign)
        "flops_p1": float(flops_p1), "flops_p2": float(flops_p2), "flops_p3": 32.0 * len(entries),
        "ndiagrams": prog.proc.ndiagrams,
    }


_CACHE = {}


def tables(n):
    if n not in _CACHE:
        _CACHE[n] = build(n)
    return _CACHE[n]
