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
  flow[f]    = { colour index, first entry, entries, classes (tensor path, below) }
  vtab[row][h] (uint16) = variant of X | variant of Y << 8 for helicity combination h (bit npar-1-p of h = particle p)

Phase 3 on the FP64 tensor path (csrc/hsg_kernel.cu, p3_tensor): one entry for all 2^npar helicity combinations is the complex
outer-product sum out[hp][hq] = sum_c P_c[hp] Q_c[hq] over the four components, i.e. 8 tiles of mma.sync.m8n8k4.f64: rows = the
helicities of three particles R (all legs of one operand, P), column pairs (re, im) = the helicities of two particles C (legs of
the other operand, Q), tile index = the helicities of the remaining three particles T.  The accumulator fragments stay in
registers as long as (R, C) do not change: the entries of a flow are grouped into CLASSES with one (R, C) each (smallest cover,
3 classes per flow at 6 gluons) and stored class by class; at a class change the flow's running sum goes through the warp's
accumulator in shared memory -- stored in the old class's (lane, tile) order, loaded back in the new one's (slot of combination h =
swz(h), conflict-free for a class's lane order where the choice of R[0] allows it).
  dentry[e]  = { first slot of X | first slot of Y << 16, row of ltab | legs of X << 16 | MASK << 20 | negative << 23 |
                 last entry of its class << 24, d0 | d1 << 16, d2 | swx << 16 | swy << 20 }: MASK bit i = T[i] is a leg of P; d_i =
                 byte distance in the warp's operand buffer between the variants that differ in the helicity of T[i] (added to the
                 A fragment's offset if MASK bit i is set, else to the B fragment's).  Operand buffer: [X: 4 component planes of
                 (2^lgx + 1) x 16 bytes], then Y the same with lgy; inside a plane the variant index has bit 2 and bit swx (swy)
                 exchanged (2 = as it is): the leg whose helicity distinguishes the lanes of one shared-memory access phase (R[0]
                 in P, C[0] in Q) sits at bit 2, which with the odd plane length makes every fragment load conflict-free
  ltab[row][lane] (uint32) = byte offset of the lane's A element (P_c[variant of row lane / 4], c = lane % 4: 16 bytes re, im)
                 | offset of its B element << 16 (Q_c[variant of column pair lane / 8], + 8 for odd lane / 4: the imaginary part)
  flowL[f][lane] (uint32) = byte 8 k: swz(h) of the lane's accumulator elements in class k of flow f for tile 0
                 (rows lane / 4 <-> R, column pair lane % 4 <-> C)
  flowT[f][2 k + {0, 1}] (uint32) = byte t of the pair: swz of the helicities of T for tile t of class k (XORed onto flowL's byte)
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


# 16-byte slot of helicity combination h in a flow's accumulator (csrc/hsg_kernel.cu acc_swz): linear over GF(2); the
# low three bits (the bank group of a 16-byte access) get a different pattern from every higher bit of h but the last
_SWZ_PAT = (3, 5, 6, 7, 1)
_SWZ_VEC = (1, 2, 4) + _SWZ_PAT           # bank-group pattern of bit b of h


def acc_swz(h):
    g = 0
    for b, pat in enumerate(_SWZ_PAT):
        if (h >> (3 + b)) & 1:
            g ^= pat
    return h ^ g


def _independent(v):
    """three vectors of GF(2)^3 linearly independent"""
    a, b, c = v
    return 0 not in (a, b, c, a ^ b, a ^ c, b ^ c, a ^ b ^ c)


def _class_cover(npar, xmasks):
    """smallest cover of the entries of a flow (bit masks of the legs of X) by classes (R, C): R = three particles that are all
    legs of one operand, C = two particles that are legs of the other one; returns [(R mask, C mask, [entry indices])], every
    entry in the first class of the cover that holds it.  Exact: the sets of entries that some (R, C) covers are few once the
    dominated ones are dropped (16 at 6 gluons), so all combinations of up to four are tried (3 classes for every flow at 6
    gluons; a greedy cover needs 4 for 330 of the 720)"""
    import itertools
    full = (1 << npar) - 1
    by_set = {}
    for R in itertools.combinations(range(npar), 3):
        rm = sum(1 << p for p in R)
        for C in itertools.combinations([p for p in range(npar) if p not in R], 2):
            cm = sum(1 << p for p in C)
            m = 0
            for i, x in enumerate(xmasks):
                if ((x & rm) == rm and (~x & full & cm) == cm) or ((~x & full & rm) == rm and (x & cm) == cm):
                    m |= 1 << i
            if m and m not in by_set:
                by_set[m] = (rm, cm)
    sets = sorted(by_set, key=lambda m: (-bin(m).count("1"), m))
    sets = [m for m in sets if not any((m | o) == o and m != o for o in sets)]
    everything = (1 << len(xmasks)) - 1
    for k in range(1, 5):
        for combo in itertools.combinations(sets, k):
            u = 0
            for m in combo:
                u |= m
            if u == everything:
                out, seen = [], 0
                for m in combo:
                    out.append(by_set[m] + ([i for i in range(len(xmasks)) if (m >> i) & 1 and not (seen >> i) & 1],))
                    seen |= m
                return out
    raise AssertionError("no cover of the entries of a flow by <= 4 classes")


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

    import itertools
    flows, entries, dentries, flowL, flowT = [], [], [], [], []
    lrows, lrow_id = [], {}
    pbit = lambda p: npar - 1 - p            # bit of particle p in the helicity combination h

    def staged(legs_d, special):
        """positions of the legs in the STAGED variant index of an operand: the natural ones (descending particle order) with
        bit 2 and the bit of `special` exchanged (so that the 8 / 16 lanes of a shared-memory access phase, which differ in the
        helicity of `special` and in the component, fall into different banks: component planes are 16 bytes longer than a
        power of two); returns ({particle: position}, natural position of special = the bit the copy exchanges with bit 2)"""
        pos = {p: i for i, p in enumerate(legs_d)}
        if len(legs_d) < 3:
            return pos, 2
        sw = pos[special]
        other = legs_d[2]
        pos[special], pos[other] = 2, sw
        return pos, sw

    def lrow(xlegs, R, C):
        """per-lane operand offsets of an entry with legs xlegs of X in a class (R, C) (ordered tuples); also the bits the copy
        of X and of Y exchanges with bit 2 and the staged positions of the legs of the row / column operand"""
        key = (xlegs, R, C)
        if key not in lrow_id:
            xd, yd = _desc(xlegs), _desc(p for p in range(npar) if p not in xlegs)
            lgx, lgy = len(xd), len(yd)
            basey = 4 * ((16 << lgx) + 16)
            if set(R) <= set(xd):
                px, swx = staged(xd, R[0])
                py, swy = staged(yd, C[0])
                pp, psp, basep, pq, psq, baseq = px, (16 << lgx) + 16, 0, py, (16 << lgy) + 16, basey
            else:
                px, swx = staged(xd, C[0])
                py, swy = staged(yd, R[0])
                pp, psp, basep, pq, psq, baseq = py, (16 << lgy) + 16, basey, px, (16 << lgx) + 16, 0
            assert set(R) <= set(pp) and set(C) <= set(pq)
            row = []
            for lane in range(32):
                r, c = lane >> 2, lane & 3
                a = basep + c * psp + 16 * sum(((r >> i) & 1) << pp[R[i]] for i in range(3))
                col = lane >> 2
                b = baseq + c * psq + 16 * sum((((col >> 1) >> i) & 1) << pq[C[i]] for i in range(2)) + 8 * (col & 1)
                assert a < 65536 and b < 65536
                row.append(a | (b << 16))
            lrow_id[key] = (len(lrows), swx, swy, pp, pq)
            lrows.append(row)
        return lrow_id[key]

    for j in g["sigmas"]:
        e0 = len(entries)
        ents = g["entries"][j]
        xm = [sum(1 << p for p in g["xobjs"][xs]["legs"]) for xs, yo, sign in ents]
        tensor = npar == 8                     # the tensor path's lane / tile split is 3 + 2 + 3 particles
        cover = _class_cover(npar, xm) if tensor else [(0, 0, list(range(len(ents))))]
        assert len(cover) <= 4
        Lw, Tw = [0] * 32, [0] * 8
        for k, (rm, cm, members) in enumerate(cover):
            if not tensor:
                for xs, yo, sign in ents:
                    xlegs = tuple(g["xobjs"][xs]["legs"])
                    nfx = sum(1 for p in xlegs if p < 3)
                    lx, ly = len(xlegs) - nfx, (npar - len(xlegs)) - (3 - nfx)
                    flags = (1 if sign < 0 else 0) | (sum(1 << p for p in xlegs if p < 3) << 1) | (lx << 4) | (ly << 7)
                    entries.append([xslot[xs], slot0[yo], vrow(xlegs), flags])
                break
            Rs, Cs = [p for p in range(npar) if (rm >> p) & 1], [p for p in range(npar) if (cm >> p) & 1]
            T = tuple(p for p in range(npar) if not ((rm | cm) >> p) & 1)
            # lane bits 0, 1 = C[0], C[1], bit 2 = R[0]: the eight lanes of a 16-byte shared-memory access phase
            R, C = tuple(Rs), tuple(Cs)
            for Rp in itertools.permutations(Rs):
                if _independent([_SWZ_VEC[pbit(Cs[0])], _SWZ_VEC[pbit(Cs[1])], _SWZ_VEC[pbit(Rp[0])]]):
                    R = Rp
                    break
            for lane in range(32):
                h = sum((((lane >> 2) >> i) & 1) << pbit(R[i]) for i in range(3)) | sum((((lane & 3) >> i) & 1) << pbit(C[i]) for i in range(2))
                Lw[lane] |= acc_swz(h) << (8 * k)
            for t in range(8):
                h = sum(((t >> i) & 1) << pbit(T[i]) for i in range(3))
                Tw[2 * k + (t >> 2)] |= acc_swz(h) << (8 * (t & 3))
            for m, i in enumerate(members):
                xs, yo, sign = ents[i]
                x = g["xobjs"][xs]
                xlegs = tuple(x["legs"])
                assert set(xlegs) | set(prog.objs[yo].legs) == set(range(npar))
                nfx = sum(1 for p in xlegs if p < 3)
                lx, ly = len(xlegs) - nfx, (npar - len(xlegs)) - (3 - nfx)
                flags = (1 if sign < 0 else 0) | (sum(1 << p for p in xlegs if p < 3) << 1) | (lx << 4) | (ly << 7)
                entries.append([xslot[xs], slot0[yo], vrow(xlegs), flags])
                lr, swx, swy, pp, pq = lrow(xlegs, R, C)
                mask, d = 0, []
                for b, p in enumerate(T):
                    if p in pp:
                        mask |= 1 << b
                        d.append(16 << pp[p])
                    else:
                        d.append(16 << pq[p])
                assert xslot[xs] < 65536 and slot0[yo] < 65536 and 4 <= len(xlegs) <= 6
                dentries.append([xslot[xs] | (slot0[yo] << 16),
                                 lr | (len(xlegs) << 16) | (mask << 20) | ((1 if sign < 0 else 0) << 23) |
                                 ((1 if m == len(members) - 1 else 0) << 24), d[0] | (d[1] << 16), d[2] | (swx << 16) | (swy << 20)])
        flows.append([j, e0, len(entries) - e0, len(cover) if tensor else 0])
        if tensor:
            flowL.append(Lw)
            flowT.append(Tw)
    assert len(lrows) < 65536
    i32 = lambda a, w: np.asarray(a, dtype=np.int64).astype(np.int32).reshape(-1, w)
    return {
        "npar": npar, "ncolor": prog.ncolor, "ns_obj": ns_obj, "nslot": nslot, "nlegsets": len(legsets),
        "obj": i32(obj_tab, 4), "term": i32(terms, 4), "p1_items": np.asarray(p1_items, np.int32),
        "p1_level": np.asarray(p1_level, np.int32), "legset_mask": np.asarray([sum(1 << p for p in l) for l in legsets], np.int32),
        "xitem": i32(xitems, 2), "entry": i32(entries, 4), "flow": i32(flows, 4), "dentry": i32(dentries, 4),        # (empty unless npar = 8)
        "ltab": np.asarray(lrows, np.int64).astype(np.uint32).reshape(-1, 32),
        "flowL": np.asarray(flowL, np.int64).astype(np.uint32).reshape(-1, 32),
        "flowT": np.asarray(flowT, np.int64).astype(np.uint32).reshape(-1, 8),
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
