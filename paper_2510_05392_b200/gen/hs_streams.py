"""Device streams of the helicity-shared program (gen/co_program.py) in the form csrc/hs_kernel.cu reads them.

co_program.Program holds the factorised diagram program of g g -> t tbar + (n-2) g (Table 2 at
PAPER.md:180-187): colour-ordered objects (phase 1), per group of colour flows the pair objects X (phase 2) and the
dot-product entries jamp[sigma][h] += sign * sum_c X_c[hx] * Y_c[hy] (phase 3).  This module lowers it to what one CTA
(= one event, NW warps) executes, with every shared-memory address precomputed:

  shared-memory layout (per event).  An area (objects; staging area of the group's pair objects) is four PLANES, one
      per wavefunction component c; plane c holds one 16-byte complex number per SLOT:  byte(c, s) = c * PLANE + 16 s.
      PLANE = 32 (mod 128) bytes.  Variant v of an object with first slot s0 lives in slot s0 + perm(v),
      perm(v) = (v & ~1) | parity(v): flipping ANY one helicity bit of v changes the slot index by an odd number.
      Consequences: lane <-> variant accesses of one component (phases 1, 2) touch distinct consecutive 16-byte bank
      groups; the FP64 tensor-core fragments of phase 3 (two variants that differ in one helicity x four components)
      touch all eight bank groups whatever helicity bit distinguishes the two rows; component c is a compile-time
      immediate offset from ONE address register.

  phase 2  "chunks": 32 lanes = 32 (pair object, variant) items whose next <= 3 terms have the same opcodes, so that a
      chunk is straight-line code (csrc/hs_kernel.cu instantiates one function per chunk type listed here) and all
      terms of a chunk are in flight together.  A chunk is four uint2 per lane:
          rec0 = { byte offset of the item's slot in the staging plane | sign bits << 16,  type | first << 12 | last << 13 }
                 (type = one hex digit (opcode - 7) per term)
          rec1..3 (term k) = { offA | offB << 16,  offC | 0 }  or for x_v3  { offA | offB << 16,  32 lsA | (32 lsB) << 16 }
      off* = byte offsets of the argument's slot in plane 0 of the object area; ls* = leg sets (momenta K_ls).
      The chunks of the same 32 items form a UNIT (the accumulators stay in registers from one chunk to the next);
      units are the work items of phase 2 (p2unit[unit] = {first chunk, chunks}; grp[group] = {first unit, units,
      first flow, flows}).

  schedule  The kernel runs an event as a sequence of STEPS with one barrier each.  With a double-buffered staging area
      (nbuf = 2) step s = the colour flows of group s - 1 (phase 3) together with the units of group s (phase 2); with
      nbuf = 1 phases 2 and 3 of a group are two steps.  The items of a step are dealt to the nw warps of the CTA at
      build time, longest processing time first, by their instruction counts (ITEM_COST).  The chunk records are stored
      in execution order, so that the phase-2 work of a warp in a step is ONE contiguous run of chunks (rec0 says where
      a unit starts -- accumulators zeroed -- and where it ends -- result stored):
          wsched[step * nw + warp] = { first flow item | flows << 16, first chunk | chunks << 16 },  witem[] = flow index

  phase 3  one work item = one colour flow.  The entries of a flow are sorted into CLASSES: a class fixes which three legs
      index the 8 rows of the m8n8k4 FP64 MMA tile (R), which two legs its 4 complex columns (C) and which legs the tiles
      (T), so that all entries of a class accumulate into the SAME register fragments; only when a class is finished are
      the fragments added to the flow's accumulator in shared memory (slot = acc_swizzle(helicity)).  An entry fits a
      class if R is inside X's legs and C inside Y's (rows from X) or R = Y's legs and C inside X's ("swapped": rows
      from Y).  Records are per (entry, row = lane / 4): six 16-bit byte offsets (A fragments then B fragments; a lane
      adds (lane % 4) * PLANE) and a flag word; per (class, lane) the accumulator offsets of the lane's tiles.  Inside a
      class the entries are sorted by SHAPE (which operand gives the rows, which tile bits select the A fragment) and
      the class header holds the number of entries of each shape, so that the kernel runs one tight loop per shape
      with no per-entry dispatch.  The classes of a flow come in a canonical order; the sequence of their headers is the
      flow's SIGNATURE (p3flow[f].y bits 24..30) and the kernel instantiates straight-line code per signature
      (HS_FLOW_SIGS_<n> in generated/hs_gen.h); with pad = 1 all flows are padded to ONE signature (skip bits).

Everything here is integer bookkeeping of an exact rewriting; tests/hs_eval.py interprets these very streams in numpy and
tests/test_generator.py compares the resulting jamps with the oracle (CPU, no kernel involved).
"""
from __future__ import annotations

import itertools
from collections import defaultdict

import numpy as np

from . import co_program

MAXCHUNK = 3                # terms per phase-2 chunk

OPS = co_program.OPS
OPNAME = {v: k for k, v in OPS.items()}
# order of the phase-2 opcodes inside an item (chunks are cut from the sorted list)
X_ORDER = ["x_v3", "x_v4s", "x_v4", "x_row", "x_col", "x_bil"]
# relative cost of a term (flops of emit_hs.FLOPS + accumulation): order of the units inside a group
X_COST = {"x_row": 72, "x_col": 72, "x_bil": 80, "x_v3": 134, "x_v4": 112, "x_v4s": 170}
# instructions per work item (counted in the SASS of csrc/hs_kernel.cu), for the static schedule: per phase-2 term by
# opcode, per chunk, per phase-3 entry, per class, per flow
ITEM_COST = {"x_row": 75, "x_col": 75, "x_bil": 85, "x_v3": 125, "x_v4": 100, "x_v4s": 140, "chunk": 35, "unit": 25,
             "entry": 62, "class": 75, "flow": 110}


def chunk_code(ops):
    """type of a phase-2 chunk: one hex digit (opcode - 7) per term, first term in the low digit"""
    return sum((OPS[o] - 7) << (4 * j) for j, o in enumerate(ops))


def perm(v):
    return (v & ~1) | (bin(v).count("1") & 1)


def plane_bytes(nslots):
    b = 16 * nslots
    while b % 128 != 32:
        b += 16
    return b


def acc_swizzle(h):
    return co_program.acc_swizzle(h)


def _subpos(parent, child):
    pos = [parent.index(p) for p in child]
    assert len(pos) <= 3 and all(q < 7 for q in pos)
    pos += [7] * (3 - len(pos))
    return pos[0] | (pos[1] << 3) | (pos[2] << 6)


def _subvar(v, parent, child):
    """variant of `child` (legs, ascending) seen from variant v of `parent`"""
    return sum(((v >> parent.index(p)) & 1) << j for j, p in enumerate(child))


class Streams:
    def __init__(self, prog: co_program.Program, nw=8, nbuf=1, pad=0):
        self.prog = prog
        self.nw, self.nbuf, self.pad = nw, nbuf, pad
        self.npar = prog.npar
        self.ncolor = prog.ncolor
        self.ntile = 1 << (self.npar - 5)
        assert self.npar >= 6, "the streams need at least one tile leg (npar >= 6)"
        self._objects()
        self._phase2()
        self._phase3()
        self._schedule()

    # ---------------------------------------------------------------------------------------------
    def _lsid(self, legs):
        legs = tuple(sorted(legs))
        if legs not in self._ls:
            self._ls[legs] = len(self.legsets)
            self.legsets.append(legs)
        return self._ls[legs]

    def _objects(self):
        prog = self.prog
        self._ls, self.legsets = {}, []
        # level by level; inside a level objects with the same sequence of opcodes are neighbours, so that the lanes of a
        # warp of phase 1 (lane = (object, variant)) mostly run the same code
        order = sorted(range(len(prog.objs)), key=lambda i: (len(prog.objs[i].legs), tuple(t.op for t in prog.objs[i].terms), i))
        self.obj_order = order
        self.obj_slot = {}
        slot = 0
        for i in order:
            self.obj_slot[i] = slot
            slot += 1 << len(prog.objs[i].legs)
        self.ns_obj = slot
        self.obj_plane = plane_bytes(slot)
        index_of = {old: new for new, old in enumerate(order)}
        terms, obj_tab = [], []
        for i in order:
            o = prog.objs[i]
            t0 = len(terms)
            for t in o.terms:
                neg = 1 if t.sign < 0 else 0
                if t.op.startswith("ext"):
                    terms.append([OPS[t.op] | (neg << 8), t.args[0], 0, 0])
                    continue
                ls = [self._lsid(prog.objs[x].legs) for x in t.args]
                w = [OPS[t.op] | (neg << 8) | (ls[0] << 16) | (ls[1] << 24), 0, 0, 0]
                for k, x in enumerate(t.args):
                    w[1 + k] = self.obj_slot[x] | (_subpos(o.legs, prog.objs[x].legs) << 16)
                terms.append(w)
            obj_tab.append([self.obj_slot[i], len(o.legs) | (self._lsid(o.legs) << 8), t0, len(o.terms)])
        # phase-1 items (object << 8 | variant) in blocks of 32 lanes with one sequence of opcodes each (-1 = idle lane); the
        # blocks of a level are dealt to the nw warps at build time, longest processing time first (cost = flops of the
        # terms), and stored warp by warp: p1sched[level * nw + warp] = (first item, blocks)
        from .emit_hs import FLOPS
        p1_items, p1_level, p1sched = [], [0], []
        for lvl in (1, 2, 3):
            by_shape = defaultdict(list)
            for new, i in enumerate(order):
                if len(prog.objs[i].legs) == lvl:
                    shape = tuple(t.op for t in prog.objs[i].terms)
                    by_shape[shape] += [(new << 8) | v for v in range(1 << lvl)]
            blocks = []
            for shape, items in sorted(by_shape.items()):
                cost = sum(FLOPS[o] + 8 for o in shape)
                for k in range(0, len(items), 32):
                    blk = items[k:k + 32]
                    blocks.append((cost, blk + [-1] * (32 - len(blk))))
            load = [0] * self.nw
            per_warp = [[] for _ in range(self.nw)]
            for cost, blk in sorted(blocks, key=lambda b: (-b[0], b[1])):
                w = min(range(self.nw), key=lambda i: (load[i], i))
                load[w] += cost
                per_warp[w].append(blk)
            for w in range(self.nw):
                p1sched.append((len(p1_items), len(per_warp[w])))
                for blk in per_warp[w]:
                    p1_items += blk
            p1_level.append(len(p1_items))
        self.p1sched = p1sched
        self.obj_tab, self.p1_terms, self.p1_items, self.p1_level = obj_tab, terms, p1_items, p1_level
        self._index_of = index_of

    def _obj_off(self, oid, var):
        """byte offset (plane 0 of the object area) of variant `var` of object `oid`"""
        return 16 * (self.obj_slot[oid] + perm(var))

    # ---------------------------------------------------------------------------------------------
    def _phase2(self):
        prog = self.prog
        chunk_types = {}          # tuple of opcodes -> id
        recs, unit_tab, grp_units = [], [], []      # recs: [chunk][4][32][2] uint32
        self.unit_cost = []
        self.xslot = []           # per group: list of first staging slots of its pair objects
        ns_stage = 0
        for g in prog.groups:
            slots, s = [], 0
            for x in g["xobjs"]:
                slots.append(s)
                s += 1 << len(x["legs"])
            self.xslot.append(slots)
            ns_stage = max(ns_stage, s)
        self.trash_slot = ns_stage                      # padding lanes store here
        self.ns_stage = ns_stage + 2
        self.stage_plane = plane_bytes(self.ns_stage)
        assert self.stage_plane < 65536 and self.obj_plane < 65536, "16-bit byte offsets inside a plane"
        for gi, g in enumerate(prog.groups):
            by_shape = defaultdict(list)
            for k, x in enumerate(g["xobjs"]):
                terms = sorted(x["terms"], key=lambda t: (X_ORDER.index(t.op), t.args))
                shape = tuple(t.op for t in terms)
                # one kind per item: vector-valued (lowered at the store) or spinor-valued
                assert len({OPS[o] >= 10 for o in shape}) == 1
                for v in range(1 << len(x["legs"])):
                    by_shape[shape].append((k, v, terms))
            units = []            # (cost, [chunk blocks])
            for shape, items in sorted(by_shape.items()):
                cuts = [shape[i:i + MAXCHUNK] for i in range(0, len(shape), MAXCHUNK)]
                if len(shape) == 4:                       # 2 + 2 rather than 3 + 1
                    cuts = [shape[:2], shape[2:]]
                for i in range(0, len(items), 32):
                    lanes = items[i:i + 32]
                    blocks, t0 = [], 0
                    for ci, ops in enumerate(cuts):
                        ct = chunk_code(ops)
                        chunk_types[ct] = tuple(OPS[o] for o in ops)
                        blk = np.zeros((4, 32, 2), dtype=np.uint32)
                        blk[0, :, 0] = 16 * self.trash_slot
                        blk[0, :, 1] = ct | ((1 if ci == 0 else 0) << 12) | ((1 if ci == len(cuts) - 1 else 0) << 13)
                        for l, (k, v, terms) in enumerate(lanes):
                            x = g["xobjs"][k]
                            signs = 0
                            for j in range(len(ops)):
                                t = terms[t0 + j]
                                assert t.op == ops[j]
                                if t.sign < 0:
                                    signs |= 1 << j
                                offs = [self._obj_off(a, _subvar(v, x["legs"], prog.objs[a].legs)) for a in t.args]
                                if t.op == "x_v3":
                                    ls = [self._lsid(prog.objs[a].legs) for a in t.args]
                                    blk[1 + j, l] = (offs[0] | (offs[1] << 16), (32 * ls[0]) | ((32 * ls[1]) << 16))
                                else:
                                    blk[1 + j, l] = (offs[0] | (offs[1] << 16), offs[2] if len(offs) > 2 else 0)
                            blk[0, l, 0] = (16 * (self.xslot[gi][k] + perm(v))) | (signs << 16)
                        blocks.append(blk)
                        t0 += len(ops)
                    units.append((sum(X_COST[o] for o in shape), blocks))
            # work items of the group, most expensive first
            u0 = len(unit_tab)
            for cost, blocks in sorted(units, key=lambda u: -u[0]):
                unit_tab.append((len(recs), len(blocks)))
                icost = ITEM_COST["unit"]
                for blk in blocks:
                    ct = int(blk[0, 0, 1]) & 0xFFF
                    icost += ITEM_COST["chunk"] + sum(ITEM_COST[OPNAME[op]] for op in chunk_types[ct])
                self.unit_cost.append(icost)
                recs += blocks
            grp_units.append((u0, len(unit_tab) - u0))
        self.chunk_types = dict(sorted(chunk_types.items()))      # code -> opcodes
        self.p2rec = np.asarray(recs, dtype=np.uint32).reshape(-1, 4, 32, 2)
        self.p2unit = np.asarray(unit_tab, dtype=np.int32).reshape(-1, 2)
        self._grp_units = grp_units

    # ---------------------------------------------------------------------------------------------
    def _classes_for(self, ents):
        """smallest set of classes (R, C, swapped-allowed) covering the entries [(X legs, Y legs)] of one colour flow"""
        legs = range(self.npar)
        cover = {}
        for R in itertools.combinations(legs, 3):
            Rs = frozenset(R)
            rest = [l for l in legs if l not in Rs]
            for C in itertools.combinations(rest, 2):
                Cs = frozenset(C)
                got = frozenset(i for i, (X, Y) in enumerate(ents)
                                if (Rs <= X and Cs <= Y) or (Rs == Y and Cs <= X))
                if got and got not in cover:
                    cover[got] = (R, C)
        sets = sorted(cover, key=lambda s: (-len(s), sorted(s)))
        full = frozenset(range(len(ents)))
        for k in range(1, 7):
            for combo in itertools.combinations(sets, k):
                if frozenset().union(*combo) == full:
                    return [cover[c] for c in combo], [set(c) for c in combo]
        raise AssertionError("no class cover")

    def _phase3(self):
        prog, npar = self.prog, self.npar
        ntile = self.ntile
        hbit = lambda p: npar - 1 - p
        self.max_flows = max(len(g["sigmas"]) for g in prog.groups)
        flows_raw = []            # per flow: (group, position in the group, jamp, [(R, C, T, [(shape, rec)])])
        shapes = set()
        for gi, g in enumerate(prog.groups):
            for fi, j in enumerate(g["sigmas"]):
                ents = [(frozenset(g["xobjs"][xs]["legs"]), frozenset(prog.objs[yo].legs), xs, yo, sign)
                        for xs, yo, sign in g["entries"][j]]
                classes, covered = self._classes_for([(e[0], e[1]) for e in ents])
                # every entry goes to the compatible class with the fewest entries so far
                members = [[] for _ in classes]
                for i in sorted(range(len(ents)), key=lambda i: sum(i in c for c in covered)):
                    k = min((k for k in range(len(classes)) if i in covered[k]), key=lambda k: len(members[k]))
                    members[k].append(i)
                assert all(members)
                cls_out = []
                for (R, C), mem in zip(classes, members):
                    T = tuple(l for l in range(npar) if l not in R and l not in C)
                    recs_c = []
                    for i in mem:
                        X, Y, xs, yo, sign = ents[i]
                        xl, yl = tuple(sorted(X)), tuple(sorted(Y))
                        swapped = not (frozenset(R) <= X)
                        al, bl = (yl, xl) if swapped else (xl, yl)          # legs of the A-side / B-side operand
                        a_off = (lambda v: self._obj_off(yo, v)) if swapped else (lambda v: 16 * (self.xslot[gi][xs] + perm(v)))
                        b_off = (lambda v: 16 * (self.xslot[gi][xs] + perm(v))) if swapped else (lambda v: self._obj_off(yo, v))
                        assert set(R) <= set(al) and set(C) <= set(bl)
                        mask = sum(1 << b for b in range(len(T)) if T[b] in al)     # tile bits that select the A fragment
                        ta = [b for b in range(len(T)) if T[b] in al]
                        tb = [b for b in range(len(T)) if T[b] not in al]
                        na, nb = 1 << len(ta), 1 << len(tb)
                        shape = (1 if swapped else 0) | (mask << 1)
                        shapes.add((shape, na, nb))
                        rec = np.zeros((8, 4), dtype=np.uint32)
                        for row in range(8):
                            offs = []
                            for a in range(na):
                                v = sum(((row >> b) & 1) << al.index(R[b]) for b in range(3))
                                v |= sum(((a >> q) & 1) << al.index(T[ta[q]]) for q in range(len(ta)))
                                offs.append(a_off(v))
                            aw = [0, 0]
                            for q, o in enumerate(offs):
                                aw[q >> 1] |= o << (16 * (q & 1))
                            offs = []
                            c2, ri = row >> 1, row & 1
                            for b_ in range(nb):
                                v = sum(((c2 >> b) & 1) << bl.index(C[b]) for b in range(2))
                                v |= sum(((b_ >> q) & 1) << bl.index(T[tb[q]]) for q in range(len(tb)))
                                offs.append(b_off(v) + 8 * ri)
                            bw = [0, 0]
                            for q, o in enumerate(offs):
                                bw[q >> 1] |= o << (16 * (q & 1))
                            # word layout: A offsets fill x (, y); B offsets follow in the next free word(s)
                            words = aw[: (na + 1) // 2] + bw[: (nb + 1) // 2]
                            assert len(words) <= 3
                            words += [0] * (3 - len(words))
                            rec[row] = words + [shape | ((1 if sign < 0 else 0) << 31)]
                        recs_c.append((shape, rec))
                    cls_out.append((R, C, T, recs_c))
                flows_raw.append((gi, fi, j, cls_out))
        self.p3shapes = sorted(shapes)
        codes = [sh for sh, _, _ in self.p3shapes]
        assert len(codes) <= 4, "the class header holds four shape counts"
        self.p3shape_codes = codes
        recs, cls_tab, cls_hdr, flows, grp = [], [], [], [], []
        counts_of = lambda recs_c: tuple(sum(1 for sh, _ in recs_c if sh == c) for c in codes)
        # A flow's classes come in a canonical order (by their shape counts); the sequence of their headers is the flow's
        # SIGNATURE, and the kernel runs every signature as its own straight-line code.  pad = 1: ONE signature for the
        # whole process -- max_cls classes, each with hmax[k] slots for the entries of shape k; missing entries / classes
        # are slots with the SKIP bit (record word w bit 8) / header 0 -- because the instruction cache of the SM is smaller
        # than the kernel (2 -> 5: three signatures measured 13 % slower than one although they execute fewer instructions).
        max_cls = max(len(f[3]) for f in flows_raw)
        hmax = [max(counts_of(co[3])[k] for f in flows_raw for co in f[3]) for k in range(len(codes))]
        assert all(c < 16 for c in hmax) and max_cls <= 5
        pack = lambda counts: sum(c << (4 * k) for k, c in enumerate(counts))
        self.flow_sigs = {}       # sequence of class headers -> signature id
        # shapes present in EVERY slot need no skip test
        self.p3_always = sum(1 << k for k in range(len(codes))
                             if not self.pad or (all(counts_of(co[3])[k] == hmax[k] for f in flows_raw for co in f[3]) and
                                                 all(len(f[3]) == max_cls for f in flows_raw)))
        skip_rec = np.zeros((8, 4), dtype=np.uint32)
        skip_rec[:, 3] = 0x100
        self.flow_real_entries = []
        for gi in range(len(prog.groups)):
            mine = [f for f in flows_raw if f[0] == gi]
            grp.append(self._grp_units[gi] + (len(flows), len(mine)))
            for _, fi, j, cls_out in mine:
                rec0, cls0 = len(recs), len(cls_tab)
                cls_out = sorted(cls_out, key=lambda co: tuple(-x for x in counts_of(co[3])))
                nreal, sig = 0, []
                for ci in range(max_cls if self.pad else len(cls_out)):
                    ct = np.zeros((32, 4), dtype=np.uint32)
                    if ci < len(cls_out):
                        R, C, T, recs_c = cls_out[ci]
                        # accumulator slot of (lane, tile): rows <-> R, complex columns <-> C, tiles <-> T
                        for lane in range(32):
                            row, c2 = lane >> 2, lane & 3
                            for t in range(ntile):
                                h = sum(((row >> b) & 1) << hbit(R[b]) for b in range(3))
                                h |= sum(((c2 >> b) & 1) << hbit(C[b]) for b in range(2))
                                h |= sum(((t >> b) & 1) << hbit(T[b]) for b in range(len(T)))
                                ct[lane, t] = 16 * acc_swizzle(h)
                        counts = counts_of(recs_c)
                        cls_hdr.append(pack(counts))
                        for k, code in enumerate(codes):
                            mine_k = [r for sh, r in recs_c if sh == code]
                            recs += mine_k + ([skip_rec] * (hmax[k] - len(mine_k)) if self.pad else [])
                        nreal += len(recs_c)
                        sig.append(pack(hmax) if self.pad else pack(counts))
                    else:
                        cls_hdr.append(0)
                        recs += [skip_rec] * sum(hmax)
                        sig.append(pack(hmax))
                    cls_tab.append(ct)
                sid = self.flow_sigs.setdefault(tuple(sig), len(self.flow_sigs))
                assert fi < 256 and sid < 128
                flows.append((rec0, len(sig) | ((len(recs) - rec0) << 8) | (fi << 16) | (sid << 24), cls0, j))
                self.flow_real_entries.append((len(cls_out), nreal))
        assert not self.pad or len(self.flow_sigs) == 1
        self.p3rec = np.asarray(recs, dtype=np.uint32).reshape(-1, 8, 4)
        self.p3cls = np.asarray(cls_tab, dtype=np.uint32).reshape(-1, 32, 4)
        self.p3clsh = np.asarray(cls_hdr, dtype=np.int32)
        self.p3flow = np.asarray(flows, dtype=np.int32).reshape(-1, 4)
        self.grp = np.asarray(grp, dtype=np.int32).reshape(-1, 4)

    # ---------------------------------------------------------------------------------------------
    def steps(self):
        """[(group whose flows run (or None), group whose units run (or None))] in execution order"""
        ng = len(self.prog.groups)
        if self.nbuf == 2:
            return [(s - 1 if s >= 1 else None, s if s < ng else None) for s in range(ng + 1)]
        return [x for g in range(ng) for x in ((None, g), (g, None))]

    def _schedule(self):
        nw = self.nw
        wsched, witem = [], []
        new_recs, new_unit = [], [None] * len(self.p2unit)
        self.step_load = []
        for g3, g2 in self.steps():
            items = []                                   # (cost, code)
            if g3 is not None:
                _, _, f0, nf = (int(x) for x in self.grp[g3])
                for f in range(f0, f0 + nf):
                    ncls_real, nent_real = self.flow_real_entries[f]
                    cost = ITEM_COST["flow"] + ITEM_COST["class"] * ncls_real + ITEM_COST["entry"] * nent_real
                    items.append((cost, f))
            if g2 is not None:
                u0, nu, _, _ = (int(x) for x in self.grp[g2])
                for u in range(u0, u0 + nu):
                    items.append((self.unit_cost[u], (1 << 31) | u))
            load = [0] * nw
            per_warp = [[] for _ in range(nw)]
            for cost, code in sorted(items, key=lambda it: (-it[0], it[1])):
                w = min(range(nw), key=lambda i: (load[i], i))
                load[w] += cost
                per_warp[w].append((cost, code))
            # hill climbing on the makespan: move or swap items between the most loaded warp and any other
            improved = True
            while improved:
                improved = False
                hi = max(range(nw), key=lambda i: (load[i], -i))
                for lo in sorted(range(nw), key=lambda i: (load[i], i)):
                    if lo == hi:
                        continue
                    best = None
                    for a_, (ca, _) in enumerate(per_warp[hi]):
                        for b_, (cb, _) in [(-1, (0, 0))] + list(enumerate(per_warp[lo])):
                            new = max(load[hi] - ca + cb, load[lo] + ca - cb)
                            if new < load[hi] and (best is None or new < best[0]):
                                best = (new, a_, b_)
                    if best is not None:
                        _, a_, b_ = best
                        ia = per_warp[hi].pop(a_)
                        load[hi] -= ia[0]; load[lo] += ia[0]
                        if b_ >= 0:
                            ib = per_warp[lo].pop(b_)
                            load[lo] -= ib[0]; load[hi] += ib[0]
                            per_warp[hi].append(ib)
                        per_warp[lo].append(ia)
                        improved = True
                        break
            self.step_load.append(load)
            for w in range(nw):
                mine = sorted(per_warp[w], key=lambda it: (-it[0], it[1]))
                fl = [code for _, code in mine if not code >> 31]
                un = [code & 0x7FFFFFFF for _, code in mine if code >> 31]          # unit indices (old numbering)
                c0 = len(new_recs)
                for u in un:
                    oc, nc = (int(x) for x in self.p2unit[u])
                    new_unit[u] = (len(new_recs), nc)
                    new_recs += [self.p2rec[oc + k] for k in range(nc)]
                assert len(witem) < 65536 and len(fl) < 65536 and len(new_recs) < 65536
                wsched.append((len(witem) | (len(fl) << 16), c0 | ((len(new_recs) - c0) << 16)))
                witem += fl
        assert len(new_recs) == len(self.p2rec) and all(u is not None for u in new_unit)
        self.p2rec = np.asarray(new_recs, dtype=np.uint32).reshape(-1, 4, 32, 2)
        self.p2unit = np.asarray(new_unit, dtype=np.int32).reshape(-1, 2)
        self.wsched = np.asarray(wsched, dtype=np.uint32).reshape(-1, 2)
        self.witem = np.asarray(witem, dtype=np.uint32)

    # ---------------------------------------------------------------------------------------------
    def tables(self):
        i32 = lambda a, w: np.asarray(a, dtype=np.int64).astype(np.int32).reshape(-1, w)
        ncls = self.p3flow[:, 1] & 0xFF
        return {
            "npar": self.npar, "ncolor": self.ncolor, "ngroups": len(self.prog.groups), "ntile": self.ntile,
            "ns_obj": self.ns_obj, "obj_plane": self.obj_plane, "ns_stage": self.ns_stage, "stage_plane": self.stage_plane,
            "nlegsets": len(self.legsets), "max_flows": self.max_flows, "max_classes": int(ncls.max()),
            "legset_mask": np.asarray([sum(1 << p for p in legs) for legs in self.legsets], np.int32),
            "obj": i32(self.obj_tab, 4), "term": i32(self.p1_terms, 4), "p1_items": np.asarray(self.p1_items, np.int32),
            "p1_level": np.asarray(self.p1_level, np.int32), "p1sched": np.asarray(self.p1sched, np.int32).reshape(-1, 2),
            "p2rec": self.p2rec, "p2unit": self.p2unit, "grp": self.grp, "chunk_types": self.chunk_types,
            "nw": self.nw, "nbuf": self.nbuf, "nsteps": len(self.steps()), "wsched": self.wsched, "witem": self.witem,
            "p3rec": self.p3rec, "p3cls": self.p3cls, "p3clsh": self.p3clsh, "p3flow": self.p3flow,
            "p3shapes": self.p3shapes, "p3shape_codes": self.p3shape_codes, "flow_sigs": dict(self.flow_sigs), "p3_pad": self.pad, "p3_always": self.p3_always,
        }


_CACHE = {}


def build(n, group_prefix, nw=8, nbuf=1, pad=0):
    key = (n, group_prefix, nw, nbuf, pad)
    if key not in _CACHE:
        _CACHE[key] = Streams(co_program.build(n, group_prefix), nw, nbuf, pad)
    return _CACHE[key]
