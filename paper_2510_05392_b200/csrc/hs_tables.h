// hs_tables.h -- device streams of the helicity-shared diagram program (written by gen/hs_streams.py through
// gen/emit_hs.py, read by hs_kernel.cu).
//
// One CTA (HsCfg<NG>::NW warps) evaluates one event for all 2^npar helicity combinations:
//   phase 1  colour-ordered objects with <= 3 legs (signed sums of Feynman off-shell currents of one leg set), every
//            helicity variant of their own legs, level by level, into the object area
//   phase 2  per group of colour flows: pair objects X = raw vertex contracted with all branches but the largest (Y),
//            into the staging area; "chunks" of 32 lanes x <= 3 terms of the same opcodes
//   phase 3  jamp[sigma][h] = sum_entries sign * sum_c X_c[variant_x(h)] * Y_c[variant_y(h)] on the FP64 tensor path,
//            one warp per colour flow, entries sorted into classes that share their register fragments
//
// Shared-memory areas: four component planes; byte(c, slot) = c * PLANE + 16 * slot, PLANE = 32 (mod 128); variant v of
// an object with first slot s0 sits in slot s0 + perm(v), perm(v) = (v & ~1) | parity(v)   (gen/hs_streams.py).
//
// Packing (int32 / uint32; variant bit j <-> helicity of the j-th leg in ascending particle order, 1 = +):
//   obj[i]    = { first slot in the object area, L | legset << 8, first term, number of terms }              (sorted by L)
//   term[t]   = { op | negative << 8 | legset(arg0) << 16 | legset(arg1) << 24, word(arg0), word(arg1), word(arg2) }
//               word(arg) = first slot of the argument object | code << 16, code = 3 x 3 bits: position in the parent's
//               variant index of the argument's j-th leg (7 = none); external ops (0..2): word(arg0) = particle number
//               ops: 0 ext_v, 1 ext_ql, 2 ext_qr, 3 v3, 4 v4, 5 ffv_l, 6 ffv_r, 7 ffv_p (currents with propagator, phase 1);
//                    8 x_row, 9 x_col, 10 x_bil, 11 x_v3, 12 x_v4, 13 x_v4s (raw vertices, phase 2; 13 = both orderings of
//                    the four-gluon vertex that share the middle argument: 2 (p.r) q - (q.r) p - (q.p) r)
//   p1_items  = obj << 8 | variant (-1: idle lane), level by level (p1_level[l] .. p1_level[l+1] is level l+1), in blocks of 32
//               lanes with one sequence of opcodes; p1sched[(level - 1) * NW + warp] = { first item, blocks }: the blocks this
//               warp evaluates (dealt at build time, longest first)
//   legset_mask[s] = particles of leg set s (bit p); K_s = sum of all-incoming momenta
//   p2rec[chunk][4][lane] (uint2):
//               rec0 = { byte offset of the item's slot in staging plane 0 | sign bits << 16, type | first << 12 | last << 13 },
//                      type = one hex digit (op - 7) per term, first term in the low digit
//               rec1..3 (term k) = { offA | offB << 16, offC }; x_v3: { offA | offB << 16, 32 legset(A) | 32 legset(B) << 16 }
//               off* = byte offset of the argument's slot in object plane 0
//   p2unit[unit] = { first chunk, number of chunks }: the chunks of the same 32 items (host side only: schedule, tests)
//   grp[group]   = { first unit, units, first flow, flows }
//   wsched[step * NW + warp] = { first flow item | flows << 16, first chunk | chunks << 16 }: the work of this warp in this
//               step (static schedule, longest processing time first): its colour flows (witem[] = flow indices), then ONE
//               contiguous run of chunks -- p2rec is stored in execution order.
//               Steps: NBUF = 2: step s = flows of group s - 1 and units of group s; NBUF = 1: units(g), flows(g) alternate
//   p3rec[entry][row = lane / 4] (uint4): x, y, z = 16-bit byte offsets of the A fragments (nA of them, whole words),
//               then of the B fragments (nB; + 8 for odd rows: the imaginary half), w = shape | skip << 8 | negative << 31,
//               shape = swapped | mask << 1 (mask: tile bits that select the A fragment); the entries of a class are
//               sorted by shape, in the order HsCfg<NG>::SHAPE0..3; skip: a slot of a padded flow that holds no entry
//   p3cls[class][lane] (uint2): 16-bit byte offsets into the flow's accumulator of this lane's complex number in tiles 0..3
//   p3clsh[class] = number of (real) entries of shape k in bits 4k .. 4k+3; 0 = a class a padded flow does not have
//   p3flow[f] = { first entry, classes | entry slots << 8 | accumulator << 16 | signature << 24, first class, jamp index };
//               signature = id of the flow's sequence of class headers (slots per shape), HS_FLOW_SIGS_<n> in
//               generated/hs_gen.h: the kernel runs each signature as straight-line code; HsCfg::P3_PAD = 1: all flows padded
//               to one signature
#pragma once

namespace mg {

struct HsTables {
    int npar, ncolor, ngroups, ntile, ns_obj, obj_plane, ns_stage, stage_plane, nlegsets, max_flows;
    int nobj, nterm, np1, nchunk, nunit, nentry, ncls, nflow, nsteps, nitem;
    int p1_level[4];
    const int* obj;
    const int* term;
    const int* p1_items;
    const int* legset_mask;
    const unsigned* p2rec;
    const int* p2unit;
    const unsigned* p3rec;
    const unsigned* p3cls;
    const int* p3clsh;
    const int* p3flow;
    const int* grp;
    const unsigned* wsched;
    const unsigned* witem;
    const int* p1sched;
    double flops_p1, flops_p2, flops_p3;      // per event (phases 1, 2) and per (event, helicity) (phase 3)
};

const HsTables* hs_tables(int ngluon);          // generated/hs_tables_gen.cu; NULL if the process has none

}  // namespace mg
