// hs_tables.h -- tables of the helicity-shared diagram program (written by gen/co_program.py, read by hs_kernel.cu).
//
// One CTA evaluates one event for all 2^npar helicity combinations:
//   phase 1  colour-ordered objects with <= 3 legs (signed sums of Feynman off-shell currents of one leg set),
//            every helicity variant of their own legs, level by level, into shared memory
//   phase 2  per group of colour flows: pair objects X = raw vertex contracted with all branches but the largest
//   phase 3  jamp[sigma][h] = sum_entries sign * sum_c X_c[variant_x(h)] * Y_c[variant_y(h)]
//
// Packing (all int32 unless stated; "slots" = 16-byte complex numbers in shared memory; an object with L legs holds
// 2^L variants x 4 components; variant bit j <-> helicity of the j-th leg in ascending particle order, 1 = +; the
// layout inside an area is hs_kernel.cu's: 64-byte blocks [variant][component], component index swizzled):
//   obj[i]    = { offset in the object area (multiple of 8 slots), L | legset<<8, first term, number of terms }   (sorted by L)
//   term[t]   = { op | negative<<8 | legset(arg0)<<16 | legset(arg1)<<24, word(arg0), word(arg1), word(arg2) }
//               word(arg) = offset of the argument object | code<<16, code = 3 x 3 bits: position in the parent's variant
//               index of the argument's j-th leg (7 = none); external ops (0..2): word(arg0) = particle number
//               ops: 0 ext_v, 1 ext_ql, 2 ext_qr, 3 v3, 4 v4, 5 ffv_l, 6 ffv_r, 7 ffv_p (currents with propagator, phase 1);
//                    8 x_row, 9 x_col, 10 x_bil, 11 x_v3, 12 x_v4, 13 x_v4s (raw vertices, phase 2; 13 = both orderings of
//                    the four-gluon vertex that share the middle argument: 2 (p.r) q - (q.r) p - (q.p) r)
//   p1_items  = obj<<8 | variant, level by level; p1_level[l] .. p1_level[l+1] is level l+1
//   legset_mask[s] = particles of leg set s (bit p); K_s = sum of all-incoming momenta
//   group[g]  = { first xobj, first x item, number of x items (multiple of 32), first sigma, number of sigmas, 0, 0, 0 }
//   xobj[k]   = { offset in the staging area, log2(variants), first term, number of terms }
//   x_items   = (xobj index within the group)<<8 | variant, or -1 (padding); 32 consecutive items = one work unit of
//               items with the same term shape, units sorted by decreasing cost
//   sigma[s]  = { jamp index, first entry, number of entries, 0 }
//   entry[e]  = { x offset | x variants<<16, y offset | y variants<<16, vtab row, sign }
//   vtab[row][h] (uint16) = x variant | y variant<<8 for helicity combination h (particle 0 = most significant bit)
//   hdep[row][v] (uint8)  = acc_swizzle(helicity bits of x variant v) for v < 32, of y variant v - 32 for v >= 32
//                           (phase 3 on the FP64 tensor path: accumulator slot of (vx, vy) = hdep[vx] ^ hdep[32 + vy])
// hs_create (hs_kernel.cu) flattens group/xobj/x_items/term and sigma/entry/hdep once more into the per-lane record
// streams the kernel actually reads in phases 2 and 3.
#pragma once

namespace mg {

struct HsTables {
    int npar, ncolor, obj_area, stage_area, nobj, nterm, nlegsets, ngroups, nxobj, nxitems, nsigma, nentry, nvrow;
    int np1;
    int p1_level[4];
    const int* obj;
    const int* term;
    const int* p1_items;
    const int* legset_mask;
    const int* group;
    const int* xobj;
    const int* x_items;
    const int* sigma;
    const int* entry;
    const unsigned short* vtab;
    const unsigned char* hdep;                // [nvrow][40]: swizzled accumulator index parts, x variants 0..31 then y variants 0..7
    double flops_p1, flops_p2, flops_p3;      // per event (phases 1, 2) and per (event, helicity) (phase 3)
};

const HsTables* hs_tables(int ngluon);          // generated/hs_tables_gen.cu; NULL if the process has none

}  // namespace mg
