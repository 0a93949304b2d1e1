// hs_tables.h -- tables of the helicity-shared diagram program (written by gen/co_program.py, read by hs_kernel.cu).
//
// One CTA evaluates one event for all 2^npar helicity combinations:
//   phase 1  colour-ordered objects with <= 3 legs (signed sums of Feynman off-shell currents of one leg set),
//            every helicity variant of their own legs, level by level, into shared memory
//   phase 2  per group of colour flows: pair objects X = raw vertex contracted with all branches but the largest
//   phase 3  jamp[sigma][h] = sum_entries sign * sum_c X_c[variant_x(h)] * Y_c[variant_y(h)]
//
// Packing (all int32 unless stated; "complex units" = 16 bytes in shared memory; an object with L legs holds
// 4 components x 2^L variants as [component][variant]; variant bit j <-> helicity of the j-th leg in ascending
// particle order, 1 = +):
//   obj[i]    = { offset in the object area, L | legset<<8, first term, number of terms }        (sorted by L)
//   term[t]   = { op | negative<<8 | sub0<<16 | sub1<<24, arg0 | arg1<<16, arg2 | sub2<<16, 0 }
//               args are object ids (external ops: arg0 = particle); sub_k = which variant bits of the parent
//               belong to argument k (argument variant = pext(parent variant, sub_k))
//   p1_items  = obj<<8 | variant, level by level; p1_level[l] .. p1_level[l+1] is level l+1
//   legset_mask[s] = particles of leg set s (bit p); K_s = sum of all-incoming momenta
//   group[g]  = { first xobj, first x item, number of x items, first sigma, number of sigmas, 0, 0, 0 }
//   xobj[k]   = { offset in the staging area, log2(variants), first term, number of terms }
//   x_items   = (xobj index within the group)<<8 | variant
//   sigma[s]  = { jamp index, first entry, number of entries, 0 }
//   entry[e]  = { x offset | x variants<<16, y offset | y variants<<16, vtab row, sign }
//   vtab[row][h] (uint16) = x variant | y variant<<8 for helicity combination h (particle 0 = most significant bit)
//   hdep[row][v] (uint8)  = acc_swizzle(helicity bits of x variant v) for v < 32, of y variant v - 32 for v >= 32
//                           (phase 3 on the FP64 tensor path: accumulator slot of (vx, vy) = hdep[vx] ^ hdep[32 + vy])
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
