// hsg_kernel.cuh -- host interface of the generic helicity-shared diagram kernel (hsg_kernel.cu) and the layout of its
// tables (written by gen/hsg_tables.py through gen/emit_hsg.py; packing documented in gen/hsg_tables.py).
#pragma once
#include <cuda_runtime.h>

#include "hs_kernel.cuh"

namespace mg {

struct HsgTables {
    int npar, ncolor, ns_obj, nslot, nlegsets, nobj, nterm, np1, nxitem, nentry, nflow, nvrow, nlevel, ndiagrams, nlrow;
    int p1_level[8];
    const int* obj;
    const int* term;
    const int* p1_items;
    const int* legset_mask;
    const int* xitem;
    const int* entry;
    const int* flow;
    const unsigned short* vtab;
    // phase 3 on the FP64 tensor path: entry records in class order, per-lane fragment offsets, per-flow class tables
    const int* dentry;
    const unsigned* ltab;
    const unsigned* flowL;
    const unsigned* flowT;
    // colour matrix: numerators (over cden) of the row of the identity permutation; C[s][s'] = row0[rank(s^-1 o s')]
    const int* cmat_row0;
    int cden;
    double flops_p1, flops_p2, flops_p3;      // per event (phases 1, 2) and per (event, helicity) (phase 3)
};

const HsgTables* hsg_tables(int ngluon);        // generated/hsg_tables_gen.cu; NULL if the process has none

struct HsgContext;

// tables and the CTAs' scratch areas go to the CURRENT device
cudaError_t hsg_create(int ngluon, HsgContext** out);
void hsg_destroy(HsgContext* c);
const HsgTables* hsg_host_tables(const HsgContext* c);
// jamps [2][ncolor][rows] (tile_major = 0) or, fp32 only, the tcgen05 operand layout (tile_major = 2, ncolor % 24 == 0)
cudaError_t hsg_launch(const HsgContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st);
// phase 3 on the FP64 tensor path (default) or on the FP64 ALU (option "p3_tensor" of include/mg5_b200.h)
void hsg_set_tensor(HsgContext* c, bool on);
bool hsg_get_tensor(const HsgContext* c);


// The no-allocation variant (mg_sigma_batch_noalloc): the same kernel with its scratch areas in a file-scope static __device__
// array of 26 MiB (8 CTAs' worth for g g -> t tbar g g g g).  hsg_static_setup: once per context with its device current
// (resolves the array's device address, cudaGetSymbolAddress); hsg_launch_static calls no allocating routine.  Launches that
// overlap on the GPU race on the shared array.
cudaError_t hsg_static_setup(HsgContext* c);
int hsg_static_ctas(const HsgContext* c);
cudaError_t hsg_launch_static(const HsgContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st);

}  // namespace mg
