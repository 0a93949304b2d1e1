// hs_kernel.cuh -- host interface of the helicity-shared diagram kernel (hs_kernel.cu).
#pragma once
#include <cuda_runtime.h>

#include "hs_tables.h"

namespace mg {

struct HsLaunch {
    const double* mom;     // DEVICE [nevt][npar][4]
    int nevt;
    const int* d_pos;      // DEVICE [2^npar]: row of helicity combination h inside its event, -1 = skipped
    int nrow_evt;          // rows per event (= number of good helicities)
    void* d_jamps;         // DEVICE [2][ncolor][rows] fp64 or fp32; row = event * nrow_evt + pos[h]
    long rows;             // row stride of the jamps buffer
    int tile_major;        // 1: [row / 128][2][ncolor][128] (one contiguous block per 128-row tile: TMA-friendly) instead
    double mt, wt;
    unsigned long long* prof;   // DEVICE [8] or NULL: clock64 sums per phase as seen by thread 0 of every CTA (diagnostics)
};

struct HsContext;          // device copies of the tables

cudaError_t hs_create(int ngluon, HsContext** out);      // cudaErrorInvalidValue if the process has no tables
void hs_destroy(HsContext* c);
const HsTables* hs_host_tables(const HsContext* c);
size_t hs_smem_bytes(const HsContext* c);
// nsplit = threads per helicity combination (1, 2 or 4; blockDim = 2^npar * nsplit <= 256)
// phase3 = 0: dot products on the scalar FP64 ALUs (thread = helicity); 1: on the FP64 tensor path (DMMA, warp = colour flow)
cudaError_t hs_launch(const HsContext* c, bool jamps_fp64, const HsLaunch& a, int nsplit, int phase3, cudaStream_t st);

}  // namespace mg
