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
    int tile_major;        // 2: the tcgen05 operand layout, TF32-rounded (fp32 jamps, ncolor % 24 == 0; color_sum_tf32.cu);
                           // 1: [row / 128][2][ncolor][128] (one contiguous block per 128-row tile: TMA-friendly) instead
    double mt, wt;
};

struct HsContext;          // device copies of the tables

// tables go to the CURRENT device; cudaErrorInvalidValue if the process has no helicity-shared program
cudaError_t hs_create(int ngluon, HsContext** out);
void hs_destroy(HsContext* c);
const HsTables* hs_host_tables(const HsContext* c);
size_t hs_smem_bytes(const HsContext* c);
cudaError_t hs_launch(const HsContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st);

}  // namespace mg
