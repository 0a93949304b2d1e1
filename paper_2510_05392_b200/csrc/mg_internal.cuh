// mg_internal.cuh -- types shared by the per-process translation units and the C-ABI layer (api.cu).
#pragma once

#include <cuda_runtime.h>

#include "helas.cuh"

namespace mg {

// physics parameters handed to the device code (couplings are inputs of the ME engine;
// here alpha_s is fixed per batch, BASELINE.json configs)
template <typename T>
struct phys {
    T mt, wt;              // top mass / width
    T ee, gl, gr;          // e, Z couplings to charged leptons (left, right)
    T mz, wz;              // Z mass / width
};

struct DiagLaunch {
    const double* mom;     // DEVICE [nevt][npar][4]
    int nevt;              // events in this launch
    int evt_stride;        // row stride of the per-helicity output (total events of the batch)
    int evt_offset;        // first event of this launch inside the batch (for me_h indexing)
    const int* d_hel;      // DEVICE list of helicity indices
    int hel_base, nhel;    // this launch covers list entries [hel_base, hel_base + nhel)
    phys<double> ph;
    double norm;           // g^(2n) / (denom * cden)
    const void* d_cmat;    // DEVICE [ncolor][ncolor] integer numerators as T2
    double* d_meh;         // DEVICE [nhel_total][evt_stride]: per-helicity terms (MG_CS_FUSED)
    void* d_jamps;         // DEVICE [2][ncolor][rows] as T2 (MG_CS_TENSOR); rows = nhel_total_in_chunk * nevt
    long rows;             // rows of the jamps buffer
    int block;             // threads per block
    int mode;              // MG_CS_FUSED / MG_CS_TENSOR
};

struct ProcessDesc {
    const char* name;
    int ngluon, npar, ncomb, ncolor, ndiagrams, namps, ncurrents, ngroups;
    double denom;
    int cden;
    const int* cmat;       // HOST [ncolor*ncolor]
    double flops;          // diagram stage, per (event, helicity)
    int coupling_order;    // norm carries g^(2*coupling_order)
    bool has_fp32;         // the all-fp32 instantiation (MG_FP32) was compiled in
    // precision: 0 = fp64 amplitudes + fp64 colour sum, 1 = fp64 + fp32, 2 = fp32 + fp32
    cudaError_t (*launch)(int precision, const DiagLaunch&, cudaStream_t);
};

const ProcessDesc* desc_epem_mupmum();
const ProcessDesc* desc_gg_ttx();
const ProcessDesc* desc_gg_ttxg();
const ProcessDesc* desc_gg_ttxgg();
const ProcessDesc* desc_gg_ttxggg();

}  // namespace mg
