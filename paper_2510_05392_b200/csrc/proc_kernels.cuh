// proc_kernels.cuh -- the diagram kernel in the paper's thread layout, generic over a process.
//
// One thread = one (event, helicity) pair: the event index runs along x ("one event <-> one
// thread"), the good-helicity index is the y dimension of the grid instead of a stream per helicity
// (MG_SCHED_STREAMS launches the same kernel with one y-slice per stream).
//   stage a0  momenta read (fp64, AOS)
//   stage a2  external wavefunctions     |
//   stage a3  currents + amplitudes      | P::jamps()  (generated, csrc/generated/<proc>_jamps.cuh)
//   stage a4  jamps: registers/local memory, or stored as [2][ncolor][rows] for the tensor-core colour sum
//   stage a5  (MG_CS_FUSED) colour sum on the scalar ALUs in the triangular form of PAPER.md:303, 328
#pragma once

#include "mg_internal.cuh"

namespace mg {

template <class P, typename T, typename T2, int MODE>
__global__ void __launch_bounds__(256) diagrams_kernel(const DiagLaunch a)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= a.nevt) return;
    const int ih = a.hel_base + blockIdx.y;
    const int ihel = a.d_hel[ih];
    phys<T> ph;
    ph.mt = T(a.ph.mt); ph.wt = T(a.ph.wt); ph.ee = T(a.ph.ee); ph.gl = T(a.ph.gl); ph.gr = T(a.ph.gr);
    ph.mz = T(a.ph.mz); ph.wz = T(a.ph.wz);
    cx<T> jamp[P::NCOLOR];
    P::template jamps<T>(a.mom + (size_t)e * (P::NPAR * 4), ihel, ph, jamp);
    if (MODE == 0) {
        // sum_ij C_ij (re_i re_j + im_i im_j) = sum_i [ C_ii |J_i|^2 + 2 sum_{j>i} C_ij (re_i re_j + im_i im_j) ]
        const T2* __restrict__ cm = reinterpret_cast<const T2*>(a.d_cmat);
        T2 acc = T2(0);
#pragma unroll 1
        for (int i = 0; i < P::NCOLOR; i++) {
            const T2 ri = T2(jamp[i].re), ii = T2(jamp[i].im);
            T2 sr = T2(0), si = T2(0);
            for (int j = i + 1; j < P::NCOLOR; j++) {
                const T2 c = cm[i * P::NCOLOR + j];
                sr += c * T2(jamp[j].re);
                si += c * T2(jamp[j].im);
            }
            const T2 cii = cm[i * P::NCOLOR + i];
            acc += ri * (cii * ri + T2(2) * sr) + ii * (cii * ii + T2(2) * si);
        }
        a.d_meh[(size_t)ih * a.evt_stride + a.evt_offset + e] = a.norm * double(acc);
    } else {
        T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
        const size_t row = (size_t)ih * a.nevt + e;
#pragma unroll 1
        for (int c = 0; c < P::NCOLOR; c++) {
            out[(size_t)c * a.rows + row] = T2(jamp[c].re);
            out[(size_t)(P::NCOLOR + c) * a.rows + row] = T2(jamp[c].im);
        }
    }
}

template <class P, typename T, typename T2>
static cudaError_t launch_t(const DiagLaunch& a, cudaStream_t st)
{
    dim3 grid((a.nevt + a.block - 1) / a.block, a.nhel, 1);
    if (a.mode == 0) diagrams_kernel<P, T, T2, 0><<<grid, a.block, 0, st>>>(a);
    else diagrams_kernel<P, T, T2, 1><<<grid, a.block, 0, st>>>(a);
    return cudaGetLastError();
}

template <class P>
static cudaError_t launch_any(int precision, const DiagLaunch& a, cudaStream_t st)
{
    switch (precision) {
        case 0: return launch_t<P, double, double>(a, st);
        case 1: return launch_t<P, double, float>(a, st);
        case 2: return P::launch_f32(a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace mg

// the all-fp32 instantiation: in this translation unit (default), in one of its own (MG_EXT_FP32: MG_DEFINE_GG_PROCESS_F32
// there), or left out (MG_NO_FP32; mg_init_process then refuses MG_FP32 for the process)
#if defined(MG_NO_FP32)
#define MG_HAS_FP32 false
#define MG_F32_BODY(NS) return cudaErrorInvalidValue;
#define MG_F32_DECL(NS)
#elif defined(MG_EXT_FP32)
#define MG_HAS_FP32 true
#define MG_F32_BODY(NS) return launch_f32_##NS(a, st);
#define MG_F32_DECL(NS) cudaError_t launch_f32_##NS(const DiagLaunch& a, cudaStream_t st);
#else
#define MG_HAS_FP32 true
#define MG_F32_BODY(NS) return launch_t<P_##NS, float, float>(a, st);
#define MG_F32_DECL(NS)
#endif

#define MG_DEFINE_GG_PROCESS_F32(NS)                                                                       \
    namespace mg {                                                                                         \
    struct P32_##NS {                                                                                      \
        static constexpr int NPAR = NS::NPAR, NCOLOR = NS::NCOLOR;                                         \
        template <typename T>                                                                              \
        static __device__ __forceinline__ void jamps(const double* pe, int ihel, const phys<T>& ph, cx<T>* j) \
        {                                                                                                  \
            NS::jamps<T>(pe, ihel, ph.mt, ph.wt, j);                                                       \
        }                                                                                                  \
    };                                                                                                     \
    cudaError_t launch_f32_##NS(const DiagLaunch& a, cudaStream_t st) { return launch_t<P32_##NS, float, float>(a, st); } \
    }

// Defines the traits struct and the descriptor of a generated process namespace NS.
#define MG_DEFINE_GG_PROCESS(NS, NGROUPS)                                                                  \
    namespace mg {                                                                                         \
    MG_F32_DECL(NS)                                                                                        \
    struct P_##NS {                                                                                        \
        static constexpr int NPAR = NS::NPAR, NCOLOR = NS::NCOLOR;                                         \
        template <typename T>                                                                              \
        static __device__ __forceinline__ void jamps(const double* pe, int ihel, const phys<T>& ph, cx<T>* j) \
        {                                                                                                  \
            NS::jamps<T>(pe, ihel, ph.mt, ph.wt, j);                                                       \
        }                                                                                                  \
        static cudaError_t launch_f32(const DiagLaunch& a, cudaStream_t st);                               \
    };                                                                                                     \
    cudaError_t P_##NS::launch_f32(const DiagLaunch& a, cudaStream_t st) { MG_F32_BODY(NS) }               \
    const ProcessDesc* desc_##NS()                                                                         \
    {                                                                                                      \
        static const ProcessDesc d = { #NS, NS::NGLUON, NS::NPAR, NS::NCOMB, NS::NCOLOR, NS::NDIAGRAMS,    \
                                       NS::NAMPS, NS::NCURRENTS, NGROUPS, NS::DENOM, NS::CDEN, NS::CMAT,   \
                                       NS::FLOPS_PER_EVENT_HELICITY, NS::NGLUON, MG_HAS_FP32, &launch_any<P_##NS> }; \
        return &d;                                                                                         \
    }                                                                                                      \
    }
