// color_sum.cu -- colour sum as a contraction over all (helicity, event) rows at once ("ihel3p1b":
// "concatenate jamps of all helicities as nGoodHel*nevt events, one multiplication").
//
//   me_row = Re(J^dagger C J) = A^T C A + B^T C B,  J = A + iB            (Eq. 1)
//
// fp64: C (integer numerators, symmetric positive definite) = L L^T, so me_row = |A L|^2 + |B L|^2: ONE
//   triangular GEMM Z = X L on the FP64 tensor path (DMMA, mma.sync.m8n8k4.f64) and a sum of squares of the
//   accumulators -- the k-tiles above the diagonal of L are skipped, which recovers the factor 2 of the
//   paper's triangular trick on the tensor cores, and removes the second (dot) step of
//   the paper's BLAS formulation (gemm + gemmStridedBatched with an intermediate buffer).
// fp32/mixed: tcgen05 kernel, see color_sum_tf32.cu.
#include <math.h>
#include <stdint.h>

#include <vector>

#include "color_sum.cuh"

namespace mg {

// ---------------------------------------------------------------------------------------------------------
// scalar-ALU reference kernel: one thread per row, triangular form
template <typename T, int NC>
__global__ void __launch_bounds__(128) color_sum_alu_kernel(const T* __restrict__ cm, const T* __restrict__ J, long nrows,
                                                            double* __restrict__ out, RowMap map)
{
    const long r = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= nrows) return;
    T re[NC], im[NC];
#pragma unroll 4
    for (int c = 0; c < NC; c++) { re[c] = J[(long)c * nrows + r]; im[c] = J[(long)(NC + c) * nrows + r]; }
    T acc = T(0);
#pragma unroll 1
    for (int i = 0; i < NC; i++) {
        T sr = T(0), si = T(0);
        for (int j = i + 1; j < NC; j++) {
            const T c = cm[i * NC + j];
            sr += c * re[j];
            si += c * im[j];
        }
        const T cii = cm[i * NC + i];
        acc += re[i] * (cii * re[i] + T(2) * sr) + im[i] * (cii * im[i] + T(2) * si);
    }
    map.store(out, r, double(acc));
}

template <typename T>
static cudaError_t alu_dispatch(int nc, const void* cm, const void* J, long nrows, double* out, RowMap map, cudaStream_t st)
{
    const int blk = 128;
    const unsigned grid = (unsigned)((nrows + blk - 1) / blk);
#define CASE(N) case N: color_sum_alu_kernel<T, N><<<grid, blk, 0, st>>>((const T*)cm, (const T*)J, nrows, out, map); break;
    switch (nc) { CASE(1) CASE(2) CASE(6) CASE(24) CASE(120) default: return cudaErrorInvalidValue; }
#undef CASE
    return cudaGetLastError();
}

cudaError_t color_sum_alu(bool is_fp64, int ncolor, const void* d_cmat, const void* d_jamps, long nrows, double* d_out,
                          cudaStream_t st, const RowMap* map)
{
    RowMap id;                        // identity: out[r]
    id.rows_valid = nrows;
    const RowMap m = map ? *map : id;
    return is_fp64 ? alu_dispatch<double>(ncolor, d_cmat, d_jamps, nrows, d_out, m, st)
                   : alu_dispatch<float>(ncolor, d_cmat, d_jamps, nrows, d_out, m, st);
}

// ---------------------------------------------------------------------------------------------------------
// DMMA kernel.  One warp = 8 rows (their Re and Im parts: two m8 tiles sharing every B fragment).
// Fragment layout of mma.sync.m8n8k4.f64: a = A[lane/4][lane%4], b = B[lane%4][lane/4],
// c0,c1 = C[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// NT = number of 8-wide n-tiles (ncolor padded to 8*NT); L: [8*NT][8*NT] row-major, lower-triangular, zero padded
template <int NT>
__global__ void __launch_bounds__(128) color_sum_dmma_kernel(const double* __restrict__ L, const double* __restrict__ X, int ncolor,
                                                             long rows_padded, RowMap map, double* __restrict__ meh)
{
    constexpr int NCP = 8 * NT;
    const int lane = threadIdx.x & 31;
    const long row0 = ((long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 8;
    if (row0 >= rows_padded) return;
    const int ar = lane >> 2, ak = lane & 3;       // A fragment: row, k
    double cre[NT][2], cim[NT][2];
#pragma unroll
    for (int j = 0; j < NT; j++) { cre[j][0] = cre[j][1] = cim[j][0] = cim[j][1] = 0.0; }
    const double* xre = X + row0 + ar;
    const double* xim = X + (long)ncolor * rows_padded + row0 + ar;
    // the A fragments (jamps, streamed from HBM) are fetched two k-steps ahead; L stays in L1/L2
    auto load_a = [&](int k0, double& are, double& aim) {
        const int k = k0 + ak;
        are = 0.0; aim = 0.0;
        if (k < ncolor) { are = __ldg(xre + (long)k * rows_padded); aim = __ldg(xim + (long)k * rows_padded); }
    };
    double a_re, a_im, n_re, n_im, m_re, m_im;
    load_a(0, a_re, a_im);
    load_a(4, n_re, n_im);
#pragma unroll 1
    for (int k0 = 0; k0 < NCP; k0 += 4) {
        load_a(k0 + 8, m_re, m_im);
        const double* lrow = L + (long)(k0 + ak) * NCP + ar;      // b = L[k0 + lane%4][8j + lane/4]
#pragma unroll
        for (int j = 0; j < NT; j++) {
            if (8 * j <= k0 + 3) {                            // lower-triangular: columns 8j.. need k >= 8j
                const double b = __ldg(lrow + 8 * j);
                dmma(cre[j][0], cre[j][1], a_re, b);
                dmma(cim[j][0], cim[j][1], a_im, b);
            }
        }
        a_re = n_re; a_im = n_im; n_re = m_re; n_im = m_im;
    }
    double s = 0.0;
#pragma unroll
    for (int j = 0; j < NT; j++)
        s += cre[j][0] * cre[j][0] + cre[j][1] * cre[j][1] + cim[j][0] * cim[j][0] + cim[j][1] * cim[j][1];
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    const long row = row0 + ar;
    if (ak == 0) map.store(meh, row, s);
}

// Cholesky factor of the integer colour matrix, computed on the host in long double and zero-padded to a
// multiple of 8 columns; the caller (api.cu) uploads it once per handle.  Returns false if C is not
// positive definite.
bool color_cholesky_padded(int ncolor, const int* cmat, std::vector<double>& lp, int* ncp_out)
{
    const int ncp = (ncolor + 7) / 8 * 8;
    std::vector<long double> l((size_t)ncolor * ncolor, 0.0L);
    for (int i = 0; i < ncolor; i++)
        for (int j = 0; j <= i; j++) {
            long double s = cmat[(size_t)i * ncolor + j];
            for (int k = 0; k < j; k++) s -= l[(size_t)i * ncolor + k] * l[(size_t)j * ncolor + k];
            if (i == j) { if (s <= 0) return false; l[(size_t)i * ncolor + i] = sqrtl(s); }
            else l[(size_t)i * ncolor + j] = s / l[(size_t)j * ncolor + j];
        }
    lp.assign((size_t)ncp * ncp, 0.0);
    for (int i = 0; i < ncolor; i++)
        for (int j = 0; j <= i; j++) lp[(size_t)i * ncp + j] = (double)l[(size_t)i * ncolor + j];
    *ncp_out = ncp;
    return true;
}

cudaError_t color_sum_tf32(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                           double* d_meh, cudaStream_t st, bool tile_major);

cudaError_t color_sum_tensor(bool is_fp64, int ncolor, const void* d_cmat, const void* d_factor, const void* d_jamps,
                             long rows_padded, const RowMap& map, double* d_meh, cudaStream_t st, bool tile_major)
{
    if (!is_fp64) return color_sum_tf32(ncolor, d_factor, d_jamps, rows_padded, map, d_meh, st, tile_major);
    if (tile_major) return cudaErrorInvalidValue;
    if (!d_factor) return cudaErrorInvalidValue;
    const double* d_chol = (const double*)d_factor;
    const int ncp = (ncolor + 7) / 8 * 8;
    const int warps = 4;
    const unsigned grid = (unsigned)((rows_padded / 8 + warps - 1) / warps);
    const double* X = (const double*)d_jamps;
#define LAUNCH(NT) color_sum_dmma_kernel<NT><<<grid, warps * 32, 0, st>>>(d_chol, X, ncolor, rows_padded, map, d_meh)
    switch (ncp / 8) {
        case 1: LAUNCH(1); break;
        case 3: LAUNCH(3); break;
        case 15: LAUNCH(15); break;
        default: return cudaErrorInvalidValue;
    }
#undef LAUNCH
    return cudaGetLastError();
}

}  // namespace mg
