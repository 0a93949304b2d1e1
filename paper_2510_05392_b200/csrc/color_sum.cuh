// color_sum.cuh -- stand-alone colour-sum kernels.
#pragma once
#include <cuda_runtime.h>

#include <vector>

namespace mg {

// rows of the jamps buffer are padded to the tensor kernels' row tile
inline long color_sum_padded_rows(long rows) { return (rows + 127) / 128 * 128; }

// where the result of row r goes: d_out[ih * evt_stride + e0 + el] = norm * value, with (ih, el) = (helicity, event)
// of the row.  Rows are helicity-major (r = ih * ne + el; hel_minor = 0) or event-major (r = el * hel_minor + ih).
struct RowMap {
    long rows_valid = 0;
    int ne = 0;            // events per helicity block (helicity-major); 0 = identity map d_out[r]
    int hel_minor = 0;     // helicities per event (event-major) or 0
    int evt_stride = 0, e0 = 0;
    double norm = 1.0;
#if defined(__CUDACC__)
    __device__ __forceinline__ void store(double* __restrict__ out, long r, double v) const
    {
        if (r >= rows_valid) return;
        if (hel_minor > 0) { const long el = r / hel_minor; const long ih = r - el * hel_minor; out[ih * evt_stride + e0 + el] = norm * v; }
        else if (ne > 0) { const long ih = r / ne; const long el = r - ih * ne; out[ih * evt_stride + e0 + el] = norm * v; }
        else out[r] = norm * v;
    }
#endif
};

// out[r] = sum_ij (Re J_i C_ij Re J_j + Im J_i C_ij Im J_j) on the scalar ALUs, triangular form.
// d_jamps: [2][ncolor][nrows] fp64 (is_fp64) or fp32; d_cmat: [ncolor][ncolor] numerators in the same type.
cudaError_t color_sum_alu(bool is_fp64, int ncolor, const void* d_cmat, const void* d_jamps, long nrows, double* d_out,
                          cudaStream_t st, const RowMap* map = nullptr);

// Tensor-core contraction.  d_jamps: [2][ncolor][rows_padded]; row r goes where `map` says, times map.norm.
//   fp64: DMMA (mma.sync m8n8k4 f64) on Z = X L with C = L L^T (Cholesky, lower-triangular: upper k-tiles skipped)
//   fp32: tcgen05.mma kind::tf32 on Z = X L, X and L split in two TF32 terms (3 products), fp32 accumulation in TMEM
//   d_factor: DEVICE Cholesky factor of C: fp64 [ncp][ncp] padded (color_cholesky_padded), or the two-term TF32
//             image of it (tf32_build_factor_image) for fp32
cudaError_t color_sum_tensor(bool is_fp64, int ncolor, const void* d_cmat, const void* d_factor, const void* d_jamps,
                             long rows_padded, const RowMap& map, double* d_meh, cudaStream_t st, int tile_major = 0);
// tile_major (fp32 only): 1: d_jamps is [rows_padded / 128][2][ncolor][128] instead of [2][ncolor][rows_padded];
// 2: the tcgen05 operand layout, TF32-rounded by the producer (color_sum_tf32.cu "direct": no converter warps, two products)

// host: L with C = L L^T (lower-triangular, row-major, zero-padded to ncp = 8*ceil(ncolor/8) columns)
bool color_cholesky_padded(int ncolor, const int* cmat, std::vector<double>& lp, int* ncp_out);
// host: the same factor in the fragment order of the persistent DMMA kernel (color_sum.cu); the device image handed to
// color_sum_tensor as d_factor in MG_FP64 is lp followed by frag
void color_cholesky_fragments(int ncp, const std::vector<double>& lp, std::vector<double>& frag);

// host: factor of the (positive semi-definite) 720 x 720 matrix in the fragment order of the large-matrix DMMA kernel
bool color_cholesky_big(int ncolor, const int* cmat, std::vector<double>& frag, int* rank_out);
// host: the row-major factor itself (zero columns at null pivots)
bool color_cholesky_semidef(int n, const int* cmat, std::vector<double>& L, int* rank_out);
// host: TF32 image [hi | lo] of that factor, slice by slice in the order color_sum_tf32_big_kernel consumes it (720 colours)
bool tf32_big_build_factor_image(int ncolor, const int* cmat, std::vector<float>& img);

// host: two-term TF32 image [hi | lo] of the Cholesky factor in the tcgen05 shared-memory layout (color_sum_tf32.cu)
bool tf32_build_factor_image(int ncolor, const int* cmat, std::vector<float>& img);

// peak probes (mg_measure_peak)
cudaError_t measure_peak(int kind, double* tflops);

}  // namespace mg
