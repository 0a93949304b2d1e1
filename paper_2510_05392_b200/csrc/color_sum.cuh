// color_sum.cuh -- stand-alone colour-sum kernels.
#pragma once
#include <cuda_runtime.h>

#include <vector>

namespace mg {

// rows of the jamps buffer are padded to the tensor kernels' row tile
inline long color_sum_padded_rows(long rows) { return (rows + 127) / 128 * 128; }

// out[r] = sum_ij (Re J_i C_ij Re J_j + Im J_i C_ij Im J_j) on the scalar ALUs, triangular form.
// d_jamps: [2][ncolor][nrows] fp64 (is_fp64) or fp32; d_cmat: [ncolor][ncolor] numerators in the same type.
cudaError_t color_sum_alu(bool is_fp64, int ncolor, const void* d_cmat, const void* d_jamps, long nrows, double* d_out,
                          cudaStream_t st);

// Tensor-core contraction.  d_jamps: [2][ncolor][rows_padded]; rows are (helicity-major, event-minor) with ne
// events per helicity; row (ih, el) goes to d_meh[ih * evt_stride + e0 + el] = norm * J^T C J.
//   fp64: DMMA (mma.sync m8n8k4 f64) on Z = X L with C = L L^T (Cholesky, lower-triangular: upper k-tiles skipped)
//   fp32: tcgen05.mma kind::tf32, exact integer C, J split in two TF32 terms, fp32 accumulation in TMEM
//   d_chol: DEVICE [ncp][ncp] padded Cholesky factor (fp64 only; see color_cholesky_padded)
cudaError_t color_sum_tensor(bool is_fp64, int ncolor, const void* d_cmat, const double* d_chol, const void* d_jamps,
                             long rows_padded, long rows_valid, int ne, int evt_stride, int e0, double norm, double* d_meh, cudaStream_t st);

// host: L with C = L L^T (lower-triangular, row-major, zero-padded to ncp = 8*ceil(ncolor/8) columns)
bool color_cholesky_padded(int ncolor, const int* cmat, std::vector<double>& lp, int* ncp_out);

// peak probes (mg_measure_peak)
cudaError_t measure_peak(int kind, double* tflops);

}  // namespace mg
