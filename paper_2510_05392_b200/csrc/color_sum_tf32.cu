// color_sum_tf32.cu -- mixed/float colour sum on the 5th-generation tensor cores (tcgen05, kind::tf32).
// (first version: placeholder that reports "not supported"; the tcgen05 kernel follows)
#include "color_sum.cuh"

namespace mg {

cudaError_t color_sum_tf32(int, const void*, const void*, long, const RowMap&, double*, cudaStream_t)
{
    return cudaErrorNotSupported;
}

cudaError_t tf32_probe(double* tflops)
{
    *tflops = 0.0;
    return cudaErrorNotSupported;
}

}  // namespace mg
