// color_sum_tf32.cu -- mixed/float colour sum on the 5th-generation tensor cores (tcgen05.mma kind::tf32, fp32
// accumulators in TMEM).  SURVEY.md §8(a) a5; PAPER.md:264-269 (Eq. 1), 275 and 633 (TF32 is worth 1e-4 in the
// paper's cuBLAS formulation), 330 ("one multiplication over nGoodHel*nevt rows").
//
//   me_row = A^T C A + B^T C B  (J = A + iB),  C = L L^T  (Cholesky of the integer numerators, host, long double)
//          = |A L|^2 + |B L|^2
//
// so the whole colour sum is ONE triangular GEMM Z = X L per part plus a sum of squares of the accumulator row;
// no second pass over J is needed (the paper's BLAS form needs gemm + a strided-batched dot).
// TF32 keeps 11 significand bits, which alone would cost ~5e-4 per row (SURVEY.md §8(d) "precision finding"), so
// both operands are split in two TF32 terms, X = Xh + Xl and L = Lh + Ll, and three products are accumulated
// (Xh Lh + Xl Lh + Xh Ll; the dropped Xl Ll is 2^-22 relative): fp32-level accuracy on the tensor pipe.
//
// Kernel (v1, not warp-specialised): one persistent CTA per SM, 256 threads, tiles of 128 rows.
//   smem: L image (hi, lo) resident; ring of A stages, each 128 rows x KC colours (hi, lo), K-major core matrices (no swizzle)
//   per chunk of KC colours: all threads load four colours of one row (coalesced across rows), split, store 16 B per term; one thread
//   issues the tcgen05.mma's and commits them to the stage's "empty" mbarrier; chunks run from the last colour
//   down so that the first MMA of a tile (accumulate = 0) has the full width and earlier chunks can use the
//   narrower N that the triangular L allows.  Accumulators: re part and im part, double-buffered across tiles
//   (4 x NP TMEM columns).  Epilogue: warps 0-3 read the re part, warps 4-7 the im part (tcgen05.ld 32x32b).
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <vector>

#include "color_sum.cuh"
#include "tc5.cuh"

namespace mg {

struct Tf32Cfg { int nc, KP, NP, KC, nchunks, stages; };

static bool tf32_cfg(int nc, Tf32Cfg* c)
{
    if (nc < 1 || nc > 128) return false;
    c->nc = nc;
    c->KP = (nc + 7) / 8 * 8;
    c->NP = (nc + 15) / 16 * 16;
    c->KC = c->KP % 24 == 0 ? 24 : 8;
    c->nchunks = c->KP / c->KC;
    c->stages = c->nchunks >= 3 ? 3 : (c->nchunks == 2 ? 2 : 2);
    return true;
}

// byte offset of B element (n, k) inside one B image: K-major core matrices (8 n-rows x 16 bytes),
// adjacent k-chunks 128 B apart (LBO), adjacent 8-row groups (KP/4)*128 B apart (SBO)
static inline size_t b_off(int n, int k, int KP) { return (size_t)(n % 8) * 16 + (size_t)(n / 8) * (KP / 4) * 128 + (size_t)(k / 4) * 128 + (k % 4) * 4; }

// host: the two-term TF32 image of L (C = L L^T), [hi | lo], each NP*KP floats in the layout of b_off
bool tf32_build_factor_image(int ncolor, const int* cmat, std::vector<float>& img)
{
    Tf32Cfg c;
    if (!tf32_cfg(ncolor, &c)) return false;
    std::vector<double> lp; int ncp = 0;
    if (!color_cholesky_padded(ncolor, cmat, lp, &ncp)) return false;
    const size_t per = (size_t)c.NP * c.KP;
    img.assign(2 * per, 0.0f);
    for (int k = 0; k < ncolor; k++)
        for (int n = 0; n <= k; n++) {
            const double l = lp[(size_t)k * ncp + n];           // B[n][k] = L[k][n]
            float hi = (float)l;
            uint32_t u; memcpy(&u, &hi, 4); u &= 0xFFFFE000u; memcpy(&hi, &u, 4);
            const float lo = (float)(l - (double)hi);
            const size_t o = b_off(n, k, c.KP) / 4;
            img[o] = hi; img[per + o] = lo;
        }
    return true;
}

size_t tf32_factor_image_bytes(int ncolor)
{
    Tf32Cfg c;
    return tf32_cfg(ncolor, &c) ? 2 * (size_t)c.NP * c.KP * sizeof(float) : 0;
}

struct Tf32Args {
    const float* X; const float* Bimg; double* out;
    long rows_padded;
    int nc, KP, NP, KC, nchunks, stages;
    RowMap map;
};

__global__ void __launch_bounds__(256, 1) color_sum_tf32_kernel(const Tf32Args a)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ uint64_t bar_empty[4];
    __shared__ uint64_t bar_acc[2];
    __shared__ uint32_t tmem_slot;
    __shared__ float im_part[128];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const size_t b_bytes = (size_t)a.NP * a.KP * 4;            // one B image
    const size_t a_bytes = (size_t)a.KC * 128 * 4;             // one A term of one stage
    float* Bs = reinterpret_cast<float*>(smem);
    unsigned char* As = smem + 2 * b_bytes;
    const uint32_t tcols = 4 * a.NP <= 32 ? 32 : (4 * a.NP <= 64 ? 64 : (4 * a.NP <= 128 ? 128 : (4 * a.NP <= 256 ? 256 : 512)));

    if (tid == 0) {
        for (int s = 0; s < a.stages; s++) tc5::mbar_init(&bar_empty[s], 1);
        tc5::mbar_init(&bar_acc[0], 1); tc5::mbar_init(&bar_acc[1], 1);
        tc5::mbar_fence_init();
    }
    if (warp == 0) tc5::tmem_alloc(&tmem_slot, tcols);
    // resident factor image
    {
        const float4* src = reinterpret_cast<const float4*>(a.Bimg);
        float4* dst = reinterpret_cast<float4*>(Bs);
        const int n4 = (int)(2 * b_bytes / 16);
        for (int i = tid; i < n4; i += blockDim.x) dst[i] = __ldg(src + i);
    }
    tc5::fence_async_smem();
    tc5::tc_fence_before();
    __syncthreads();
    tc5::tc_fence_after();
    const uint32_t tmem = tmem_slot;
    const uint32_t b_base = tc5::smem_u32(Bs), a_base = tc5::smem_u32(As);
    const uint32_t sbo_b = (uint32_t)(a.KP / 4) * 128, sbo_a = (uint32_t)(a.KC / 4) * 128;

    const long ntiles = a.rows_padded / 128;
    uint32_t it = 0;                 // chunk-stage uses so far (same sequence in every thread)
    uint32_t tl = 0;                 // tiles done by this CTA
    for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, tl++) {
        const long row0 = tile * 128;
        const uint32_t accbuf = tl & 1;
        for (int part = 0; part < 2; part++) {
            const uint32_t tm_d = tmem + accbuf * 2 * a.NP + part * a.NP;
            for (int ci = 0; ci < a.nchunks; ci++, it++) {
                const int c = a.nchunks - 1 - ci;                     // last colours first (full N, accumulate = 0)
                const int k0 = c * a.KC;
                const uint32_t s = it % a.stages, use = it / a.stages;
                if (use > 0) tc5::mbar_wait(&bar_empty[s], (use - 1) & 1);        // MMAs that read this stage are done
                unsigned char* st_hi = As + (size_t)s * 2 * a_bytes;
                unsigned char* st_lo = st_hi + a_bytes;
                // K-major core matrices (8 rows x 16 B): [row / 8][k / 4][row % 8][k % 4]; item = (k-quad, row): four
                // coalesced loads (one colour each, 128 consecutive rows per warp-quad), one 16-byte store per term
                const int items = (a.KC / 4) * 128;
                for (int i = tid; i < items; i += blockDim.x) {
                    const int m = i & 127, kc = i >> 7;
                    float x[4];
#pragma unroll
                    for (int j = 0; j < 4; j++) {
                        const int k = k0 + 4 * kc + j;
                        x[j] = k < a.nc ? __ldg(a.X + ((size_t)part * a.nc + k) * a.rows_padded + row0 + m) : 0.f;
                    }
                    float4 h, l;
                    h.x = __uint_as_float(__float_as_uint(x[0]) & 0xFFFFE000u); l.x = x[0] - h.x;
                    h.y = __uint_as_float(__float_as_uint(x[1]) & 0xFFFFE000u); l.y = x[1] - h.y;
                    h.z = __uint_as_float(__float_as_uint(x[2]) & 0xFFFFE000u); l.z = x[2] - h.z;
                    h.w = __uint_as_float(__float_as_uint(x[3]) & 0xFFFFE000u); l.w = x[3] - h.w;
                    const size_t o = (size_t)(m >> 3) * sbo_a + (size_t)kc * 128 + (m & 7) * 16;
                    *reinterpret_cast<float4*>(st_hi + o) = h;
                    *reinterpret_cast<float4*>(st_lo + o) = l;
                }
                tc5::fence_async_smem();
                tc5::tc_fence_before();
                __syncthreads();
                if (tid == 0) {
                    tc5::tc_fence_after();
                    int n = (k0 + a.KC + 15) / 16 * 16;
                    if (n > a.NP) n = a.NP;
                    const uint32_t idesc = tc5::idesc_tf32(n, 0, 0);
                    const uint32_t ah = a_base + (uint32_t)(s * 2 * a_bytes), al = ah + (uint32_t)a_bytes;
                    for (int ks = 0; ks < a.KC / 8; ks++) {
                        const uint64_t dah = tc5::smem_desc(ah + ks * 256, 128, sbo_a);
                        const uint64_t dal = tc5::smem_desc(al + ks * 256, 128, sbo_a);
                        const uint32_t bo = (uint32_t)((k0 / 4 + ks * 2) * 128);
                        const uint64_t dbh = tc5::smem_desc(b_base + bo, 128, sbo_b);
                        const uint64_t dbl = tc5::smem_desc(b_base + (uint32_t)b_bytes + bo, 128, sbo_b);
                        tc5::mma_tf32(tm_d, dah, dbh, idesc, (ci | ks) != 0);
                        tc5::mma_tf32(tm_d, dal, dbh, idesc, 1);
                        tc5::mma_tf32(tm_d, dah, dbl, idesc, 1);
                    }
                    tc5::mma_commit(&bar_empty[s]);
                    if (part == 1 && ci == a.nchunks - 1) tc5::mma_commit(&bar_acc[accbuf]);
                }
            }
        }
        // epilogue of this tile: sum of squares of the accumulator row
        tc5::mbar_wait(&bar_acc[accbuf], (tl >> 1) & 1);
        tc5::tc_fence_after();
        {
            const int part = warp >> 2;
            const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + accbuf * 2 * a.NP + part * a.NP;
            float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
            for (int c0 = 0; c0 < a.NP; c0 += 16) {
                float v[16];
                tc5::tmem_ld16(taddr + c0, v);
#pragma unroll
                for (int i = 0; i < 16; i += 4) {
                    s0 = fmaf(v[i], v[i], s0); s1 = fmaf(v[i + 1], v[i + 1], s1);
                    s2 = fmaf(v[i + 2], v[i + 2], s2); s3 = fmaf(v[i + 3], v[i + 3], s3);
                }
            }
            const float sum = (s0 + s1) + (s2 + s3);
            const int r = (warp & 3) * 32 + lane;
            if (part == 1) im_part[r] = sum;
            tc5::tc_fence_before();
            __syncthreads();
            if (part == 0) a.map.store(a.out, row0 + r, (double)sum + (double)im_part[r]);
        }
    }
    tc5::tc_fence_before();
    __syncthreads();
    if (warp == 0) tc5::tmem_free(tmem, tcols);
}

static size_t tf32_smem_bytes(const Tf32Cfg& c)
{
    return 2 * (size_t)c.NP * c.KP * 4 + (size_t)c.stages * 2 * c.KC * 128 * 4 + 1024;
}

cudaError_t color_sum_tf32(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                           double* d_meh, cudaStream_t st)
{
    Tf32Cfg c;
    if (!tf32_cfg(ncolor, &c) || !d_factor_img || rows_padded % 128) return cudaErrorInvalidValue;
    static int sms = 0;
    static size_t smem_set = 0;
    if (!sms) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    }
    const size_t smem = tf32_smem_bytes(c);
    if (smem > smem_set) {
        cudaError_t e = cudaFuncSetAttribute(color_sum_tf32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        smem_set = smem;
    }
    Tf32Args a;
    a.X = (const float*)d_jamps; a.Bimg = (const float*)d_factor_img; a.out = d_meh; a.rows_padded = rows_padded;
    a.nc = c.nc; a.KP = c.KP; a.NP = c.NP; a.KC = c.KC; a.nchunks = c.nchunks; a.stages = c.stages; a.map = map;
    const long ntiles = rows_padded / 128;
    // NP <= 32: several CTAs per SM would each need their TMEM columns; one per SM keeps the allocation uncontended
    const int grid = (int)(ntiles < sms ? ntiles : sms);
    color_sum_tf32_kernel<<<grid, 256, smem, st>>>(a);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------
// peak probe: back-to-back 128 x 256 x 8 kind::tf32 MMAs on every SM (operands: whatever is in shared memory)
__global__ void __launch_bounds__(128, 1) tf32_probe_kernel(int iters, float* sink)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ uint64_t bar;
    __shared__ uint32_t slot;
    const int tid = threadIdx.x;
    for (int i = tid; i < (4096 + 8192) / 4; i += blockDim.x) reinterpret_cast<float*>(smem)[i] = 1.0f;
    if (tid == 0) { tc5::mbar_init(&bar, 1); tc5::mbar_fence_init(); }
    if (tid < 32) tc5::tmem_alloc(&slot, 512);
    tc5::fence_async_smem();
    tc5::tc_fence_before();
    __syncthreads();
    tc5::tc_fence_after();
    const uint32_t tmem = slot;
    if (tid == 0) {
        const uint32_t sa = tc5::smem_u32(smem), sb = sa + 4096;
        const uint64_t da = tc5::smem_desc(sa, 128, 256);             // A: 128 rows x 8, K-major
        const uint64_t db = tc5::smem_desc(sb, 128, 256);             // B: 256 rows x 8, K-major
        const uint32_t idesc = tc5::idesc_tf32(256, 0, 0);
        for (int i = 0; i < iters; i++) {
            tc5::mma_tf32(tmem, da, db, idesc, i > 0);
            tc5::mma_tf32(tmem + 256, da, db, idesc, i > 0);
        }
        tc5::mma_commit(&bar);
    }
    tc5::mbar_wait(&bar, 0);
    tc5::tc_fence_after();
    float v[16];
    tc5::tmem_ld16(tmem + ((uint32_t)((tid >> 5) * 32) << 16), v);
    if (v[0] == -1.f) sink[0] = v[0];
    tc5::tc_fence_before();
    __syncthreads();
    if (tid < 32) tc5::tmem_free(tmem, 512);
}

cudaError_t tf32_probe(double* tflops)
{
    *tflops = 0.0;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    float* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 64);
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int iters = 20000;
    double best = 0.0;
    for (int rep = 0; rep < 3 && e == cudaSuccess; rep++) {
        cudaEventRecord(t0);
        tf32_probe_kernel<<<sms, 128, 16384>>>(iters, sink);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, t0, t1);
        const double tf = 2.0 * 128 * 256 * 8 * 2.0 * iters * sms / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(sink);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace mg
