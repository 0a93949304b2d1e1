// color_sum_tf32_big.cu -- mixed-precision colour sum of g g -> t tbar g g g g (720 colour flows) on the 5th-generation tensor
// cores: tcgen05.mma kind::tf32, fp32 accumulators in TMEM.  SURVEY.md §8(f) row 3; PAPER.md:580-613 (Table 8: the colour sum
// of the 2 -> 6 process as a BLAS / TF32 contraction), 264-269 (Eq. 1).
//
// Same form as color_sum_tf32.cu: me_row = |A L|^2 + |B L|^2 with C = L L^T (semi-definite at 6 gluons: zero columns, DESIGN.md
// A16), jamps TF32-rounded by the diagram kernel and stored in the operand layout, L split in two TF32 terms (J Lhi + J Llo).
// What changes at 720 colours: neither the factor (2 x 2 MB) nor a tile's accumulators (2 x 720 fp32 columns; TMEM has 512)
// fit on chip, so the contraction is tiled in N and K:
//   - a tile = 128 rows; three PASSES over column blocks of 240 (accumulators: re at TMEM columns 0-239, im at 256-495);
//   - a pass runs the 24-colour chunks from the last one down to the block's diagonal (L is lower triangular: chunks above it
//     contribute nothing; the chunks that cross the diagonal use a narrower MMA); 30 + 20 + 10 = 60 steps per tile;
//   - a step's operands travel through a 3-stage ring, ONE mbarrier per stage: the factor's (block, chunk) slice, 240 x 24 hi
//     and lo terms, prepared on the host in the K-major core-matrix layout and in consumption order (one 46 KB bulk copy,
//     L2-resident: 2.8 MB in all), and the chunk's re and im jamps (12 KB each, one bulk copy each);
//   - warp 0: TMA producer; warps 1 and 3: one MMA-issuing thread each (re / im part: 6 MMAs 128 x N x 8 per step);
//     warp 2: TMEM allocation; warps 4-7: epilogue per pass (tcgen05.ld, sum of squares kept in registers over the passes).
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <vector>

#include "color_sum.cuh"
#include "tc5.cuh"

namespace mg {

namespace {
constexpr int BN = 240, KC = 24, NC = 720, NBLK = NC / BN, NCHUNK = NC / KC, CPB = BN / KC;     // 3 blocks, 30 chunks, 10 chunks per block
constexpr int NSTEP = 60;                                    // sum over blocks of (NCHUNK - CPB * block)
constexpr int B_TERM = BN * KC * 4;                          // bytes of one term of a factor slice
constexpr int A_PART = 128 * KC * 4;                         // bytes of one part of a jamps chunk
constexpr int STAGE = 2 * B_TERM + 2 * A_PART;               // 70 656 B
constexpr int NSTAGE = 3;
constexpr int THREADS = 256;

inline size_t b_off(int n, int kk) { return (size_t)(n % 8) * 16 + (size_t)(n / 8) * (KC / 4) * 128 + (size_t)(kk / 4) * 128 + (kk % 4) * 4; }
inline int step_width(int blk, int chunk)
{
    int w = (KC * (chunk - CPB * blk + 1) + 15) / 16 * 16;
    return w > BN ? BN : w;
}
}  // namespace

struct Tf32BigArgs {
    const float* X; const unsigned char* Bimg; double* out;
    long rows_padded;
    RowMap map;
};

__global__ void __launch_bounds__(THREADS, 1) color_sum_tf32_big_kernel(const Tf32BigArgs a)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ uint64_t full[NSTAGE], empty[NSTAGE], acc_full, acc_empty;
    __shared__ uint32_t tmem_slot;
    __shared__ uint32_t tab_id[NSTEP];        // instruction descriptor per step (accumulator width)
    __shared__ uint16_t tab_chunk[NSTEP];     // chunk of the step

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < NSTAGE; s++) { tc5::mbar_init(&full[s], 1); tc5::mbar_init(&empty[s], 2); }
        tc5::mbar_init(&acc_full, 2);
        tc5::mbar_init(&acc_empty, 4);
        tc5::mbar_fence_init();
        int st = 0;
        for (int blk = 0; blk < NBLK; blk++)
            for (int c = NCHUNK - 1; c >= CPB * blk; c--, st++) {
                int w = (KC * (c - CPB * blk + 1) + 15) / 16 * 16;
                if (w > BN) w = BN;
                tab_id[st] = tc5::idesc_tf32(w, 0, 0);
                tab_chunk[st] = (uint16_t)c;
            }
    }
    if (warp == 2) tc5::tmem_alloc(&tmem_slot, 512);
    tc5::tc_fence_before();
    __syncthreads();
    tc5::tc_fence_after();
    const uint32_t tmem = tmem_slot;
    const long ntiles = a.rows_padded / 128;

    if (warp == 0) {
        // ---- TMA producer ----
        if (lane == 0) {
            uint32_t s = 0, ph = 1;
            for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const float* xt = a.X + (size_t)tile * (256 * NC);
                for (int st = 0; st < NSTEP; st++) {
                    const int c = tab_chunk[st];
                    unsigned char* dst = smem + (size_t)s * STAGE;
                    tc5::mbar_wait(&empty[s], ph);
                    tc5::mbar_arrive_expect_tx(&full[s], (uint32_t)STAGE);
                    tc5::tma_load_1d(dst, a.Bimg + (size_t)st * (2 * B_TERM), (uint32_t)(2 * B_TERM), &full[s]);
                    tc5::tma_load_1d(dst + 2 * B_TERM, xt + (size_t)(c * KC) * 128, (uint32_t)A_PART, &full[s]);
                    tc5::tma_load_1d(dst + 2 * B_TERM + A_PART, xt + (size_t)(NC + c * KC) * 128, (uint32_t)A_PART, &full[s]);
                    if (++s == NSTAGE) { s = 0; ph ^= 1; }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1 || warp == 3) {
        // ---- MMA issuers: warp 1 the re part, warp 3 the im part (independent accumulator columns, the same stages) ----
        if (lane == 0) {
            const int part = warp == 3 ? 1 : 0;
            const uint32_t base = tc5::smem_u32(smem);
            const uint32_t sbo = (uint32_t)(KC / 4) * 128, ks_step = 256 >> 4;
            const uint32_t tm_d = tmem + part * 256;
            uint32_t s = 0, ph = 0, pass = 0;
            for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                int st = 0;
                for (int blk = 0; blk < NBLK; blk++, pass++) {
                    tc5::mbar_wait(&acc_empty, (pass & 1) ^ 1);
                    tc5::tc_fence_after();
                    const int nst = NCHUNK - CPB * blk;
                    for (int i = 0; i < nst; i++, st++) {
                        const uint32_t id = tab_id[st];
                        const uint32_t sb = base + s * STAGE;
                        const uint64_t bh = tc5::smem_desc(sb, 128, sbo), bl = tc5::smem_desc(sb + B_TERM, 128, sbo);
                        const uint64_t da = tc5::smem_desc(sb + 2 * B_TERM + part * A_PART, 128, sbo);
                        tc5::mbar_wait(&full[s], ph);
                        tc5::tc_fence_after();
#pragma unroll
                        for (int ks = 0; ks < KC / 8; ks++) {
                            tc5::mma_tf32(tm_d, da + ks_step * ks, bh + ks_step * ks, id, (i | ks) != 0);
                            tc5::mma_tf32(tm_d, da + ks_step * ks, bl + ks_step * ks, id, 1);
                        }
                        tc5::mma_commit(&empty[s]);
                        if (++s == NSTAGE) { s = 0; ph ^= 1; }
                    }
                    tc5::mma_commit(&acc_full);
                }
            }
        }
        __syncwarp();
    } else if (warp >= 4) {
        // ---- epilogue: per pass the sum of squares of this row's 240 re and 240 im accumulators ----
        const int r = (warp & 3) * 32 + lane;
        const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16);
        uint32_t pass = 0;
        for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            double tot = 0.0;
            for (int blk = 0; blk < NBLK; blk++, pass++) {
                tc5::mbar_wait(&acc_full, pass & 1);
                tc5::tc_fence_after();
                float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
                for (int part = 0; part < 2; part++)
                    for (int c0 = 0; c0 < BN; c0 += 16) {
                        float v[16];
                        tc5::tmem_ld16(taddr + part * 256 + c0, v);
#pragma unroll
                        for (int i = 0; i < 16; i += 4) {
                            s0 = fmaf(v[i], v[i], s0); s1 = fmaf(v[i + 1], v[i + 1], s1);
                            s2 = fmaf(v[i + 2], v[i + 2], s2); s3 = fmaf(v[i + 3], v[i + 3], s3);
                        }
                    }
                tc5::tc_fence_before();
                __syncwarp();
                if (lane == 0) tc5::mbar_arrive(&acc_empty);
                tot += (double)s0 + (double)s1 + ((double)s2 + (double)s3);
            }
            a.map.store(a.out, tile * 128 + r, tot);
        }
    }
    tc5::tc_fence_before();
    __syncthreads();
    if (warp == 2) tc5::tmem_free(tmem, 512);
}

// host: the factor (C = L L^T, zero columns at null pivots) as two TF32 terms, slice by slice in the order the kernel
// consumes them: for block b = 0..2, chunk c = 29 .. 10 b: [hi | lo], each 240 x 24 in the K-major core-matrix layout
// (B[n][k] = L[24 c + k][240 b + n])
bool tf32_big_build_factor_image(int ncolor, const int* cmat, std::vector<float>& img)
{
    if (ncolor != NC) return false;
    std::vector<double> L;
    int rank = 0;
    if (!color_cholesky_semidef(ncolor, cmat, L, &rank)) return false;
    img.assign((size_t)NSTEP * 2 * B_TERM / 4, 0.0f);
    int st = 0;
    for (int blk = 0; blk < NBLK; blk++)
        for (int c = NCHUNK - 1; c >= CPB * blk; c--, st++) {
            float* hi = img.data() + (size_t)st * (2 * B_TERM / 4);
            float* lo = hi + B_TERM / 4;
            for (int n = 0; n < BN; n++)
                for (int kk = 0; kk < KC; kk++) {
                    const int k = KC * c + kk, col = BN * blk + n;
                    if (col > k) continue;
                    const double l = L[(size_t)k * ncolor + col];
                    float h = (float)l;
                    uint32_t u; memcpy(&u, &h, 4); u &= 0xFFFFE000u; memcpy(&h, &u, 4);
                    hi[b_off(n, kk) / 4] = h;
                    lo[b_off(n, kk) / 4] = (float)(l - (double)h);
                }
        }
    return st == NSTEP;
}

// d_jamps: the tcgen05 operand layout written by the generic diagram kernel (tile_major = 2, TF32-rounded)
cudaError_t color_sum_tf32_big(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                               double* d_meh, cudaStream_t st)
{
    if (ncolor != NC || !d_factor_img || rows_padded % 128) return cudaErrorInvalidValue;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t smem = (size_t)NSTAGE * STAGE + 1024;
    cudaError_t e = cudaFuncSetAttribute(color_sum_tf32_big_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    Tf32BigArgs a;
    a.X = (const float*)d_jamps; a.Bimg = (const unsigned char*)d_factor_img; a.out = d_meh; a.rows_padded = rows_padded; a.map = map;
    const long ntiles = rows_padded / 128;
    const int grid = (int)(ntiles < sms ? ntiles : sms);      // one CTA per SM: each owns all 512 TMEM columns
    color_sum_tf32_big_kernel<<<grid, THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace mg
