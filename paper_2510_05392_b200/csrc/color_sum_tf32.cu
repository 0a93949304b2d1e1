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
// Kernel: one persistent CTA per SM, warp-specialised, tiles of 128 rows, chunks of KC colours.
//   warp 0      TMA producer: cp.async.bulk into a ring of raw fp32 stages, completion counted on the stage's "raw full"
//               mbarrier.  Tile-major jamps ([row / 128][2][nc][128], written so by the helicity-shared kernel): ONE
//               bulk copy of KC x 512 B per chunk; plain [2][nc][rows] jamps (mg_color_sum): one 512-B copy per colour
//   warp 1      MMA issuer: per chunk 3 x KC/8 tcgen05.mma (M = 128, N = the width the triangular L needs for this
//               chunk), tcgen05.commit to the A stage's "empty" barrier and, after a tile's last chunk, to "acc full"
//   warp 2      TMEM allocation / release
//   warps 4-7   epilogue: tcgen05.ld of the re and im accumulator rows, sum of squares, store (TMEM lane quarter = warp % 4)
//   warps 8-15  converters: raw stage -> hi/lo TF32 terms in the K-major no-swizzle core-matrix layout of the A ring
//   Chunks run from the last colour down: the first MMA of a tile (accumulate = 0) has the full width.
//   Accumulators (re, im) are double-buffered across tiles (4 x NP TMEM columns).
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <vector>

#include "color_sum.cuh"
#include "tc5.cuh"

namespace mg {

struct Tf32Cfg { int nc, KP, NP, KC, nchunks, raw_stages, a_stages; };

static bool tf32_cfg(int nc, Tf32Cfg* c)
{
    if (nc < 1 || nc > 128) return false;
    c->nc = nc;
    c->KP = (nc + 7) / 8 * 8;
    c->NP = (nc + 15) / 16 * 16;
    c->KC = c->KP % 24 == 0 ? 24 : 8;
    c->nchunks = c->KP / c->KC;
    c->raw_stages = 5; c->a_stages = 3;
    return true;
}

// width of the accumulator columns that chunk c (colours [c KC, (c+1) KC)) touches: L is lower triangular
static inline int chunk_n(const Tf32Cfg& c, int chunk)
{
    int n = ((chunk + 1) * c.KC + 15) / 16 * 16;
    return n > c.NP ? c.NP : n;
}
// float offset of chunk c inside one factor image: chunk c holds chunk_n rows x KC colours
static inline size_t chunk_off(const Tf32Cfg& c, int chunk)
{
    size_t o = 0;
    for (int i = 0; i < chunk; i++) o += (size_t)chunk_n(c, i) * c.KC;
    return o;
}
// byte offset of element (n, kk) inside a chunk: K-major core matrices (8 n-rows x 16 bytes), adjacent k-quads 128 B
// apart (LBO), adjacent 8-row groups (KC / 4) * 128 B apart (SBO)
static inline size_t b_off(int n, int kk, int KC) { return (size_t)(n % 8) * 16 + (size_t)(n / 8) * (KC / 4) * 128 + (size_t)(kk / 4) * 128 + (kk % 4) * 4; }

// host: the two-term TF32 image of L (C = L L^T), [hi | lo], chunk by chunk, each chunk in the layout of b_off
bool tf32_build_factor_image(int ncolor, const int* cmat, std::vector<float>& img)
{
    Tf32Cfg c;
    if (!tf32_cfg(ncolor, &c)) return false;
    std::vector<double> lp; int ncp = 0;
    if (!color_cholesky_padded(ncolor, cmat, lp, &ncp)) return false;
    const size_t per = chunk_off(c, c.nchunks);
    img.assign(2 * per, 0.0f);
    for (int k = 0; k < ncolor; k++)
        for (int n = 0; n <= k; n++) {
            const double l = lp[(size_t)k * ncp + n];           // B[n][k] = L[k][n]
            float hi = (float)l;
            uint32_t u; memcpy(&u, &hi, 4); u &= 0xFFFFE000u; memcpy(&hi, &u, 4);
            const float lo = (float)(l - (double)hi);
            const int chunk = k / c.KC;
            const size_t o = chunk_off(c, chunk) + b_off(n, k % c.KC, c.KC) / 4;
            img[o] = hi; img[per + o] = lo;
        }
    return true;
}

struct Tf32Args {
    const float* X; const float* Bimg; double* out;
    long rows_padded;
    int nc, KP, NP, KC, nchunks, raw_stages, a_stages;
    int tile_major;                // jamps as [row / 128][2][nc][128]: one bulk copy per chunk
    int b_floats;                  // floats of one factor image
    int chunk_off[8], chunk_n[8];  // per chunk: float offset inside an image, accumulator width
    RowMap map;
};

constexpr int TF32_THREADS = 512;
constexpr int TF32_MAX_RAW = 8;
constexpr int TF32_MAX_A = 12;

template <bool DIRECT>
__global__ void __launch_bounds__(TF32_THREADS, 1) color_sum_tf32_kernel(const Tf32Args a)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    __shared__ uint64_t raw_full[TF32_MAX_RAW], raw_empty[TF32_MAX_RAW];
    __shared__ uint64_t a_full[TF32_MAX_A], a_empty[TF32_MAX_A], acc_full[2], acc_empty[2];
    __shared__ uint32_t tmem_slot;
    __shared__ uint64_t tab_b[8][2];          // per chunk: descriptors of its slice of L_hi / L_lo (MMA issuer)
    __shared__ uint32_t tab_id[8];            // per chunk: instruction descriptor (accumulator width)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const size_t b_bytes = (size_t)a.b_floats * 4;             // one factor image
    const size_t a_bytes = (size_t)a.KC * 128 * 4;             // one A term of one stage = one raw stage
    float* Bs = reinterpret_cast<float*>(smem);
    unsigned char* As = smem + 2 * b_bytes;                    // [a_stages][hi | lo]
    // direct mode (tile_major = 2): the A ring holds one TF32 term per stage and takes the raw ring's space as well --
    // the ring depth is what hides the HBM latency (3 stages: 2.3 TB/s, 11 stages: measured in profiles/)
    constexpr bool direct = DIRECT;            // (a.tile_major == 2)
    const int R = a.raw_stages, NA = direct ? (2 * a.a_stages + a.raw_stages < TF32_MAX_A ? 2 * a.a_stages + a.raw_stages : TF32_MAX_A) : a.a_stages;
    const size_t a_stride = direct ? a_bytes : 2 * a_bytes;   // bytes per A stage
    unsigned char* Rs = As + (size_t)2 * a.a_stages * a_bytes; // [raw_stages][KC][128] fp32 (not in direct mode)
    const uint32_t tcols = 4 * a.NP <= 32 ? 32 : (4 * a.NP <= 64 ? 64 : (4 * a.NP <= 128 ? 128 : (4 * a.NP <= 256 ? 256 : 512)));

    if (tid == 0) {
        for (int s = 0; s < R; s++) { tc5::mbar_init(&raw_full[s], 1); tc5::mbar_init(&raw_empty[s], 8); }
        for (int s = 0; s < NA; s++) { tc5::mbar_init(&a_full[s], direct ? 1 : 8); tc5::mbar_init(&a_empty[s], 1); }
        for (int s = 0; s < 2; s++) { tc5::mbar_init(&acc_full[s], direct ? 2 : 1); tc5::mbar_init(&acc_empty[s], 4); }
        tc5::mbar_fence_init();
        // per chunk: descriptors of its slice of L_hi / L_lo and the instruction descriptor (read by the MMA issuers)
        const uint32_t b_base = tc5::smem_u32(Bs), sbo0 = (uint32_t)(a.KC / 4) * 128;
        for (int c = 0; c < a.nchunks; c++) {
            tab_b[c][0] = tc5::smem_desc(b_base + (uint32_t)a.chunk_off[c] * 4, 128, sbo0);
            tab_b[c][1] = tc5::smem_desc(b_base + (uint32_t)a.chunk_off[c] * 4 + (uint32_t)b_bytes, 128, sbo0);
            tab_id[c] = tc5::idesc_tf32(a.chunk_n[c], 0, 0);
        }
    }
    if (warp == 2) tc5::tmem_alloc(&tmem_slot, tcols);
    {   // resident factor image
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
    const long ntiles = a.rows_padded / 128;
    const int cpt = 2 * a.nchunks;                             // chunks per tile (re part, then im part)

    if (warp == 0 && direct) {
        // ---- TMA producer, direct: the jamps are already TF32 values in the operand layout: one 12 KB bulk copy per chunk
        //      straight into the A ring (no raw ring, no converters, no low term of X) ----
        if (lane == 0) {
            uint32_t sa = 0, ph = 1;                 // stage and the parity to wait for (no division in this loop)
            for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                const float* xt = a.X + (size_t)tile * (256 * a.nc);
                for (int c = a.nchunks - 1; c >= 0; c--)
                    for (int part = 0; part < 2; part++) {             // re, im alternate: one MMA-issuing thread each
                        tc5::mbar_wait(&a_empty[sa], ph);
                        tc5::mbar_arrive_expect_tx(&a_full[sa], (uint32_t)a_bytes);
                        tc5::tma_load_1d(As + (size_t)sa * a_stride, xt + ((size_t)part * a.nc + c * a.KC) * 128, (uint32_t)a_bytes, &a_full[sa]);
                        if (++sa == (uint32_t)NA) { sa = 0; ph ^= 1; }
                    }
            }
        }
        __syncwarp();
    } else if (warp == 0) {
        // ---- TMA producer: lane 0 waits for the stage and posts the byte count, then lane kk copies colour kk ----
        uint32_t q = 0;
        for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const long row0 = tile * 128;
            for (int j = 0; j < cpt; j++, q++) {
                const int part = j / a.nchunks, c = a.nchunks - 1 - j % a.nchunks;
                const int k0 = c * a.KC;
                const uint32_t s = q % R;
                int nk = a.nc - k0;
                if (nk > a.KC) nk = a.KC;
                if (lane == 0) {
                    tc5::mbar_wait(&raw_empty[s], ((q / R) & 1) ^ 1);
                    tc5::mbar_arrive_expect_tx(&raw_full[s], (uint32_t)nk * 512u);
                }
                __syncwarp();
                float* dst = reinterpret_cast<float*>(Rs + (size_t)s * a_bytes);
                if (a.tile_major) {
                    if (lane == 0)
                        tc5::tma_load_1d(dst, a.X + (size_t)tile * (256 * a.nc) + ((size_t)part * a.nc + k0) * 128, (uint32_t)nk * 512u, &raw_full[s]);
                } else if (lane < nk)
                    tc5::tma_load_1d(dst + lane * 128, a.X + ((size_t)part * a.nc + k0 + lane) * a.rows_padded + row0, 512u, &raw_full[s]);
            }
        }
        __syncwarp();
    } else if (warp == 1 || (direct && warp == 3)) {
        // ---- MMA issuer(s).  Each is ONE thread: nothing but waits, descriptor additions and the MMAs may be in its loop (the
        //      first version divided by nchunks and by the ring depth per chunk and rebuilt every descriptor: 10 us per tile).
        //      Direct mode has two of them, warp 1 for the re part and warp 3 for the im part (independent accumulator
        //      columns, alternate stages of the ring): the issue rate of one thread was the limit of the kernel ----
        if (lane == 0) {
            const int me = warp == 3 ? 1 : 0;
            const uint32_t a_base = tc5::smem_u32(As);
            const uint32_t sbo = (uint32_t)(a.KC / 4) * 128;
            const int nks = a.KC / 8;
            const uint32_t ks_step = 256 >> 4;                       // one k-step (two core-matrix columns) in descriptor units
            const uint64_t da0 = tc5::smem_desc(a_base, 128, sbo);
            const uint32_t a_step = (uint32_t)(a_stride >> 4), al_off = (uint32_t)(a_bytes >> 4);
            const uint32_t adv = direct ? 2 : 1;                     // stages per chunk of this thread
            uint32_t sa = direct ? me : 0, ph = 0, tl = 0;
            for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, tl++) {
                const uint32_t buf = tl & 1;
                tc5::mbar_wait(&acc_empty[buf], ((tl >> 1) & 1) ^ 1);
                tc5::tc_fence_after();
                for (int part = direct ? me : 0; part < (direct ? me + 1 : 2); part++) {
                    const uint32_t tm_d = tmem + buf * 2 * a.NP + part * a.NP;
                    for (int ci = 0; ci < a.nchunks; ci++) {
                        const int c = a.nchunks - 1 - ci;
                        const uint64_t bh = tab_b[c][0], bl = tab_b[c][1];
                        const uint32_t id = tab_id[c];
                        const uint64_t dah = da0 + a_step * sa;
                        tc5::mbar_wait(&a_full[sa], ph);
                        tc5::tc_fence_after();
                        for (int ks = 0; ks < nks; ks++) {
                            tc5::mma_tf32(tm_d, dah + ks_step * ks, bh + ks_step * ks, id, (ci | ks) != 0);
                            if (!direct) tc5::mma_tf32(tm_d, dah + al_off + ks_step * ks, bh + ks_step * ks, id, 1);
                            tc5::mma_tf32(tm_d, dah + ks_step * ks, bl + ks_step * ks, id, 1);
                        }
                        tc5::mma_commit(&a_empty[sa]);
                        sa += adv;
                        if (sa >= (uint32_t)NA) { sa -= NA; ph ^= 1; }
                    }
                }
                tc5::mma_commit(&acc_full[buf]);
            }
        }
        __syncwarp();
    } else if (warp >= 4 && warp < 8) {
        // ---- epilogue ----
        uint32_t tl = 0;
        const int r = (warp & 3) * 32 + lane;
        for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, tl++) {
            const uint32_t buf = tl & 1;
            tc5::mbar_wait(&acc_full[buf], (tl >> 1) & 1);
            tc5::tc_fence_after();
            const uint32_t taddr = tmem + ((uint32_t)((warp & 3) * 32) << 16) + buf * 2 * a.NP;
            float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
            for (int c0 = 0; c0 < 2 * a.NP; c0 += 16) {
                float v[16];
                tc5::tmem_ld16(taddr + c0, v);
#pragma unroll
                for (int i = 0; i < 16; i += 4) {
                    s0 = fmaf(v[i], v[i], s0); s1 = fmaf(v[i + 1], v[i + 1], s1);
                    s2 = fmaf(v[i + 2], v[i + 2], s2); s3 = fmaf(v[i + 3], v[i + 3], s3);
                }
            }
            tc5::tc_fence_before();
            __syncwarp();
            if (lane == 0) tc5::mbar_arrive(&acc_empty[buf]);
            a.map.store(a.out, tile * 128 + r, (double)s0 + (double)s1 + ((double)s2 + (double)s3));
        }
    } else if (warp >= 8 && !direct) {
        // ---- converters: 8 warps; thread = (row m of the tile, half of the chunk's colour quads) ----
        const int m = (tid - 256) & 127, half = (tid - 256) >> 7;
        const int nq = a.KC / 4, q0 = half * nq / 2, q1 = (half + 1) * nq / 2;
        const uint32_t sbo = (uint32_t)(a.KC / 4) * 128;
        uint32_t q = 0;
        for (long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            for (int j = 0; j < cpt; j++, q++) {
                const int c = a.nchunks - 1 - j % a.nchunks;
                int nk = a.nc - c * a.KC;
                if (nk > a.KC) nk = a.KC;
                const uint32_t s = q % R, sa = q % NA;
                tc5::mbar_wait(&raw_full[s], (q / R) & 1);
                tc5::mbar_wait(&a_empty[sa], ((q / NA) & 1) ^ 1);
                const float* src = reinterpret_cast<const float*>(Rs + (size_t)s * a_bytes) + m;
                unsigned char* st_hi = As + (size_t)sa * 2 * a_bytes + (size_t)(m >> 3) * sbo + (m & 7) * 16;
                unsigned char* st_lo = st_hi + a_bytes;
                for (int kc = q0; kc < q1; kc++) {
                    float x[4];
#pragma unroll
                    for (int i = 0; i < 4; i++) x[i] = 4 * kc + i < nk ? src[(4 * kc + i) * 128] : 0.f;
                    float4 h, l;
                    h.x = __uint_as_float(__float_as_uint(x[0]) & 0xFFFFE000u); l.x = x[0] - h.x;
                    h.y = __uint_as_float(__float_as_uint(x[1]) & 0xFFFFE000u); l.y = x[1] - h.y;
                    h.z = __uint_as_float(__float_as_uint(x[2]) & 0xFFFFE000u); l.z = x[2] - h.z;
                    h.w = __uint_as_float(__float_as_uint(x[3]) & 0xFFFFE000u); l.w = x[3] - h.w;
                    *reinterpret_cast<float4*>(st_hi + kc * 128) = h;
                    *reinterpret_cast<float4*>(st_lo + kc * 128) = l;
                }
                tc5::fence_async_smem();
                __syncwarp();
                if (lane == 0) { tc5::mbar_arrive(&a_full[sa]); tc5::mbar_arrive(&raw_empty[s]); }
            }
        }
    }
    tc5::tc_fence_before();
    __syncthreads();
    if (warp == 2) tc5::tmem_free(tmem, tcols);
}

static size_t tf32_smem_bytes(const Tf32Cfg& c)
{
    return 2 * chunk_off(c, c.nchunks) * 4 + (size_t)(2 * c.a_stages + c.raw_stages) * c.KC * 128 * 4 + 1024;
}

cudaError_t color_sum_tf32(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                           double* d_meh, cudaStream_t st, int tile_major)
{
    Tf32Cfg c;
    if (tile_major == 2 && ncolor % 24 != 0) return cudaErrorInvalidValue;
    if (!tf32_cfg(ncolor, &c) || !d_factor_img || rows_padded % 128 || c.nchunks > 8 || c.a_stages > 4 || c.raw_stages > TF32_MAX_RAW)
        return cudaErrorInvalidValue;
    // per call, for the CURRENT device: the attribute is per device and a process may hold handles on several
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t smem = tf32_smem_bytes(c);
    {
        cudaError_t e = cudaFuncSetAttribute(color_sum_tf32_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(color_sum_tf32_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    Tf32Args a;
    a.X = (const float*)d_jamps; a.Bimg = (const float*)d_factor_img; a.out = d_meh; a.rows_padded = rows_padded;
    a.nc = c.nc; a.KP = c.KP; a.NP = c.NP; a.KC = c.KC; a.nchunks = c.nchunks; a.raw_stages = c.raw_stages; a.a_stages = c.a_stages; a.map = map; a.tile_major = tile_major;
    a.b_floats = (int)chunk_off(c, c.nchunks);
    for (int i = 0; i < 8; i++) { a.chunk_off[i] = i < c.nchunks ? (int)chunk_off(c, i) : 0; a.chunk_n[i] = i < c.nchunks ? chunk_n(c, i) : 0; }
    const long ntiles = rows_padded / 128;
    const int grid = (int)(ntiles < sms ? ntiles : sms);      // one CTA per SM: each owns its TMEM columns
    if (tile_major == 2) color_sum_tf32_kernel<true><<<grid, TF32_THREADS, smem, st>>>(a);
    else color_sum_tf32_kernel<false><<<grid, TF32_THREADS, smem, st>>>(a);
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
