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

#include <type_traits>
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

// ---------------------------------------------------------------------------------------------------------
// DMMA kernel for ncolor a multiple of 24 (24, 120 colours): persistent CTAs of 16 warps, one per SM.
//   - the Cholesky factor sits in shared memory in FRAGMENT order: one 32-double block per (k-step, n-tile) pair on or
//     below the diagonal, element [lane] = L[4 ks + lane % 4][8 j + lane / 4], so that a B fragment is one conflict-free
//     LDS.64 per lane (color_cholesky_fragments);
//   - the jamps stream through a 4-stage cp.async ring of [2 parts][24 colours][64 rows] chunks (row stride 68 doubles:
//     the A-fragment reads of a half-warp, 4 rows x 4 colours, fall into 16 different bank pairs);
//   - a tile = 64 rows; warps 2 p and 2 p + 1 share the rows 8 p .. 8 p + 7 (re and im parts: two m8 tiles per B fragment)
//     and split the n-tiles between them with equal numbers of MMAs (lists TA / TB below); the k loop is fully unrolled,
//     so the triangular skipping costs no predicated issue slots;
//   - epilogue: sum of squares of the accumulators, quad reduction, the two warps of a pair meet at a named barrier.
// Issued MMAs per 8 complex rows: 2 * 240 of 2 * 450 (ncolor = 120) -- the factor 2 of the paper's triangular trick
// (PAPER.md:303, 328).
template <int NT> struct CsCfg {
    static constexpr int NC = 8 * NT, KC = 24, NCHUNK = NC / KC, ROWS = 64, RS = 68, STAGES = 4, WARPS = 16;
    static constexpr int NKS = NC / 4;                                       // k-steps
    static constexpr int STAGE_DOUBLES = 2 * KC * RS;
    __host__ __device__ static constexpr int ntile_of(int ks) { return ks / 2 + 1; }      // n-tiles with 8 j <= 4 ks + 3
    __host__ __device__ static constexpr int block_of(int ks, int j)
    {
        int o = 0;
        for (int i = 0; i < ks; i++) o += ntile_of(i);
        return o + j;
    }
    static constexpr int NBLK = block_of(NKS, 0);
    static constexpr size_t SMEM = sizeof(double) * ((size_t)NBLK * 32 + (size_t)STAGES * STAGE_DOUBLES + 2 * WARPS * 8);
    // n-tiles of the two warps of a pair: tile j costs (NT - j) k-step pairs; dealt heaviest first to the lighter warp
    __host__ __device__ static constexpr bool in_half(int j, int half)
    {
        int la = 0, lb = 0;
        bool mine = false;
        for (int t = 0; t < NT; t++) {
            const bool to_a = la <= lb;
            if (to_a) la += NT - t; else lb += NT - t;
            if (t == j) mine = (half == 0) == to_a;
        }
        return mine;
    }
    // accumulator slot of n-tile j inside its half, and the largest number of n-tiles of a half
    __host__ __device__ static constexpr int slot_of(int j, int half)
    {
        int s = 0;
        for (int t = 0; t < j; t++) s += in_half(t, half) ? 1 : 0;
        return s;
    }
    static constexpr int MAXS = slot_of(NT, 0) > slot_of(NT, 1) ? slot_of(NT, 0) : slot_of(NT, 1);
};

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void pair_barrier(int id) { asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory"); }

template <int NT, int HALF>
__device__ __forceinline__ void cs2_chunk(const double* __restrict__ Ls, const double* __restrict__ xs, int chunk, int lane,
                                          double (&acc)[CsCfg<NT>::MAXS][4])
{
    using C = CsCfg<NT>;
    const int ar = lane >> 2, ak = lane & 3;
    // this lane's A elements of the chunk: colour kk + ak, row ar (re part, then im part)
    const double* __restrict__ xa = xs + ak * C::RS + ar;
#pragma unroll
    for (int c = 0; c < C::NCHUNK; c++) {
        if (c != chunk) continue;               // (chunk is uniform; the body below is specialised per chunk)
#pragma unroll
        for (int kk = 0; kk < C::KC; kk += 4) {
            const int ks = (c * C::KC + kk) / 4;
            const double a_re = xa[kk * C::RS], a_im = xa[(C::KC + kk) * C::RS];
#pragma unroll
            for (int j = 0; j < NT; j++) {
                if (j < C::ntile_of(ks) && C::in_half(j, HALF)) {
                    const double b = Ls[C::block_of(ks, j) * 32 + lane];
                    const int sl = C::slot_of(j, HALF);          // (constant after unrolling)
                    dmma(acc[sl][0], acc[sl][1], a_re, b);
                    dmma(acc[sl][2], acc[sl][3], a_im, b);
                }
            }
        }
    }
}

template <int NT>
__global__ void __launch_bounds__(512, 1) color_sum_dmma2_kernel(const double* __restrict__ Lfrag, const double* __restrict__ X,
                                                                 long rows_padded, RowMap map, double* __restrict__ meh)
{
    using C = CsCfg<NT>;
    extern __shared__ __align__(16) double csm[];
    double* __restrict__ Ls = csm;
    double* __restrict__ Xs = Ls + (size_t)C::NBLK * 32;
    double* __restrict__ part = Xs + (size_t)C::STAGES * C::STAGE_DOUBLES;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, pair = warp >> 1, half = warp & 1;
    for (int i = tid; i < C::NBLK * 32; i += blockDim.x) Ls[i] = Lfrag[i];
    const long ntile_rows = rows_padded / C::ROWS;
    const long my_tiles = blockIdx.x < ntile_rows ? (ntile_rows - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const long nq = my_tiles * C::NCHUNK;                      // chunks this CTA streams
    auto issue = [&](long q) {                                 // chunk q -> stage q % STAGES (16-byte pieces, 1536 per chunk)
        if (q < nq) {
            const long tile = blockIdx.x + (q / C::NCHUNK) * gridDim.x;
            const int c0 = (int)(q % C::NCHUNK) * C::KC;
            double* dst = Xs + (size_t)(q % C::STAGES) * C::STAGE_DOUBLES;
            for (int pc = tid; pc < 2 * C::KC * (C::ROWS / 2); pc += 512) {
                const int seg = pc % (C::ROWS / 2), pk = pc / (C::ROWS / 2);          // pk = part * KC + colour
                const int prt = pk / C::KC, kc = pk % C::KC;
                cp_async16(dst + pk * C::RS + 2 * seg, X + ((long)prt * C::NC + c0 + kc) * rows_padded + tile * C::ROWS + 2 * seg);
            }
        }
        cp_async_commit();
    };
    for (int q = 0; q < C::STAGES - 1; q++) issue(q);
    double acc[C::MAXS][4];
#pragma unroll
    for (int j = 0; j < C::MAXS; j++) { acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.0; }
    for (long q = 0; q < nq; q++) {
        cp_async_wait<C::STAGES - 2>();
        __syncthreads();                                       // chunk q has landed; everybody is done with chunk q - 1
        issue(q + C::STAGES - 1);
        const double* xs = Xs + (size_t)(q % C::STAGES) * C::STAGE_DOUBLES + 8 * pair;
        const int chunk = (int)(q % C::NCHUNK);
        if (half == 0) cs2_chunk<NT, 0>(Ls, xs, chunk, lane, acc);
        else cs2_chunk<NT, 1>(Ls, xs, chunk, lane, acc);
        if (chunk == C::NCHUNK - 1) {
            double s = 0.0;
#pragma unroll
            for (int j = 0; j < C::MAXS; j++) {          // (a slot this half does not use stays zero)
                s += acc[j][0] * acc[j][0] + acc[j][1] * acc[j][1] + acc[j][2] * acc[j][2] + acc[j][3] * acc[j][3];
                acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.0;
            }
            s += __shfl_xor_sync(0xffffffffu, s, 1);
            s += __shfl_xor_sync(0xffffffffu, s, 2);
            if (half == 1 && (lane & 3) == 0) part[warp * 8 + (lane >> 2)] = s;
            pair_barrier(1 + pair);
            if (half == 0 && (lane & 3) == 0) {
                const long tile = blockIdx.x + (q / C::NCHUNK) * gridDim.x;
                map.store(meh, tile * C::ROWS + 8 * pair + (lane >> 2), s + part[(warp + 1) * 8 + (lane >> 2)]);
            }
        }
    }
    cp_async_wait<0>();
}

// the Cholesky factor in the fragment order of color_sum_dmma2_kernel: block (ks, j), j <= ks / 2, element [lane] =
// L[4 ks + lane % 4][8 j + lane / 4]; lp = the padded row-major factor of color_cholesky_padded
void color_cholesky_fragments(int ncp, const std::vector<double>& lp, std::vector<double>& frag)
{
    frag.clear();
    for (int ks = 0; ks < ncp / 4; ks++)
        for (int j = 0; j <= ks / 2; j++)
            for (int lane = 0; lane < 32; lane++) frag.push_back(lp[(size_t)(4 * ks + lane % 4) * ncp + 8 * j + lane / 4]);
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

// ---------------------------------------------------------------------------------------------------------
// DMMA kernel for a colour matrix that does not fit in shared memory (720 colours: g g -> t tbar g g g g, SURVEY.md §8(f)
// row 3; PAPER.md:580-613 makes this contraction the point of the 2 -> 6 process).  Same triangular form Z = X L.
//   - a CTA (16 warps) = 16 rows, their Re and Im parts: M = 32 = four m8 tiles; all 32 x NC accumulators stay in
//     registers (units of two m8 tiles x one n-tile; warp w: part w % 2, n-tiles w / 2 + 8 k);
//   - jamps AND factor stream through a 3-stage cp.async ring, 8 colours (two k-steps) per chunk: [8][32] jamps (row stride 40
//     doubles: the A-fragment reads fall into distinct bank pairs) and, per k-step, the factor's fragments of the n-tiles on or
//     below the diagonal.  The factor lives in global memory (4 MB, L2-resident) in FRAGMENT order, element [lane] of block
//     (k-step, n-tile) = L[4 ks + lane % 4][8 j + lane / 4], so that the blocks a k-step needs are ONE contiguous range and a B
//     fragment is one conflict-free LDS.64 per lane; every A fragment serves all n-tiles of the warp.
// C is only positive SEMI-definite at 6 gluons (rank 685 of 720): the factor has zero columns there (color_cholesky_big).
template <int NC>
struct CsBig {
    static constexpr int NT8 = NC / 8, NPAIR = NT8 / 2, KC = 8, NCHUNK = NC / KC, STG = 3, STRIDE = 36;   // (36 = 4 mod 16: the 16 lanes of an A-fragment load phase, 4 k x 4 rows, hit 16 different 8-byte banks; 40 gave a two-way conflict)
    static constexpr int SLOTS = (NT8 + 7) / 8;                               // n-tiles per warp: (warp / 2) + 8 k
    static constexpr size_t L_STAGE = (size_t)(KC / 4) * NT8 * 32;            // doubles: the two k-steps of a chunk, all n-tiles
    static constexpr size_t SMEM = sizeof(double) * (STG * L_STAGE + STG * KC * STRIDE + 16 * 32);
};

template <int NC>
__global__ void __launch_bounds__(512, 1) color_sum_big_kernel(const double* __restrict__ Lf, const double* __restrict__ X,
                                                               long rows_padded, RowMap map, double* __restrict__ meh)
{
    using Cfg = CsBig<NC>;
    static_assert(NC % 16 == 0, "pairs of n-tiles");
    constexpr int NT8 = Cfg::NT8, NPAIR = Cfg::NPAIR, KC = Cfg::KC, NCHUNK = Cfg::NCHUNK, STG = Cfg::STG, STRIDE = Cfg::STRIDE;
    constexpr int SLOTS = Cfg::SLOTS;
    extern __shared__ __align__(16) double sm_big[];
    double* __restrict__ ls = sm_big;                                     // [STG][KC / 4][NT8][32]: factor fragments
    double* __restrict__ js = ls + STG * Cfg::L_STAGE;                    // [STG][KC][STRIDE]: jamps
    double* __restrict__ red = js + STG * KC * STRIDE;                    // [16][32]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long r0 = (long)blockIdx.x * 16;
    // chunk c = colours 8 c .. 8 c + 7 = k-steps 2 c, 2 c + 1: the jamps (thread t < 128 copies 16 bytes: colour t / 16,
    // part (t / 8) % 2, rows 2 (t % 8) ..) and, of either k-step, the fragments of the n-tiles 0 .. c (on or below the diagonal)
    auto load_chunk = [&](int c) {
        if (c < NCHUNK) {
            const int st = c % STG;
            if (tid < 128) {
                const int k = tid >> 4, part = (tid >> 3) & 1, q = tid & 7;
                const double* src = X + ((long)part * NC + c * KC + k) * rows_padded + r0 + 2 * q;
                const unsigned dst = (unsigned)__cvta_generic_to_shared(js + ((size_t)st * KC + k) * STRIDE + part * 16 + 2 * q);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
            }
            const int n16 = (c + 1) * 16;                                // 16-byte pieces per k-step
            for (int i = tid; i < 2 * n16; i += 512) {
                const int kk = i >= n16, o = i - kk * n16;
                const double* src = Lf + ((long)(2 * c + kk) * NT8) * 32 + 2 * o;
                const unsigned dst = (unsigned)__cvta_generic_to_shared(ls + (size_t)st * Cfg::L_STAGE + (size_t)kk * NT8 * 32 + 2 * o);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
            }
        }
        asm volatile("cp.async.commit_group;");
    };
    // Work units = (n-tile, half of the M rows): warp w takes the Re part (even w) or the Im part (odd w) of the rows -- two m8
    // tiles -- and the n-tiles (w / 2) + 8 k, k = 0 .. SLOTS - 1.  At chunk c the n-tiles 0 .. c are on or below the diagonal, so
    // a warp's active tiles are a PREFIX of its slots (its length picks a branch-free body: a predicated-off DMMA still occupies
    // the tensor pipe -- measured: predication made this kernel 2x slower) and the warps' counts differ by at most one with
    // max = ceil((c + 1) / 8) units of 4 DMMAs.  (First version: units of four m8 tiles dealt in pairs (j, NT8 - 1 - j), max =
    // ceil((c + 1) / 16) units of 8 DMMAs: 8 % more tensor instructions on the critical path of the chunks.)
    double acc[SLOTS][2][2];
#pragma unroll
    for (int s = 0; s < SLOTS; s++)
#pragma unroll
        for (int m = 0; m < 2; m++) acc[s][m][0] = acc[s][m][1] = 0.0;
    const int half = warp & 1, j0 = warp >> 1;
    static_assert(SLOTS == 12, "the switch below lists 1 .. 12 active tiles");
    load_chunk(0);
    load_chunk(1);
    const int ak = lane & 3, ar = lane >> 2;
#pragma unroll 1
    for (int c = 0; c < NCHUNK; c++) {
        asm volatile("cp.async.wait_group 1;");
        __syncthreads();
        load_chunk(c + 2);
        const double* __restrict__ jt = js + (size_t)(c % STG) * KC * STRIDE + 16 * half + ar;
        const double* __restrict__ lt = ls + (size_t)(c % STG) * Cfg::L_STAGE + (size_t)j0 * 32 + lane;
        // active slots: n-tiles j0 + 8 k <= c, and < NT8
        int nact = c >= j0 ? (c - j0) / 8 + 1 : 0;
        const int nmax = (NT8 - 1 - j0) / 8 + 1;
        nact = nact < nmax ? nact : nmax;
        auto body = [&](auto NA) {
            constexpr int NACT = decltype(NA)::value;
#pragma unroll
            for (int kk = 0; kk < KC / 4; kk++) {
                const double a0 = jt[(4 * kk + ak) * STRIDE], a1 = jt[(4 * kk + ak) * STRIDE + 8];
#pragma unroll
                for (int s = 0; s < NACT; s++) {
                    const double b = lt[((size_t)kk * NT8 + 8 * s) * 32];
                    dmma(acc[s][0][0], acc[s][0][1], a0, b);
                    dmma(acc[s][1][0], acc[s][1][1], a1, b);
                }
            }
        };
        switch (nact) {
            case 1: body(std::integral_constant<int, 1>()); break;
            case 2: body(std::integral_constant<int, 2>()); break;
            case 3: body(std::integral_constant<int, 3>()); break;
            case 4: body(std::integral_constant<int, 4>()); break;
            case 5: body(std::integral_constant<int, 5>()); break;
            case 6: body(std::integral_constant<int, 6>()); break;
            case 7: body(std::integral_constant<int, 7>()); break;
            case 8: body(std::integral_constant<int, 8>()); break;
            case 9: body(std::integral_constant<int, 9>()); break;
            case 10: body(std::integral_constant<int, 10>()); break;
            case 11: body(std::integral_constant<int, 11>()); break;
            case 12: body(std::integral_constant<int, 12>()); break;
            default: break;
        }
    }
    // sum of squares per row of this warp's part: lanes of a quad hold the 8 columns of a row
#pragma unroll
    for (int m = 0; m < 2; m++) {
        double v = 0.0;
#pragma unroll
        for (int s = 0; s < SLOTS; s++) v += acc[s][m][0] * acc[s][m][0] + acc[s][m][1] * acc[s][m][1];
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        if (ak == 0) red[warp * 16 + 8 * m + ar] = v;
    }
    __syncthreads();
    if (tid < 16) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < 16; w++) v += red[w * 16 + tid];                 // Re part (even warps) + Im part (odd warps) of the row
        map.store(meh, r0 + tid, v);
    }
}

// host: factor L (row-major, lower triangular, C = L L^T) of a positive SEMI-definite integer matrix, in long double.  A pivot
// that vanishes (relative to its diagonal element) gives a zero column; the rest of that column must vanish too (it does for a
// semi-definite matrix), else false.  color_cholesky_big: the same factor in the fragment order of color_sum_big_kernel (full
// rectangle of (k-step, n-tile) blocks).
bool color_cholesky_semidef(int n, const int* cmat, std::vector<double>& L, int* rank_out)
{
    std::vector<long double> l((size_t)n * n, 0.0L);
    std::vector<char> null(n, 0);
    int rank = 0;
    for (int j = 0; j < n; j++) {
        long double s = cmat[(size_t)j * n + j];
        for (int k = 0; k < j; k++) s -= l[(size_t)j * n + k] * l[(size_t)j * n + k];
        const long double tol = 1e-10L * cmat[(size_t)j * n + j];
        if (s < -tol) return false;
        if (s <= tol) null[j] = 1; else { l[(size_t)j * n + j] = sqrtl(s); rank++; }
        for (int i = j + 1; i < n; i++) {
            long double t = cmat[(size_t)i * n + j];
            for (int k = 0; k < j; k++) t -= l[(size_t)i * n + k] * l[(size_t)j * n + k];
            if (null[j]) { if (fabsl(t) > 1e-8L * cmat[(size_t)j * n + j]) return false; }
            else l[(size_t)i * n + j] = t / l[(size_t)j * n + j];
        }
    }
    L.resize((size_t)n * n);
    for (size_t i = 0; i < L.size(); i++) L[i] = (double)l[i];
    if (rank_out) *rank_out = rank;
    return true;
}

bool color_cholesky_big(int ncolor, const int* cmat, std::vector<double>& frag, int* rank_out)
{
    if (ncolor % 16) return false;
    const int n = ncolor;
    std::vector<double> l;
    if (!color_cholesky_semidef(n, cmat, l, rank_out)) return false;
    frag.assign((size_t)(n / 4) * (n / 8) * 32, 0.0);
    for (int ks = 0; ks < n / 4; ks++)
        for (int j = 0; j < n / 8; j++)
            for (int lane = 0; lane < 32; lane++) {
                const int k = 4 * ks + lane % 4, c = 8 * j + lane / 4;
                if (k >= c) frag[((size_t)ks * (n / 8) + j) * 32 + lane] = l[(size_t)k * n + c];
            }
    return true;
}

cudaError_t color_sum_tf32_big(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                               double* d_meh, cudaStream_t st);

cudaError_t color_sum_tf32(int ncolor, const void* d_factor_img, const void* d_jamps, long rows_padded, const RowMap& map,
                           double* d_meh, cudaStream_t st, int tile_major);

cudaError_t color_sum_tensor(bool is_fp64, int ncolor, const void* d_cmat, const void* d_factor, const void* d_jamps,
                             long rows_padded, const RowMap& map, double* d_meh, cudaStream_t st, int tile_major)
{
    if (!is_fp64 && ncolor == 720)           // operand layout only (the generic diagram kernel writes it)
        return tile_major == 2 ? color_sum_tf32_big(ncolor, d_factor, d_jamps, rows_padded, map, d_meh, st) : cudaErrorInvalidValue;
    if (!is_fp64) return color_sum_tf32(ncolor, d_factor, d_jamps, rows_padded, map, d_meh, st, tile_major);
    if (tile_major) return cudaErrorInvalidValue;
    if (!d_factor) return cudaErrorInvalidValue;
    const double* d_chol = (const double*)d_factor;
    if (ncolor == 720) {            // d_factor: the fragment-order factor of color_cholesky_big
        cudaError_t e_ = cudaFuncSetAttribute(color_sum_big_kernel<720>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CsBig<720>::SMEM);
        if (e_ != cudaSuccess) return e_;
        color_sum_big_kernel<720><<<(unsigned)(rows_padded / 16), 512, CsBig<720>::SMEM, st>>>(d_chol, (const double*)d_jamps, rows_padded, map, d_meh);
        return cudaGetLastError();
    }
    const int ncp = (ncolor + 7) / 8 * 8;
    const int warps = 4;
    const unsigned grid = (unsigned)((rows_padded / 8 + warps - 1) / warps);
    const double* X = (const double*)d_jamps;
    if (ncp / 8 == 1) {
        color_sum_dmma_kernel<1><<<grid, warps * 32, 0, st>>>(d_chol, X, ncolor, rows_padded, map, d_meh);
        return cudaGetLastError();
    }
    // 24 / 120 colours: the persistent kernel; d_chol holds the row-major factor followed by its fragment-order copy
    const double* d_frag = d_chol + (size_t)ncp * ncp;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long tiles = rows_padded / 64;
    const unsigned g2 = (unsigned)(tiles < sms ? tiles : sms);
#define LAUNCH2(NT)                                                                                                       \
    {                                                                                                                     \
        cudaError_t e_ = cudaFuncSetAttribute(color_sum_dmma2_kernel<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize,    \
                                              (int)CsCfg<NT>::SMEM);                                                      \
        if (e_ != cudaSuccess) return e_;                                                                                 \
        color_sum_dmma2_kernel<NT><<<g2, 512, CsCfg<NT>::SMEM, st>>>(d_frag, X, rows_padded, map, d_meh);                 \
    }
    switch (ncp / 8) {
        case 3: LAUNCH2(3); break;
        case 15: LAUNCH2(15); break;
        default: return cudaErrorInvalidValue;
    }
#undef LAUNCH2
    return cudaGetLastError();
}

}  // namespace mg
