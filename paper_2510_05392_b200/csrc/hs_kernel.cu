// hs_kernel.cu -- helicity-shared diagram kernel: one CTA = one event; interprets the tables of
// gen/co_program.py (layout: hs_tables.h) and the record streams hs_create builds from them.
//
// Why this shape on B200: the paper keeps one thread per (event, helicity) and lets every helicity
// recompute every wavefunction, with up to 121 wavefunctions + 120 jamps of per-thread state (PAPER.md:101-119, 141,
// 187) -- 12 KB per thread, i.e. local-memory traffic.  Here the state that depends on few helicities lives once per
// event in shared memory (<= 8 variants per object; phase 1), the vertices are contracted with all branches but the
// largest once per variant (phase 2, work units handed to warps dynamically), and the per-helicity work is a stream of
// 4-component complex dot products evaluated for all helicities at once on the FP64 tensor path (phase 3).  Every
// jamp is finished on chip and written once, coalesced, to the jamps buffer, rows ordered (event, helicity).
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include <vector>

#include "helas.cuh"
#include "hs_kernel.cuh"

namespace mg {

struct HsDev {
    const int4* obj; const int4* term; const int* p1_items; const int* legset_mask; const int4* group;
    const int4* xobj; const int* x_items; const int4* sigma; const int4* entry; const unsigned short* vtab;
    const unsigned char* hdep;
    const uint4* p3tab; int maxe;                // phase-3 stream: [colour flow][entry k < maxe][lane] records
    const uint4* p2tab; int maxt;                // phase-2 stream: [unit][term k < maxt][lane] records (built in hs_create)
    int npar, ncolor, ngroups, obj_area, stage_area, nlegsets;
    int nw3;               // jamp accumulators = colour flows per group (phase 3 on the FP64 tensor path); 0 = scalar phase 3
    int p1_level[4];
};

// variant of an argument object: bit j = bit ((code >> 3j) & 7) of the parent's variant (7 = none; variants are < 128)
__device__ __forceinline__ int sub_variant(int var, int code)
{
    return ((var >> (code & 7)) & 1) | (((var >> ((code >> 3) & 7)) & 1) << 1) | (((var >> ((code >> 6) & 7)) & 1) << 2);
}

// Shared-memory layout of an area: 64-byte blocks, block b = (object offset / 4 + variant) holds the 4 components of one
// variant as 16-byte complex numbers, the component index XOR-swizzled with bits 1-2 of the BLOCK index:
//     slot(off, var, c) = 4 b + (c ^ ((b >> 1) & 3)),   b = off / 4 + var      (offsets are multiples of 8 slots)
// Eight consecutive variants of one component (phases 1, 2: lane <-> variant) and the 2 variants x 4 components of a
// DMMA fragment quarter-warp (phase 3) both fall into eight different 16-byte bank groups.  Using the block index
// (not the variant) lets a precomputed block number address an argument without knowing its object (argument table).
__device__ __forceinline__ int slot(int off, int var, int c)
{
    const int b = (off >> 2) + var;
    return 4 * b + (c ^ ((b >> 1) & 3));
}

__device__ __forceinline__ void load_blk(const double2* __restrict__ area, int b, wf<double>& w)
{
    const char* p = reinterpret_cast<const char*>(area) + b * 64;
    const int sw = (b & 6) << 3;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const double2 v = *reinterpret_cast<const double2*>(p + ((c * 16) ^ sw));
        w.c[c].re = v.x; w.c[c].im = v.y;
    }
}

__device__ __forceinline__ void load_obj(const double2* __restrict__ area, int off, int var, wf<double>& w)
{
    load_blk(area, (off >> 2) + var, w);
}

__device__ __forceinline__ void store_obj(double2* __restrict__ area, int off, int var, const wf<double>& w)
{
#pragma unroll
    for (int c = 0; c < 4; c++) area[slot(off, var, c)] = make_double2(w.c[c].re, w.c[c].im);
}

__device__ __forceinline__ p4<double> load_k(const double* __restrict__ Ks, int ls)
{
    p4<double> k = { Ks[4 * ls], Ks[4 * ls + 1], Ks[4 * ls + 2], Ks[4 * ls + 3] };
    return k;
}

__device__ __forceinline__ void lower(wf<double>& w)
{
#pragma unroll
    for (int c = 1; c < 4; c++) { w.c[c].re = -w.c[c].re; w.c[c].im = -w.c[c].im; }
}

// both orderings of the four-gluon vertex that share the middle leg: (x y | z out) + (z y | x out)
//   J = 2 (X.Z) Y - (Y.Z) X - (Y.X) Z      (raw vertex, no propagator factor)
template <typename T> __device__ __forceinline__ void v4s_raw(const wf<T>& X, const wf<T>& Y, const wf<T>& Z, wf<T>& out)
{
    cx<T> xz = dot(X, Z);
    xz = xz + xz;
    const cx<T> yz = dot(Y, Z), yx = dot(Y, X);
    for (int mu = 0; mu < 4; mu++) out.c[mu] = cfms(yx, Z.c[mu], cfms(yz, X.c[mu], xz * Y.c[mu]));
}

// argument of a term: word = offset in the area (16 bits) | sub-variant code (9 bits) << 16
__device__ __forceinline__ void load_arg(const double2* __restrict__ area, int word, int var, wf<double>& w)
{
    load_obj(area, word & 0xFFFF, sub_variant(var, (word >> 16) & 0x1FF), w);
}

// Sum of the terms [t0, t0 + nt) for helicity variant `var` of an object whose leg set has total momentum K(ls_out).
// Inlined at its two call sites (phases 1 and 2) so that the accumulator stays in registers; the next term's table
// word is fetched while the current one is evaluated.
// PRE (phase 2): the block numbers of the three arguments of (this lane's item, term t) come precomputed from the
// argument table `at` (entry t * 32; built on the host in hs_create), which removes the per-lane variant gather.
template <bool PRE>
__device__ __forceinline__ void run_terms(const HsDev& d, const double2* __restrict__ area, const double* __restrict__ Ks,
                                          const double* __restrict__ pm, int t0, int nt, int var, int ls_out, double mt,
                                          double wt, wf<double>& acc, const uint2* __restrict__ at = nullptr)
{
#pragma unroll
    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
    int4 w = __ldg(d.term + t0);
    uint2 aw = make_uint2(0u, 0u);
    if (PRE) aw = __ldg(at);
    for (int t = 0; t < nt; t++) {
        const int tn = t + 1 < nt ? t + 1 : t;
        const int4 wn = __ldg(d.term + t0 + tn);
        uint2 awn = make_uint2(0u, 0u);
        if (PRE) awn = __ldg(at + 32 * tn);
        const int op = w.x & 0xFF, neg = (w.x >> 8) & 1;
        wf<double> r;
        if (op <= 2) {
            const int hel = (var & 1) ? 1 : -1;
            const double* p = pm + 4 * w.y;
            if (op == 0) ext_eps(p, hel, w.y >= 2, r);
            else if (op == 1) ext_ubar(p, mt, hel, r);
            else ext_v(p, mt, hel, r);
        } else {
            wf<double> A, B;
            if (PRE) { load_blk(area, aw.x & 0xFFFF, A); load_blk(area, aw.x >> 16, B); }
            else { load_arg(area, w.y, var, A); load_arg(area, w.z, var, B); }
            switch (op) {
                case 3: v3_off(A, load_k(Ks, (w.x >> 16) & 0xFF), B, load_k(Ks, (w.x >> 24) & 0xFF), 1.0 / m2(load_k(Ks, ls_out)), r); break;
                case 11: v3_raw(A, load_k(Ks, (w.x >> 16) & 0xFF), B, load_k(Ks, (w.x >> 24) & 0xFF), r); lower(r); break;
                case 13: { wf<double> Z; load_arg(area, w.w, var, Z); v4s_raw(A, B, Z, r); lower(r); break; }
                case 4: case 12: {
                    wf<double> Z;
                    if (PRE) load_blk(area, aw.y, Z);
                    else load_arg(area, w.w, var, Z);
                    if (op == 4) v4_off(A, B, Z, 1.0 / m2(load_k(Ks, ls_out)), r);
                    else { v4_raw(A, B, Z, r); lower(r); }
                    break;
                }
                case 5: { const p4<double> K = load_k(Ks, ls_out); ffv_l(A, B, -K, mt, inv_prop(m2(K), mt, wt), r); break; }
                case 6: { const p4<double> K = load_k(Ks, ls_out); ffv_r(A, B, K, mt, inv_prop(m2(K), mt, wt), r); break; }
                case 7: ffv_p(A, B, 1.0 / m2(load_k(Ks, ls_out)), r); break;
                case 8: row_slash(A, make_slashed(B), r); break;
                case 9: slash_col(make_slashed(A), B, r); break;
                default: ffv_p_raw(A, B, r); lower(r); break;       // 10: x_bil
            }
        }
        const double sg = neg ? -1.0 : 1.0;
#pragma unroll
        for (int c = 0; c < 4; c++) { acc.c[c].re = fma(sg, r.c[c].re, acc.c[c].re); acc.c[c].im = fma(sg, r.c[c].im, acc.c[c].im); }
        w = wn;
        aw = awn;
    }
}

// Phase-2 record of (work unit, term k, lane), built on the host from the tables (hs_create):
//   x = block of argument A | block of argument B << 16      (shared-memory block = offset / 4 + variant)
//   y = block of argument C | block of the item's own result in the staging area << 16
//   z = opcode | negative << 8 | leg set of A << 16 | leg set of B << 24;  opcode 0xFF = this lane has no term k
//   w = number of terms of the unit (largest over its lanes)
// The address depends on the unit number only, so the next unit's first record is fetched while this one is evaluated.
__device__ __forceinline__ void eval_x_term(const double2* __restrict__ area, const double* __restrict__ Ks, const uint4 e,
                                            wf<double>& acc)
{
    const int op = e.z & 0xFF;
    if (op == 0xFF) return;
    const double sg = ((e.z >> 8) & 1) ? -1.0 : 1.0;
    // the accumulation is repeated in every case (no merge of the per-case result registers), and the index lowering of
    // the raw vertices (components 1-3 negated) is folded into its sign
    auto add = [&](const wf<double>& r, double s123) {
        acc.c[0].re = fma(sg, r.c[0].re, acc.c[0].re); acc.c[0].im = fma(sg, r.c[0].im, acc.c[0].im);
#pragma unroll
        for (int c = 1; c < 4; c++) { acc.c[c].re = fma(s123, r.c[c].re, acc.c[c].re); acc.c[c].im = fma(s123, r.c[c].im, acc.c[c].im); }
    };
    wf<double> A, B, r;
    load_blk(area, e.x & 0xFFFF, A);
    load_blk(area, e.x >> 16, B);
    switch (op) {
        case 11: v3_raw(A, load_k(Ks, (e.z >> 16) & 0xFF), B, load_k(Ks, (e.z >> 24) & 0xFF), r); add(r, -sg); break;
        case 12: { wf<double> Z; load_blk(area, e.y & 0xFFFF, Z); v4_raw(A, B, Z, r); add(r, -sg); break; }
        case 13: { wf<double> Z; load_blk(area, e.y & 0xFFFF, Z); v4s_raw(A, B, Z, r); add(r, -sg); break; }
        case 8: row_slash(A, make_slashed(B), r); add(r, sg); break;
        case 9: slash_col(make_slashed(A), B, r); add(r, sg); break;
        default: ffv_p_raw(A, B, r); add(r, -sg); break;                 // 10: x_bil
    }
}

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// accumulator slot of helicity combination h (gen/co_program.py acc_swizzle)
__device__ __forceinline__ int acc_swizzle(int h)
{
    const int hi = h >> 3;
    return h ^ (((hi & 1) * 3) ^ (((hi >> 1) & 1) * 5) ^ (((hi >> 2) & 1) * 6) ^ (((hi >> 3) & 1) * 7));
}

// Phase 3 on the FP64 tensor path (DMMA, mma.sync.m8n8k4.f64): ONE warp evaluates one dot entry for all 2^npar
// helicity combinations.  With hx/hy the variants of X/Y, the entry is the complex product sum
//     out[hx][hy] = sum_c X_c[hx] * Y_c[hy]      (c = 4 components)
// i.e. a real GEMM  [nvx x 8] . [8 x 2 nvy]:  A = [Re X | Im X],  B = [Re Y, Im Y ; -Im Y, Re Y]  (columns (hy, re/im)).
// A-fragment lane (row r = lane/4, k = lane%4) reads X_k[8 mt + r] once (16 bytes: the k-step 0 and k-step 1 values),
// B-fragment lane (k = lane%4, col = lane/4) reads Y_k[4 nt + col/2]; the C fragment of a lane is the complex number
// (hx = 8 mt + lane/4, hy = 4 nt + lane%4).  Operand traffic per entry: <= 6 LDS.128 per lane instead of 8 per
// helicity.  Entries of one colour flow have different leg partitions, so the fragments are added into a per-warp
// accumulator in shared memory indexed by the helicity combination (swizzled; tables hdep) and the finished jamp is
// written once, coalesced over helicities.
// Phase-3 record of (colour flow, entry k, lane), built on the host (hs_create); everything a lane needs is
// precomputed so that an entry costs few integer instructions (a warp with phase-3 work runs almost alone on its
// scheduler, so its time is instructions x dependent latency):
//   x = 16-byte slot of X variant (lane / 4), component (lane % 4), m-tile 0 (m-tile mt adds 32 slots: same swizzle)
//       | slot of Y variant (lane / 8), n-tile 0 << 16
//   y = slot of Y, n-tile 1 | shape << 16 | negative << 18 | number of entries of the flow << 24
//       shape 0: (MT, NT) = (4, 1), 1: (2, 2), 2: (2, 1), 3: (1, 2)
//   z = accumulator slots of this lane's complex number in tiles 0..3, one byte each (tile t = mt * NT + nt)
//   w = jamp index of the flow
// The FP64 MMA has a dependent-issue latency of ~200 cycles on B200 (measured; a DFMA has ~10), so the two k-steps of
// a tile go to SEPARATE accumulators: f[4 t + {0,1}] = sum_c Re X (Re Y | Im Y), f[4 t + {2,3}] = sum_c Im X (Im Y | Re Y),
// re = f[4t] - f[4t+2], im = f[4t+1] + f[4t+3]  (no negated operand, no select: a lane loads its 8-byte halves directly).
template <int MT, int NT>
__device__ __forceinline__ void p3_issue(const double2* __restrict__ stage, const double2* __restrict__ area, const uint4 e,
                                         int o0, double (&f)[16])
{
    const double2* __restrict__ xp = stage + (e.x & 0xFFFF);
    double2 xa[MT];
    double b0[NT], b1[NT];
#pragma unroll
    for (int mt = 0; mt < MT; mt++) xa[mt] = xp[32 * mt];
#pragma unroll
    for (int nt = 0; nt < NT; nt++) {
        const char* yp = reinterpret_cast<const char*>(area + (nt == 0 ? (e.x >> 16) : (e.y & 0xFFFF)));
        b0[nt] = *reinterpret_cast<const double*>(yp + o0);           // odd column (im out): Im Y, even: Re Y
        b1[nt] = *reinterpret_cast<const double*>(yp + (8 - o0));     // odd column: Re Y, even: Im Y
    }
#pragma unroll
    for (int i = 0; i < 16; i++) f[i] = 0.0;
#pragma unroll
    for (int mt = 0; mt < MT; mt++)
#pragma unroll
        for (int nt = 0; nt < NT; nt++) {
            const int t = mt * NT + nt;
            dmma884(f[4 * t], f[4 * t + 1], xa[mt].x, b0[nt]);
            dmma884(f[4 * t + 2], f[4 * t + 3], xa[mt].y, b1[nt]);
        }
}

// add the fragments of one entry into the flow's accumulator (all loads first: the slots of one entry are distinct)
template <int NTILE>
__device__ __forceinline__ void p3_update(const uint4 e, const double (&f)[16], double2* __restrict__ acc, bool first)
{
    const double sgn = ((e.y >> 18) & 1) ? -1.0 : 1.0;
    double2 v[NTILE];
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        v[t] = make_double2(0.0, 0.0);
        if (!first) v[t] = acc[(e.z >> (8 * t)) & 0xFF];
    }
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        v[t].x = fma(sgn, f[4 * t] - f[4 * t + 2], v[t].x);
        v[t].y = fma(sgn, f[4 * t + 1] + f[4 * t + 3], v[t].y);
        acc[(e.z >> (8 * t)) & 0xFF] = v[t];
    }
}

__device__ __forceinline__ void p3_entry(const double2* __restrict__ stage, const double2* __restrict__ area, const uint4 e,
                                         int o0, double2* __restrict__ acc, bool first)
{
    double f[16];
    switch ((e.y >> 16) & 3) {
        case 0: p3_issue<4, 1>(stage, area, e, o0, f); p3_update<4>(e, f, acc, first); break;
        case 1: p3_issue<2, 2>(stage, area, e, o0, f); p3_update<4>(e, f, acc, first); break;
        case 2: p3_issue<2, 1>(stage, area, e, o0, f); p3_update<2>(e, f, acc, first); break;
        default: p3_issue<1, 2>(stage, area, e, o0, f); p3_update<2>(e, f, acc, first); break;
    }
}

template <typename T2>
__device__ __forceinline__ void phase3_dmma(const HsDev& d, const HsLaunch& a, const double2* __restrict__ area,
                                            const double2* __restrict__ stage, double2* __restrict__ accs, int e, const int4 g0,
                                            const int4 g1, int* ctr, int lane)
{
    const int nh = 1 << d.npar;
    const int o0 = ((lane >> 2) & 1) * 8;                  // B-fragment column parity: which 8-byte half of Y is k-step 0
    const size_t sstride = (size_t)d.maxe * 32;
    const uint4* __restrict__ tab = d.p3tab + (size_t)g0.w * sstride + lane;
    // colour flows of the group are handed to the warps dynamically; flow s owns accumulator s (g1.x <= nw3)
    int s = 0;
    if (lane == 0) s = atomicAdd(ctr, 1);
    s = __shfl_sync(0xffffffffu, s, 0);
    uint4 cur = make_uint4(0u, 0u, 0u, 0u);
    if (s < g1.x) cur = __ldg(tab + s * sstride);
    while (s < g1.x) {
        int sn = 0;                                         // next flow and its first record, fetched early
        if (lane == 0) sn = atomicAdd(ctr, 1);
        sn = __shfl_sync(0xffffffffu, sn, 0);
        uint4 nxt = make_uint4(0u, 0u, 0u, 0u);
        if (sn < g1.x) nxt = __ldg(tab + sn * sstride);
        double2* __restrict__ acc = accs + (s << d.npar);
        const uint4* __restrict__ p = tab + s * sstride;
        const int nent = (int)(cur.y >> 24), jamp = (int)cur.w;
        const long long tp0 = a.prof ? clock64() : 0;
        int posr[4];                                        // rows of this lane's helicity combinations (write-out below)
#pragma unroll
        for (int j = 0; j < 4; j++) posr[j] = lane + 32 * j < nh ? a.d_pos[lane + 32 * j] : -1;
        // records are fetched three entries ahead: the L2 latency of the record stream under load (~1000+ cycles,
        // measured with MG_HS_PROFILE) is several entry times
        uint4 en = cur;
        uint4 enn = __ldg(p + 32 * (nent > 1 ? 1 : 0));
        uint4 en2 = __ldg(p + 32 * (nent > 2 ? 2 : nent - 1));
        for (int k = 0; k < nent; k++) {
            const uint4 en3 = __ldg(p + 32 * (k + 3 < nent ? k + 3 : nent - 1));
            p3_entry(stage, area, en, o0, acc, k == 0);
            __syncwarp();
            en = enn; enn = en2; en2 = en3;
        }
        const long long tp1 = a.prof ? clock64() : 0;
        // the finished jamp of this colour flow, all helicity combinations
        T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
#pragma unroll
        for (int j = 0; j < 4; j++) {
            const int h = lane + 32 * j, pos = posr[j];
            if (pos >= 0) {
                const double2 v = acc[acc_swizzle(h)];
                const size_t row = (size_t)e * a.nrow_evt + pos;
                if (a.tile_major) {
                    T2* __restrict__ o = out + (row >> 7) * (size_t)(256 * d.ncolor) + (size_t)jamp * 128 + (row & 127);
                    o[0] = T2(v.x); o[(size_t)d.ncolor * 128] = T2(v.y);
                } else {
                    out[(size_t)jamp * a.rows + row] = T2(v.x);
                    out[(size_t)(d.ncolor + jamp) * a.rows + row] = T2(v.y);
                }
            }
        }
        __syncwarp();
        if (a.prof && lane == 0) { atomicAdd(a.prof + 6, (unsigned long long)(tp1 - tp0)); atomicAdd(a.prof + 7, (unsigned long long)(clock64() - tp1)); }
        s = sn; cur = nxt;
    }
}

// T2 = type of the jamps buffer (double: MG_FP64, float: MG_MIXED -- PAPER.md:122 "FPTYPE=m")
// blockDim.x = 2^npar * nsplit: thread = (sigma split s, helicity combination h)
template <typename T2>
__global__ void __launch_bounds__(256) hs_diagrams_kernel(const HsDev d, const HsLaunch a)
{
    extern __shared__ double2 sm[];
    __shared__ int ctr[2];                            // work-unit counters of phases 2 and 3
    if (threadIdx.x < 2) ctr[threadIdx.x] = 0;
    double2* __restrict__ area = sm;
    double2* __restrict__ stage = sm + d.obj_area;
    double2* __restrict__ accs = stage + d.stage_area;
    double* __restrict__ Ks = reinterpret_cast<double*>(accs + (d.nw3 << d.npar));
    double* __restrict__ pm = Ks + 4 * d.nlegsets;
    const int tid = threadIdx.x, nth = blockDim.x;
    const int nh = 1 << d.npar;
    const int h = tid & (nh - 1), split = tid >> d.npar, nsplit = nth >> d.npar;
    const int pos = a.d_pos[h];                       // row of this helicity inside the event, -1 = not a good helicity
    long long tprof = a.prof ? clock64() : 0;
#define HS_PROF(i) do { if (a.prof && tid == 0) { const long long t_ = clock64(); atomicAdd(a.prof + (i), (unsigned long long)(t_ - tprof)); tprof = t_; } } while (0)
    for (int e = blockIdx.x; e < a.nevt; e += gridDim.x) {
        // a0: momenta (AOS fp64) -> shared; leg-set momenta in the all-incoming convention
        for (int i = tid; i < 4 * d.npar; i += nth) pm[i] = a.mom[(size_t)e * (4 * d.npar) + i];
        __syncthreads();
        for (int s = tid; s < d.nlegsets; s += nth) {
            const int m = __ldg(d.legset_mask + s);
            double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
            for (int p = 0; p < d.npar; p++)
                if ((m >> p) & 1) {
                    const double sg = p < 2 ? 1.0 : -1.0;
                    k0 += sg * pm[4 * p]; k1 += sg * pm[4 * p + 1]; k2 += sg * pm[4 * p + 2]; k3 += sg * pm[4 * p + 3];
                }
            Ks[4 * s] = k0; Ks[4 * s + 1] = k1; Ks[4 * s + 2] = k2; Ks[4 * s + 3] = k3;
        }
        __syncthreads();
        HS_PROF(0);
        // phase 1: objects, level by level
        for (int lvl = 0; lvl < 3; lvl++) {
            for (int i = d.p1_level[lvl] + tid; i < d.p1_level[lvl + 1]; i += nth) {
                const int it = __ldg(d.p1_items + i);
                const int4 o = __ldg(d.obj + (it >> 8));
                const int var = it & 0xFF;
                wf<double> acc;
                run_terms<false>(d, area, Ks, pm, o.z, o.w, var, o.y >> 8, a.mt, a.wt, acc);
                store_obj(area, o.x, var, acc);
            }
            __syncthreads();
        }
        HS_PROF(1);
        const size_t row = (size_t)e * a.nrow_evt + pos;
        for (int g = 0; g < d.ngroups; g++) {
            const int4 g0 = __ldg(d.group + 2 * g), g1 = __ldg(d.group + 2 * g + 1);
            // phase 2: pair objects of this group; work units of 32 (pair object, variant) items with the same term
            // shape are handed to the warps dynamically, most expensive first (gen/co_program.py)
            {
                const int lane = tid & 31, nunits = g0.z >> 5;
                const size_t ustride = (size_t)d.maxt * 32;
                const uint4* __restrict__ tab = d.p2tab + (size_t)(g0.y >> 5) * ustride + lane;
                int u = 0;
                if (lane == 0) u = atomicAdd(&ctr[0], 1);
                u = __shfl_sync(0xffffffffu, u, 0);
                uint4 cur = make_uint4(0u, 0u, 0xFFu, 0u);
                if (u < nunits) cur = __ldg(tab + u * ustride);
                while (u < nunits) {
                    int un = 0;                                 // next unit and its first record, fetched early
                    if (lane == 0) un = atomicAdd(&ctr[0], 1);
                    un = __shfl_sync(0xffffffffu, un, 0);
                    uint4 nxt = make_uint4(0u, 0u, 0xFFu, 0u);
                    if (un < nunits) nxt = __ldg(tab + un * ustride);
                    const uint4* __restrict__ p = tab + u * ustride;
                    const int ntm = (int)cur.w;
                    wf<double> acc;
#pragma unroll
                    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
                    uint4 en = cur;                             // records are fetched three terms ahead (L2 latency under load)
                    uint4 enn = __ldg(p + 32 * (ntm > 1 ? 1 : 0));
                    uint4 en2 = __ldg(p + 32 * (ntm > 2 ? 2 : ntm - 1));
                    for (int k = 0; k < ntm; k++) {
                        const uint4 en3 = __ldg(p + 32 * (k + 3 < ntm ? k + 3 : ntm - 1));
                        eval_x_term(area, Ks, en, acc);
                        en = enn; enn = en2; en2 = en3;
                    }
                    if ((cur.z & 0xFF) != 0xFF) {
                        const int bs = (int)(cur.y >> 16);
                        const int sw = (bs >> 1) & 3;
#pragma unroll
                        for (int c = 0; c < 4; c++) stage[4 * bs + (c ^ sw)] = make_double2(acc.c[c].re, acc.c[c].im);
                    }
                    u = un; cur = nxt;
                }
            }
            HS_PROF(2);
            __syncthreads();
            HS_PROF(3);
            if (tid == 0) ctr[0] = 0;                 // every warp has left the loop above; next use is after the barrier below
            // phase 3: the jamps of this group, one colour flow at a time
            if (d.nw3 > 0) {
                phase3_dmma<T2>(d, a, area, stage, accs, e, g0, g1, &ctr[1], tid & 31);
            } else if (pos >= 0) {
                for (int s = split; s < g1.x; s += nsplit) {
                    const int4 sg = __ldg(d.sigma + g0.w + s);
                    double re = 0.0, im = 0.0;
#pragma unroll 2
                    for (int k = 0; k < sg.z; k++) {
                        const int4 en = __ldg(d.entry + sg.y + k);
                        const int vv = __ldg(d.vtab + en.z * nh + h);
                        const int vx = vv & 0xFF, vy = vv >> 8;
                        const int xoff = en.x & 0xFFFF, yoff = en.y & 0xFFFF;
                        double tr = 0.0, ti = 0.0;
#pragma unroll
                        for (int c = 0; c < 4; c++) {
                            const double2 x = stage[slot(xoff, vx, c)], y = area[slot(yoff, vy, c)];
                            tr = fma(x.x, y.x, tr); tr = fma(-x.y, y.y, tr);
                            ti = fma(x.x, y.y, ti); ti = fma(x.y, y.x, ti);
                        }
                        const double sgn = (double)en.w;
                        re = fma(sgn, tr, re); im = fma(sgn, ti, im);
                    }
                    T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
                    if (a.tile_major) {
                        T2* __restrict__ o = out + (row >> 7) * (size_t)(256 * d.ncolor) + (size_t)sg.x * 128 + (row & 127);
                        o[0] = T2(re); o[(size_t)d.ncolor * 128] = T2(im);
                    } else {
                        out[(size_t)sg.x * a.rows + row] = T2(re);
                        out[(size_t)(d.ncolor + sg.x) * a.rows + row] = T2(im);
                    }
                }
            }
            HS_PROF(4);
            __syncthreads();
            HS_PROF(5);
            if (tid == 0) ctr[1] = 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// Overlapped variant (hs_phase3 = 2): ONE 512-thread CTA per SM with a double-buffered staging area.  Phase 3 of group g
// (few, long, latency-bound colour-flow units) and phase 2 of group g + 1 (many short units) are drawn from ONE work
// queue, so that no warp idles while the colour flows of a group are finished; one barrier per group instead of two.
__device__ __forceinline__ void p2_unit(const HsDev& d, const double2* __restrict__ area, double2* __restrict__ stagew,
                                        const double* __restrict__ Ks, const int4 g0, int u, int lane)
{
    const size_t ustride = (size_t)d.maxt * 32;
    const uint4* __restrict__ p = d.p2tab + ((size_t)(g0.y >> 5) + u) * ustride + lane;
    const uint4 cur = __ldg(p);
    const int ntm = (int)cur.w;
    wf<double> acc;
#pragma unroll
    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
    uint4 en = cur;
    uint4 enn = __ldg(p + 32 * (ntm > 1 ? 1 : 0));
    uint4 en2 = __ldg(p + 32 * (ntm > 2 ? 2 : ntm - 1));
    for (int k = 0; k < ntm; k++) {
        const uint4 en3 = __ldg(p + 32 * (k + 3 < ntm ? k + 3 : ntm - 1));
        eval_x_term(area, Ks, en, acc);
        en = enn; enn = en2; en2 = en3;
    }
    if ((cur.z & 0xFF) != 0xFF) {
        const int bs = (int)(cur.y >> 16);
        const int sw = (bs >> 1) & 3;
#pragma unroll
        for (int c = 0; c < 4; c++) stagew[4 * bs + (c ^ sw)] = make_double2(acc.c[c].re, acc.c[c].im);
    }
}

template <typename T2>
__device__ __forceinline__ void p3_flow(const HsDev& d, const HsLaunch& a, const double2* __restrict__ area,
                                        const double2* __restrict__ stager, double2* __restrict__ accs, int e, const int4 g0,
                                        int s, int lane)
{
    const int nh = 1 << d.npar;
    const int o0 = ((lane >> 2) & 1) * 8;
    const uint4* __restrict__ p = d.p3tab + ((size_t)g0.w + s) * ((size_t)d.maxe * 32) + lane;
    double2* __restrict__ acc = accs + (s << d.npar);
    const uint4 cur = __ldg(p);
    const int nent = (int)(cur.y >> 24), jamp = (int)cur.w;
    int posr[4];
#pragma unroll
    for (int j = 0; j < 4; j++) posr[j] = lane + 32 * j < nh ? a.d_pos[lane + 32 * j] : -1;
    uint4 en = cur;
    uint4 enn = __ldg(p + 32 * (nent > 1 ? 1 : 0));
    uint4 en2 = __ldg(p + 32 * (nent > 2 ? 2 : nent - 1));
    for (int k = 0; k < nent; k++) {
        const uint4 en3 = __ldg(p + 32 * (k + 3 < nent ? k + 3 : nent - 1));
        p3_entry(stager, area, en, o0, acc, k == 0);
        __syncwarp();
        en = enn; enn = en2; en2 = en3;
    }
    T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
#pragma unroll
    for (int j = 0; j < 4; j++) {
        const int h = lane + 32 * j, pos = posr[j];
        if (pos >= 0) {
            const double2 v = acc[acc_swizzle(h)];
            const size_t row = (size_t)e * a.nrow_evt + pos;
            if (a.tile_major) {
                T2* __restrict__ o = out + (row >> 7) * (size_t)(256 * d.ncolor) + (size_t)jamp * 128 + (row & 127);
                o[0] = T2(v.x); o[(size_t)d.ncolor * 128] = T2(v.y);
            } else {
                out[(size_t)jamp * a.rows + row] = T2(v.x);
                out[(size_t)(d.ncolor + jamp) * a.rows + row] = T2(v.y);
            }
        }
    }
    __syncwarp();
}

template <typename T2>
__global__ void __launch_bounds__(512, 1) hs_overlap_kernel(const HsDev d, const HsLaunch a)
{
    extern __shared__ double2 sm[];
    __shared__ int ctr;
    if (threadIdx.x == 0) ctr = 0;
    double2* __restrict__ area = sm;
    double2* __restrict__ stage0 = sm + d.obj_area;
    double2* __restrict__ stage1 = stage0 + d.stage_area;
    double2* __restrict__ accs = stage1 + d.stage_area;
    double* __restrict__ Ks = reinterpret_cast<double*>(accs + (d.nw3 << d.npar));
    double* __restrict__ pm = Ks + 4 * d.nlegsets;
    const int tid = threadIdx.x, nth = blockDim.x, lane = tid & 31;
    auto grab = [&]() { int u = 0; if (lane == 0) u = atomicAdd(&ctr, 1); return __shfl_sync(0xffffffffu, u, 0); };
    for (int e = blockIdx.x; e < a.nevt; e += gridDim.x) {
        for (int i = tid; i < 4 * d.npar; i += nth) pm[i] = a.mom[(size_t)e * (4 * d.npar) + i];
        __syncthreads();
        for (int s = tid; s < d.nlegsets; s += nth) {
            const int m = __ldg(d.legset_mask + s);
            double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
            for (int p = 0; p < d.npar; p++)
                if ((m >> p) & 1) {
                    const double sg = p < 2 ? 1.0 : -1.0;
                    k0 += sg * pm[4 * p]; k1 += sg * pm[4 * p + 1]; k2 += sg * pm[4 * p + 2]; k3 += sg * pm[4 * p + 3];
                }
            Ks[4 * s] = k0; Ks[4 * s + 1] = k1; Ks[4 * s + 2] = k2; Ks[4 * s + 3] = k3;
        }
        __syncthreads();
        for (int lvl = 0; lvl < 3; lvl++) {
            for (int i = d.p1_level[lvl] + tid; i < d.p1_level[lvl + 1]; i += nth) {
                const int it = __ldg(d.p1_items + i);
                const int4 o = __ldg(d.obj + (it >> 8));
                const int var = it & 0xFF;
                wf<double> acc;
                run_terms<false>(d, area, Ks, pm, o.z, o.w, var, o.y >> 8, a.mt, a.wt, acc);
                store_obj(area, o.x, var, acc);
            }
            __syncthreads();
        }
        // prologue: pair objects of group 0
        {
            const int4 g0 = __ldg(d.group);
            const int nu = g0.z >> 5;
            for (int u = grab(); u < nu; u = grab()) p2_unit(d, area, stage0, Ks, g0, u, lane);
        }
        __syncthreads();
        if (tid == 0) ctr = 0;
        __syncthreads();
        for (int g = 0; g < d.ngroups; g++) {
            const int4 g0 = __ldg(d.group + 2 * g), g1 = __ldg(d.group + 2 * g + 1);
            const double2* __restrict__ sr = (g & 1) ? stage1 : stage0;
            double2* __restrict__ sw = (g & 1) ? stage0 : stage1;
            int4 n0 = make_int4(0, 0, 0, 0);
            if (g + 1 < d.ngroups) n0 = __ldg(d.group + 2 * (g + 1));
            const int ns = g1.x, total = ns + (n0.z >> 5);
            // colour flows first (long units), then the next group's pair objects
            for (int u = grab(); u < total; u = grab()) {
                if (u < ns) p3_flow<T2>(d, a, area, sr, accs, e, g0, u, lane);
                else p2_unit(d, area, sw, Ks, n0, u - ns, lane);
            }
            __syncthreads();
            if (tid == 0) ctr = 0;
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
struct HsContext {
    const HsTables* t = nullptr;
    HsDev d;
    void* blob = nullptr;
    void* p2tab = nullptr;
    void* p3tab = nullptr;
    size_t smem = 0;
    int sms = 148;
    int max_sigma = 0;
    size_t smem_overlap = 0;   // 0 = the overlapped variant does not fit / does not apply
};

const HsTables* hs_host_tables(const HsContext* c) { return c->t; }
size_t hs_smem_bytes(const HsContext* c) { return c->smem; }

cudaError_t hs_create(int ngluon, HsContext** out)
{
    *out = nullptr;
    const HsTables* t = hs_tables(ngluon);
    if (!t) return cudaErrorInvalidValue;
    HsContext* c = new HsContext;
    c->t = t;
    // one device blob, every table 16-byte aligned
    struct Part { const void* src; size_t bytes; size_t off; };
    const int nh = 1 << t->npar;
    Part parts[11] = { { t->obj, sizeof(int) * 4 * t->nobj, 0 }, { t->term, sizeof(int) * 4 * t->nterm, 0 },
                       { t->p1_items, sizeof(int) * t->np1, 0 }, { t->legset_mask, sizeof(int) * t->nlegsets, 0 },
                       { t->group, sizeof(int) * 8 * t->ngroups, 0 }, { t->xobj, sizeof(int) * 4 * t->nxobj, 0 },
                       { t->x_items, sizeof(int) * t->nxitems, 0 }, { t->sigma, sizeof(int) * 4 * t->nsigma, 0 },
                       { t->entry, sizeof(int) * 4 * t->nentry, 0 }, { t->vtab, sizeof(unsigned short) * nh * t->nvrow, 0 },
                       { t->hdep, (size_t)40 * t->nvrow, 0 } };
    size_t total = 0;
    for (auto& p : parts) { p.off = total; total += (p.bytes + 255) & ~size_t(255); }
    cudaError_t e = cudaMalloc(&c->blob, total ? total : 256);
    if (e != cudaSuccess) { delete c; return e; }
    for (auto& p : parts)
        if (p.bytes) {
            e = cudaMemcpy((char*)c->blob + p.off, p.src, p.bytes, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
        }
    char* b = (char*)c->blob;
    HsDev& d = c->d;
    d.obj = (const int4*)(b + parts[0].off); d.term = (const int4*)(b + parts[1].off);
    d.p1_items = (const int*)(b + parts[2].off); d.legset_mask = (const int*)(b + parts[3].off);
    d.group = (const int4*)(b + parts[4].off); d.xobj = (const int4*)(b + parts[5].off);
    d.x_items = (const int*)(b + parts[6].off); d.sigma = (const int4*)(b + parts[7].off);
    d.entry = (const int4*)(b + parts[8].off); d.vtab = (const unsigned short*)(b + parts[9].off);
    d.hdep = (const unsigned char*)(b + parts[10].off); d.nw3 = 0;
    // phase-2 stream: fixed-size records [unit][term k < maxt][lane] (see eval_x_term)
    {
        int maxt = 1;
        for (int i = 0; i < t->nxobj; i++) if (t->xobj[4 * i + 3] > maxt) maxt = t->xobj[4 * i + 3];
        auto subv = [](int var, int code) {
            return ((var >> (code & 7)) & 1) | (((var >> ((code >> 3) & 7)) & 1) << 1) | (((var >> ((code >> 6) & 7)) & 1) << 2);
        };
        const size_t nunits = (size_t)t->nxitems / 32;
        std::vector<uint4> tab(nunits * maxt * 32 + 1, make_uint4(0u, 0u, 0xFFu, 0u));
        for (int g = 0; g < t->ngroups; g++) {
            const int* G = t->group + 8 * g;
            for (int u = 0; u < G[2] / 32; u++) {
                const size_t base = ((size_t)(G[1] / 32 + u) * maxt) * 32;
                unsigned ntm = 0;
                for (int l = 0; l < 32; l++) {
                    const int it = t->x_items[G[1] + 32 * u + l];
                    if (it >= 0 && (unsigned)t->xobj[4 * (G[0] + (it >> 8)) + 3] > ntm) ntm = t->xobj[4 * (G[0] + (it >> 8)) + 3];
                }
                for (int l = 0; l < 32; l++) {
                    const int it = t->x_items[G[1] + 32 * u + l];
                    for (int k = 0; k < maxt; k++) tab[base + 32 * k + l].w = ntm;
                    if (it < 0) continue;
                    const int* X = t->xobj + 4 * (G[0] + (it >> 8));
                    const int var = it & 0xFF;
                    const unsigned sblk = (unsigned)(X[0] >> 2) + var;
                    for (int k = 0; k < X[3]; k++) {
                        const int* w = t->term + 4 * (X[2] + k);
                        unsigned blk[3] = { 0, 0, 0 };
                        for (int j = 0; j < 3; j++) {
                            const unsigned word = (unsigned)w[1 + j];
                            blk[j] = ((word & 0xFFFF) >> 2) + subv(var, (word >> 16) & 0x1FF);
                        }
                        uint4& r = tab[base + 32 * k + l];
                        r.x = blk[0] | (blk[1] << 16); r.y = blk[2] | (sblk << 16); r.z = (unsigned)w[0];
                    }
                    tab[base + l].y |= sblk << 16;          // the store block is read from record 0
                }
            }
        }
        e = cudaMalloc(&c->p2tab, tab.size() * sizeof(uint4));
        if (e == cudaSuccess) e = cudaMemcpy(c->p2tab, tab.data(), tab.size() * sizeof(uint4), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { cudaFree(c->p2tab); cudaFree(c->blob); delete c; return e; }
        d.p2tab = (const uint4*)c->p2tab; d.maxt = maxt;
    }
    // phase-3 stream (FP64 tensor path): fixed-size records [colour flow][entry k < maxe][lane] (see p3_entry)
    if (t->npar >= 6) {
        int maxe = 1;
        for (int i = 0; i < t->nsigma; i++) if (t->sigma[4 * i + 2] > maxe) maxe = t->sigma[4 * i + 2];
        std::vector<uint4> tab((size_t)t->nsigma * maxe * 32 + 1, make_uint4(0u, 0u, 0u, 0u));
        for (int sgi = 0; sgi < t->nsigma; sgi++) {
            const int* S = t->sigma + 4 * sgi;
            for (int k = 0; k < S[2]; k++) {
                const int* E = t->entry + 4 * (S[1] + k);
                const int xoff = E[0] & 0xFFFF, nvx = E[0] >> 16, yoff = E[1] & 0xFFFF, nvy = E[1] >> 16;
                const unsigned char* hd = t->hdep + 40 * E[2];
                unsigned shape;
                if (nvx == 32 && nvy == 4) shape = 0;
                else if (nvx == 16 && nvy == 8) shape = 1;
                else if (nvx == 16 && nvy == 4) shape = 2;
                else if (nvx == 8 && nvy == 8) shape = 3;
                else { cudaFree(c->p2tab); cudaFree(c->blob); delete c; return cudaErrorInvalidValue; }
                const int MT = nvx / 8, NT = nvy / 4;
                auto slot_of = [](int off, int var, int comp) { const int bb = (off >> 2) + var; return 4 * bb + (comp ^ ((bb >> 1) & 3)); };
                for (int l = 0; l < 32; l++) {
                    const int r = l >> 2, cc = l & 3;
                    uint4& rec = tab[((size_t)sgi * maxe + k) * 32 + l];
                    const unsigned ys1 = NT == 2 ? (unsigned)slot_of(yoff, 4 + (r >> 1), cc) : 0u;
                    rec.x = (unsigned)slot_of(xoff, r, cc) | ((unsigned)slot_of(yoff, r >> 1, cc) << 16);
                    rec.y = ys1 | (shape << 16) | ((E[3] < 0 ? 1u : 0u) << 18) | ((unsigned)S[2] << 24);
                    rec.z = 0;
                    for (int mt = 0; mt < MT; mt++)
                        for (int nt = 0; nt < NT; nt++)
                            rec.z |= (unsigned)(hd[8 * mt + r] ^ hd[32 + 4 * nt + cc]) << (8 * (mt * NT + nt));
                    rec.w = (unsigned)S[0];
                }
            }
        }
        e = cudaMalloc(&c->p3tab, tab.size() * sizeof(uint4));
        if (e == cudaSuccess) e = cudaMemcpy(c->p3tab, tab.data(), tab.size() * sizeof(uint4), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { cudaFree(c->p3tab); cudaFree(c->p2tab); cudaFree(c->blob); delete c; return e; }
        d.p3tab = (const uint4*)c->p3tab; d.maxe = maxe;
    } else { d.p3tab = nullptr; d.maxe = 0; }
    d.npar = t->npar; d.ncolor = t->ncolor; d.ngroups = t->ngroups; d.obj_area = t->obj_area; d.stage_area = t->stage_area;
    d.nlegsets = t->nlegsets;
    for (int i = 0; i < 4; i++) d.p1_level[i] = t->p1_level[i];
    c->smem = sizeof(double2) * ((size_t)t->obj_area + t->stage_area) + sizeof(double) * 4 * (t->nlegsets + t->npar);
    // colour flows per group (phase-3 tasks): at most that many warps get a jamp accumulator
    for (int g = 0; g < t->ngroups; g++) if (t->group[8 * g + 4] > c->max_sigma) c->max_sigma = t->group[8 * g + 4];
    const size_t smem_max = c->smem + sizeof(double2) * ((size_t)8 << t->npar);
    e = cudaFuncSetAttribute(hs_diagrams_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hs_diagrams_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
    if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
    {
        const size_t smem_ov = c->smem + sizeof(double2) * ((size_t)t->stage_area + ((size_t)c->max_sigma << t->npar));
        if (t->npar >= 6 && smem_ov <= 226 * 1024) {
            e = cudaFuncSetAttribute(hs_overlap_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ov);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(hs_overlap_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_ov);
            if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
            c->smem_overlap = smem_ov;
        }
    }
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
    *out = c;
    return cudaSuccess;
}

void hs_destroy(HsContext* c)
{
    if (!c) return;
    cudaFree(c->blob); cudaFree(c->p2tab); cudaFree(c->p3tab);
    delete c;
}

cudaError_t hs_launch(const HsContext* c, bool jamps_fp64, const HsLaunch& a, int nsplit, int phase3, cudaStream_t st)
{
    if (a.nevt <= 0) return cudaSuccess;
    const int threads = (1 << c->t->npar) * nsplit;
    if (nsplit < 1 || threads > 256) return cudaErrorInvalidValue;
    HsDev d = c->d;
    size_t smem = c->smem;
    if (phase3 == 2) {                               // overlapped variant: one 512-thread CTA per SM
        if (!c->smem_overlap) return cudaErrorInvalidValue;
        d.nw3 = c->max_sigma;
        HsLaunch al2 = a;
        al2.prof = nullptr;
        if (jamps_fp64) hs_overlap_kernel<double><<<a.nevt, 512, c->smem_overlap, st>>>(d, al2);
        else hs_overlap_kernel<float><<<a.nevt, 512, c->smem_overlap, st>>>(d, al2);
        return cudaGetLastError();
    }
    if (phase3 == 1) {                               // FP64 tensor path: needs the 8 x 4 fragment shapes (>= 3 legs on the X side)
        if (c->t->npar < 6) return cudaErrorInvalidValue;
        d.nw3 = c->max_sigma;                        // one accumulator per colour flow of a group
        smem += sizeof(double2) * ((size_t)d.nw3 << d.npar);
    }
    const int grid = a.nevt;                         // one CTA per event; the hardware scheduler keeps every SM full
    // diagnostics: MG_HS_PROFILE=1 prints the share of each phase as seen by thread 0 of every CTA (synchronises)
    static const bool profile = getenv("MG_HS_PROFILE") != nullptr;
    HsLaunch al = a;
    al.prof = nullptr;
    if (profile) {
        static unsigned long long* buf = nullptr;
        if (!buf) cudaMallocManaged(&buf, 8 * sizeof(unsigned long long));
        cudaDeviceSynchronize();
        for (int i = 0; i < 8; i++) buf[i] = 0;
        al.prof = buf;
    }
    if (jamps_fp64) hs_diagrams_kernel<double><<<grid, threads, smem, st>>>(d, al);
    else hs_diagrams_kernel<float><<<grid, threads, smem, st>>>(d, al);
    if (profile) {
        cudaDeviceSynchronize();
        double tot = 0;
        for (int i = 0; i < 6; i++) tot += (double)al.prof[i];
        fprintf(stderr, "[hs profile] setup %.1f%% | phase 1 %.1f%% | phase 2 work %.1f%% wait %.1f%% | phase 3 work %.1f%% wait %.1f%% | %.0f cycles/event\n",
                100 * al.prof[0] / tot, 100 * al.prof[1] / tot, 100 * al.prof[2] / tot, 100 * al.prof[3] / tot, 100 * al.prof[4] / tot,
                100 * al.prof[5] / tot, tot / a.nevt);
        fprintf(stderr, "[hs profile] per colour flow: entries %.0f cycles, write-out %.0f cycles\n",
                (double)al.prof[6] / ((double)a.nevt * c->t->ncolor), (double)al.prof[7] / ((double)a.nevt * c->t->ncolor));
    }
    return cudaGetLastError();
}

}  // namespace mg
