// hs_kernel.cu -- helicity-shared diagram kernel: one CTA = one event; executes the device streams
// of gen/hs_streams.py (layout: hs_tables.h).
//
// Why this shape on B200: the paper keeps one thread per (event, helicity) and lets every helicity
// recompute every wavefunction, with up to 121 wavefunctions + 120 jamps of per-thread state (PAPER.md:101-119, 141,
// 187) -- 12 KB per thread, i.e. local-memory traffic.  Here the state that depends on few helicities lives once per
// event in shared memory (<= 8 variants per object; phase 1), the vertices are contracted with all branches but the
// largest once per variant (phase 2: straight-line code per chunk type) and the per-helicity work is a stream of
// 4-component complex dot products evaluated for all helicities at once on the FP64 tensor path (phase 3), accumulated in
// register fragments per class of entries.  Every jamp is finished on chip and written once, coalesced, to the jamps
// buffer, rows ordered (event, helicity).
//
// Scheduling inside the CTA: the work items of a step -- the colour flows of group g (phase 3) and, when the staging area
// is double-buffered (HsCfg::NBUF = 2), the phase-2 units of group g + 1 -- are dealt to the warps at build time by their
// instruction counts (gen/hs_streams.py _schedule), with ONE barrier per step; phase 1 is dealt the same way, in blocks of
// 32 items with one sequence of opcodes.  The paper's counterpart is the sequence of diagram-group kernels on helicity
// streams; here a "group" never leaves the SM.
//
// Every shared-memory address of phases 2 and 3 comes precomputed from the streams: an argument costs one 16-bit
// extraction, its four components are immediate offsets (component planes), and there is no interpretation of opcodes
// inside a chunk or an entry (the opcode sequence / the shape is a template parameter).
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "generated/hs_gen.h"
#include "helas.cuh"
#include "hs_kernel.cuh"

namespace mg {

struct HsDev {
    const int4* obj; const int4* term; const int* p1_items; const int* legset_mask;
    const uint2* p2rec; const uint2* wsched; const unsigned* witem;
    const uint4* p3rec; const uint2* p3cls; const int* p3clsh; const int4* p3flow;
    int ncolor, nflow, ncls, nsched, nitem;
    int2 p1sched[3][16];       // [level - 1][warp] = { first item, blocks of 32 items }
};

// the small tables every work item starts from, copied to shared memory once per (persistent) CTA
struct HsSmemTabs {
    const int4* p3flow; const int* p3clsh; const uint2* wsched; const unsigned* witem;
};

// variant of an argument object: bit j = bit ((code >> 3j) & 7) of the parent's variant (7 = none; variants are < 128)
__device__ __forceinline__ int sub_variant(int var, int code)
{
    return ((var >> (code & 7)) & 1) | (((var >> ((code >> 3) & 7)) & 1) << 1) | (((var >> ((code >> 6) & 7)) & 1) << 2);
}

// slot of variant v relative to the first slot of its object (gen/hs_streams.py perm)
__device__ __forceinline__ int perm(int v) { return (v & ~1) | (__popc(v) & 1); }

// the four components of one slot: immediate offsets from one address (component planes)
template <int PLANE> __device__ __forceinline__ void ld_wf(const char* __restrict__ area, unsigned off, wf<double>& w)
{
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const double2 v = *reinterpret_cast<const double2*>(area + off + c * PLANE);
        w.c[c].re = v.x; w.c[c].im = v.y;
    }
}

template <int PLANE> __device__ __forceinline__ void st_wf(char* __restrict__ area, unsigned off, const wf<double>& w)
{
#pragma unroll
    for (int c = 0; c < 4; c++) *reinterpret_cast<double2*>(area + off + c * PLANE) = make_double2(w.c[c].re, w.c[c].im);
}

// fp32 -> TF32 (10 explicit significand bits), round to nearest: the tensor core would truncate
__device__ __forceinline__ float to_tf32(float x)
{
    unsigned u;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
    return __uint_as_float(u);
}

__device__ __forceinline__ p4<double> ld_k(const char* __restrict__ Ks, unsigned off)
{
    const double2 a = *reinterpret_cast<const double2*>(Ks + off), b = *reinterpret_cast<const double2*>(Ks + off + 16);
    p4<double> k = { a.x, a.y, b.x, b.y };
    return k;
}

// ------------------------------------------------------------------------------------------------------------
// phase 1: sum of the terms [t0, t0 + nt) for helicity variant `var` of an object whose leg set has total momentum
// K(ls_out); the term table is interpreted directly (2 % of the flops)
template <int OBJ_PLANE>
__device__ __forceinline__ void p1_terms(const HsDev& d, const char* __restrict__ obj, const char* __restrict__ Ks,
                                         const double* __restrict__ pm, int t0, int nt, int var, int ls_out, double mt,
                                         double wt, wf<double>& acc)
{
    auto arg = [&](int word, wf<double>& w) {
        ld_wf<OBJ_PLANE>(obj, 16u * (unsigned)((word & 0xFFFF) + perm(sub_variant(var, (word >> 16) & 0x1FF))), w);
    };
#pragma unroll
    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
    for (int t = 0; t < nt; t++) {
        const int4 w = __ldg(d.term + t0 + t);
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
            arg(w.y, A); arg(w.z, B);
            const p4<double> K = ld_k(Ks, 32u * ls_out);
            switch (op) {
                case 3: v3_off(A, ld_k(Ks, 32u * ((w.x >> 16) & 0xFF)), B, ld_k(Ks, 32u * ((w.x >> 24) & 0xFF)), 1.0 / m2(K), r); break;
                case 4: { wf<double> Z; arg(w.w, Z); v4_off(A, B, Z, 1.0 / m2(K), r); break; }
                case 5: ffv_l(A, B, -K, mt, inv_prop(m2(K), mt, wt), r); break;
                case 6: ffv_r(A, B, K, mt, inv_prop(m2(K), mt, wt), r); break;
                default: ffv_p(A, B, 1.0 / m2(K), r); break;       // 7
            }
        }
        const double sg = neg ? -1.0 : 1.0;
#pragma unroll
        for (int c = 0; c < 4; c++) { acc.c[c].re = fma(sg, r.c[c].re, acc.c[c].re); acc.c[c].im = fma(sg, r.c[c].im, acc.c[c].im); }
    }
}

// ------------------------------------------------------------------------------------------------------------
// phase 2: one term of a chunk; OP is a compile-time constant, the record holds the byte offsets of the arguments
//   r.x = offA | offB << 16,  r.y = offC  (x_v3: 32 legset(A) | 32 legset(B) << 16)
// The term's sign (smask = 0 or 0x80000000) goes onto the scalar coefficients of the vertex with integer XORs and the
// vertex is accumulated straight into acc (no separate signed add); acc is kept contravariant, the index lowering for the
// plain dot of phase 3 happens once per item at the store (p2_chunk).
__device__ __forceinline__ double flip(double v, unsigned smask)
{
    return __hiloint2double(__double2hiint(v) ^ (int)smask, __double2loint(v));
}
__device__ __forceinline__ cx<double> flip(cx<double> v, unsigned smask) { return mk<double>(flip(v.re, smask), flip(v.im, smask)); }

template <int OP, int OBJ_PLANE>
__device__ __forceinline__ void x_term(const char* __restrict__ obj, const char* __restrict__ Ks, const uint2 r, const unsigned smask,
                                       wf<double>& acc)
{
    wf<double> A, B;
    ld_wf<OBJ_PLANE>(obj, r.x & 0xFFFFu, A);
    ld_wf<OBJ_PLANE>(obj, r.x >> 16, B);
    if constexpr (OP == 11) {
        // (A.B)(kA - kB) + ((2 kB + kA).A) B - ((2 kA + kB).B) A
        const p4<double> kA = ld_k(Ks, r.y & 0xFFFFu), kB = ld_k(Ks, r.y >> 16);
        const p4<double> ea = { fma(2.0, kB.e, kA.e), fma(2.0, kB.x, kA.x), fma(2.0, kB.y, kA.y), fma(2.0, kB.z, kA.z) };
        const p4<double> eb = { fma(2.0, kA.e, kB.e), fma(2.0, kA.x, kB.x), fma(2.0, kA.y, kB.y), fma(2.0, kA.z, kB.z) };
        const cx<double> ab = flip(dot(A, B), smask), xa = flip(dot(ea, A), smask), xb = flip(dot(eb, B), smask);
        const double dd[4] = { kA.e - kB.e, kA.x - kB.x, kA.y - kB.y, kA.z - kB.z };
#pragma unroll
        for (int mu = 0; mu < 4; mu++) {
            const cx<double> t = mk<double>(fma(dd[mu], ab.re, acc.c[mu].re), fma(dd[mu], ab.im, acc.c[mu].im));
            acc.c[mu] = cfms(xb, A.c[mu], cfma(xa, B.c[mu], t));
        }
    } else if constexpr (OP == 12) {
        // (A.Z) B - (B.Z) A
        wf<double> Z; ld_wf<OBJ_PLANE>(obj, r.y & 0xFFFFu, Z);
        const cx<double> xz = flip(dot(A, Z), smask), yz = flip(dot(B, Z), smask);
#pragma unroll
        for (int mu = 0; mu < 4; mu++) acc.c[mu] = cfms(yz, A.c[mu], cfma(xz, B.c[mu], acc.c[mu]));
    } else if constexpr (OP == 13) {
        // both orderings of the four-gluon vertex that share the middle leg: 2 (A.Z) B - (B.Z) A - (B.A) Z
        wf<double> Z; ld_wf<OBJ_PLANE>(obj, r.y & 0xFFFFu, Z);
        cx<double> xz = dot(A, Z);
        xz = flip(xz + xz, smask);
        const cx<double> yz = flip(dot(B, Z), smask), yx = flip(dot(B, A), smask);
#pragma unroll
        for (int mu = 0; mu < 4; mu++) acc.c[mu] = cfms(yx, Z.c[mu], cfms(yz, A.c[mu], cfma(xz, B.c[mu], acc.c[mu])));
    } else {
        wf<double> q;
        if constexpr (OP == 8) row_slash(A, make_slashed(B), q);
        else if constexpr (OP == 9) slash_col(make_slashed(A), B, q);
        else {
            static_assert(OP == 10, "unknown phase-2 opcode");
            ffv_p_raw(A, B, q);
        }
        const double sg = flip(1.0, smask);
#pragma unroll
        for (int c = 0; c < 4; c++) { acc.c[c].re = fma(sg, q.c[c].re, acc.c[c].re); acc.c[c].im = fma(sg, q.c[c].im, acc.c[c].im); }
    }
}

// a chunk = up to three terms of fixed opcodes for 32 items (CT: one hex digit (opcode - 7) per term); sign of term j =
// bit 16 + j of r0.x.  All terms of an item are of one kind: vector-valued (opcodes >= 10: the pair object is contracted
// with a gluon-type Y, components 1-3 are negated at the store) or spinor-valued (8, 9).
template <int CT, int OBJ_PLANE, int STG_PLANE>
__device__ __forceinline__ void p2_chunk(const char* __restrict__ obj, const char* __restrict__ Ks, char* __restrict__ stage,
                                         const uint2 r0, const uint2 r1, const uint2 r2, const uint2 r3, wf<double>& acc)
{
    constexpr int O0 = CT & 0xF, O1 = (CT >> 4) & 0xF, O2 = (CT >> 8) & 0xF;
    x_term<O0 + 7, OBJ_PLANE>(obj, Ks, r1, (r0.x << 15) & 0x80000000u, acc);
    if constexpr (O1 != 0) x_term<O1 + 7, OBJ_PLANE>(obj, Ks, r2, (r0.x << 14) & 0x80000000u, acc);
    if constexpr (O2 != 0) x_term<O2 + 7, OBJ_PLANE>(obj, Ks, r3, (r0.x << 13) & 0x80000000u, acc);
    if (r0.y & 0x2000u) {
        wf<double> o = acc;
        if constexpr (O0 + 7 >= 10) {
#pragma unroll
            for (int c = 1; c < 4; c++) o.c[c] = flip(o.c[c], 0x80000000u);
        }
        st_wf<STG_PLANE>(stage, r0.x & 0xFFFFu, o);
    }
}

// ------------------------------------------------------------------------------------------------------------
// phase 3 on the FP64 tensor path (mma.sync.m8n8k4.f64).  One entry for all 2^npar helicity combinations is the complex
// outer-product sum  out[hx][hy] = sum_c X_c[hx] * Y_c[hy]  (c = 4 components), i.e. real GEMM tiles [8 x 8] . [8 x 8]:
// A = [Re | Im] of the row operand, B = [Re, Im ; -Im, Re] of the column operand (columns (variant, re/im)).
// Fragment layout: a = A[lane / 4][lane % 4], b = B[lane % 4][lane / 4], c0, c1 = C[lane / 4][2 (lane % 4) + {0, 1}].
// The two k-steps of a tile (real and imaginary part of the row operand) go to SEPARATE accumulators -- the FP64 MMA has
// a dependent-issue latency of ~200 cycles on B200 (measured) and no negated operand is needed this way:
//   f[4t + {0,1}] = sum Re A (Re B | Im B),  f[4t + {2,3}] = sum Im A (Im B | Re B),  re = f[4t] - f[4t+2], im = f[4t+1] + f[4t+3].
// All entries of a CLASS map (lane, tile) to the same helicity combination, so f stays in registers over the class.
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__host__ __device__ constexpr int popc_c(int m)
{
    int r = 0;
    for (int b = 0; b < 8; b++) r += (m >> b) & 1;
    return r;
}
// bits of t selected by mask m, packed (tile index -> fragment index)
__host__ __device__ constexpr int pext_c(int t, int m)
{
    int r = 0, k = 0;
    for (int b = 0; b < 8; b++)
        if ((m >> b) & 1) { r |= ((t >> b) & 1) << k; k++; }
    return r;
}

// SWAP = 0: rows from the pair object X (staging area), columns from Y (object area); 1: the other way round.
// MASK: tile bits that select the A fragment.  abase / bbase = plane (lane % 4) of the A / B operand's area.
template <int SWAP, int MASK, int NTILE>
__device__ __forceinline__ void p3_entry(const char* __restrict__ abase, const char* __restrict__ bbase, const uint4 e,
                                         double (&f)[4 * NTILE])
{
    constexpr int NA = 1 << popc_c(MASK), NB = NTILE / NA, AW = (NA + 1) / 2;
    const unsigned w[3] = { e.x, e.y, e.z };
    const unsigned smask = e.w & 0x80000000u;
    double2 xa[NA];
    double b0[NB], b1[NB];
#pragma unroll
    for (int a = 0; a < NA; a++) {
        const unsigned word = w[a >> 1];
        const unsigned off = (a & 1) ? (word >> 16) : (word & 0xFFFFu);
        xa[a] = *reinterpret_cast<const double2*>(abase + off);
    }
#pragma unroll
    for (int b = 0; b < NB; b++) {
        const unsigned word = w[AW + (b >> 1)];
        const unsigned off = (b & 1) ? (word >> 16) : (word & 0xFFFFu);
        b0[b] = *reinterpret_cast<const double*>(bbase + off);           // odd column (im out): Im, even: Re
        b1[b] = *reinterpret_cast<const double*>(bbase + (off ^ 8u));    // odd column: Re, even: Im
    }
    if constexpr (NA <= NB) {
#pragma unroll
        for (int a = 0; a < NA; a++) { xa[a].x = flip(xa[a].x, smask); xa[a].y = flip(xa[a].y, smask); }
    } else {
#pragma unroll
        for (int b = 0; b < NB; b++) { b0[b] = flip(b0[b], smask); b1[b] = flip(b1[b], smask); }
    }
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        constexpr int NM = NTILE - 1;
        const int ai = pext_c(t, MASK), bi = pext_c(t, ~MASK & NM);
        dmma884(f[4 * t], f[4 * t + 1], xa[ai].x, b0[bi]);
        dmma884(f[4 * t + 2], f[4 * t + 3], xa[ai].y, b1[bi]);
    }
}

// add the fragments of a finished class to the flow's accumulator (first class: plain store)
template <int NTILE>
__device__ __forceinline__ void p3_flush(char* __restrict__ acc, const uint2 cl, const double (&f)[4 * NTILE], bool first)
{
    double2 v[NTILE];
    unsigned off[NTILE];
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        const unsigned word = t < 2 ? cl.x : cl.y;
        off[t] = (t & 1) ? (word >> 16) : (word & 0xFFFFu);
        v[t] = make_double2(0.0, 0.0);
        if (!first) v[t] = *reinterpret_cast<const double2*>(acc + off[t]);
    }
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        v[t].x += f[4 * t] - f[4 * t + 2];
        v[t].y += f[4 * t + 1] + f[4 * t + 3];
        *reinterpret_cast<double2*>(acc + off[t]) = v[t];
    }
}

// Class changes, second form (HS_STLD): the flow's running sum travels in the fragments.  A finished class STORES (re, im) = (f[4t] - f[4t+2], f[4t+1]
// + f[4t+3]) to the flow's accumulator; the next class LOADS it back into f[4t], f[4t+1] in its own (lane, tile) order and the tensor
// instructions add onto it.  (A read-add-write flush had 16 FP64 additions per class waiting in the FP64 pipe's queue behind the
// other warps' tensor instructions.  Measured: generic kernel -3 % (hsg_kernel.cu), g g -> t tbar g g -2.3 % (13.34 -> 13.03 ms per
// 262 144 events), g g -> t tbar g g g +1.4 % (36.60 -> 37.12 ms: the warp barrier and the load in front of every class's first
// tensor instruction cost more there) -- hence per process.)
template <int NG> struct HsStLd { static constexpr bool value = NG == 4; };
template <int NTILE>
__device__ __forceinline__ void p3_store(char* __restrict__ acc, const uint2 cl, const double (&f)[4 * NTILE])
{
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        const unsigned word = t < 2 ? cl.x : cl.y;
        const unsigned off = (t & 1) ? (word >> 16) : (word & 0xFFFFu);
        *reinterpret_cast<double2*>(acc + off) = make_double2(f[4 * t] - f[4 * t + 2], f[4 * t + 1] + f[4 * t + 3]);
    }
}
template <int NTILE>
__device__ __forceinline__ void p3_load(const char* __restrict__ acc, const uint2 cl, double (&f)[4 * NTILE])
{
#pragma unroll
    for (int t = 0; t < NTILE; t++) {
        const unsigned word = t < 2 ? cl.x : cl.y;
        const unsigned off = (t & 1) ? (word >> 16) : (word & 0xFFFFu);
        const double2 v = *reinterpret_cast<const double2*>(acc + off);
        f[4 * t] = v.x; f[4 * t + 1] = v.y; f[4 * t + 2] = 0.0; f[4 * t + 3] = 0.0;
    }
}

// accumulator slot of helicity combination h (gen/co_program.py acc_swizzle)
__device__ __forceinline__ int acc_swizzle(int h)
{
    const int hi = h >> 3;
    return h ^ (((hi & 1) * 3) ^ (((hi >> 1) & 1) * 5) ^ (((hi >> 2) & 1) * 6) ^ (((hi >> 3) & 1) * 7));
}

// ------------------------------------------------------------------------------------------------------------
// one colour flow (phase 3) as STRAIGHT-LINE code.  The classes of a flow come in a canonical order and the sequence of
// their headers H0 .. H4 (count of entries per shape; the flow's SIGNATURE, gen/hs_streams.py) is a template parameter,
// so every entry's shape, every record's address and every class boundary is a compile-time constant: no loop, no
// dispatch inside a flow; the records of a class are loaded while the previous class is evaluated.  HsCfg::P3_PAD: all
// flows of the process are padded to ONE signature -- a slot a flow does not use carries the skip bit (record word w,
// bit 8), a class it does not use has header 0 in p3clsh -- because the SM's instruction cache is smaller than this
// kernel (2 -> 5: three instantiations measured 13 % slower than one although they execute 17 % fewer instructions).
template <int NG> __host__ __device__ constexpr int shape_code(int k)
{
    return k == 0 ? HsCfg<NG>::SHAPE0 : k == 1 ? HsCfg<NG>::SHAPE1 : k == 2 ? HsCfg<NG>::SHAPE2 : HsCfg<NG>::SHAPE3;
}
__host__ __device__ constexpr int hdr_entries(int h) { return (h & 15) + ((h >> 4) & 15) + ((h >> 8) & 15) + ((h >> 12) & 15); }
__host__ __device__ constexpr int max_c(int a, int b) { return a > b ? a : b; }

template <int N> struct P3Recs { uint4 r[N]; };

template <int NE, int NMAX> __device__ __forceinline__ void p3_load_class(P3Recs<NMAX>& q, const uint4* __restrict__ rp, int e0)
{
#pragma unroll
    for (int i = 0; i < NE; i++) q.r[i] = __ldg(rp + 8 * (e0 + i));
}

template <int NG, int H, int K, int I0, int NMAX>
__device__ __forceinline__ void p3_static_run(const P3Recs<NMAX>& q, const char* __restrict__ objl, const char* __restrict__ stgl,
                                              double (&f)[4 * HsCfg<NG>::NTILE])
{
    constexpr int CODE = shape_code<NG>(K), N = (H >> (4 * K)) & 15, NTILE = HsCfg<NG>::NTILE;
    if constexpr (CODE >= 0 && N > 0) {
#pragma unroll
        for (int i = 0; i < N; i++) {
            if (((HsCfg<NG>::P3_ALWAYS >> K) & 1) || !(q.r[I0 + i].w & 0x100u)) {        // (uniform over the warp)
                if constexpr (CODE & 1) p3_entry<1, (CODE >> 1), NTILE>(objl, stgl, q.r[I0 + i], f);
                else p3_entry<0, (CODE >> 1), NTILE>(stgl, objl, q.r[I0 + i], f);
            }
        }
    }
}

// class C of the flow (header H, first entry E0); HN = header of the next class (its records are put in flight first)
template <int NG, int H, int HN, int E0, int C, int NMAX>
__device__ __forceinline__ void p3_static_class(const P3Recs<NMAX>& q, P3Recs<NMAX>& qn, const uint4* __restrict__ rp,
                                                const uint2* __restrict__ cp, const int* __restrict__ hp,
                                                const char* __restrict__ objl, const char* __restrict__ stgl, char* __restrict__ acc)
{
    constexpr int NTILE = HsCfg<NG>::NTILE;
    if constexpr (H != 0) {
        if constexpr (HN != 0) p3_load_class<hdr_entries(HN), NMAX>(qn, rp, E0 + hdr_entries(H));
        if (HsCfg<NG>::P3_PAD && C > 0 && hp[C] == 0) return;      // a padded flow does not have this class
        const uint2 cl = __ldg(cp + 32 * C);
        double f[4 * NTILE];
        if constexpr (C == 0 || !HsStLd<NG>::value) {
#pragma unroll
            for (int i = 0; i < 4 * NTILE; i++) f[i] = 0.0;
        } else {
            __syncwarp();                                   // the previous class's stores (other lanes' slots)
            p3_load<NTILE>(acc, cl, f);
        }
        constexpr int n0 = H & 15, n1 = (H >> 4) & 15, n2 = (H >> 8) & 15;
        p3_static_run<NG, H, 0, 0, NMAX>(q, objl, stgl, f);
        p3_static_run<NG, H, 1, n0, NMAX>(q, objl, stgl, f);
        p3_static_run<NG, H, 2, n0 + n1, NMAX>(q, objl, stgl, f);
        p3_static_run<NG, H, 3, n0 + n1 + n2, NMAX>(q, objl, stgl, f);
        if constexpr (HsStLd<NG>::value) p3_store<NTILE>(acc, cl, f);
        else p3_flush<NTILE>(acc, cl, f, C == 0);
    }
}

template <int NG, typename T2, int H0, int H1, int H2, int H3, int H4>
__device__ __forceinline__ void p3_flow_sig(const HsDev& d, const HsSmemTabs& tb, const HsLaunch& a, const int4 fd, int e,
                                            const char* __restrict__ objl, const char* __restrict__ stgl, char* __restrict__ accs,
                                            int warp, int lane, const int (&posr)[(1 << HsCfg<NG>::NPAR) / 32])
{
    using Cfg = HsCfg<NG>;
    constexpr int NH = 1 << Cfg::NPAR;
    constexpr int NMAX = max_c(max_c(max_c(hdr_entries(H0), hdr_entries(H1)), max_c(hdr_entries(H2), hdr_entries(H3))), hdr_entries(H4));
    constexpr int E1 = hdr_entries(H0), E2 = E1 + hdr_entries(H1), E3 = E2 + hdr_entries(H2), E4 = E3 + hdr_entries(H3);
    const int jamp = fd.w;
    // one accumulator per flow of the group, or per warp when a group has more flows than the CTA has warps
    char* __restrict__ acc = accs + (size_t)(Cfg::MAX_FLOWS > Cfg::NW ? warp : ((fd.y >> 16) & 0xFF)) * (NH * 16);
    const uint4* __restrict__ rp = d.p3rec + (size_t)fd.x * 8 + (lane >> 2);
    const uint2* __restrict__ cp = d.p3cls + (size_t)fd.z * 32 + lane;
    const int* __restrict__ hp = tb.p3clsh + fd.z;
    P3Recs<NMAX> qa, qb;                      // record sets of the current / the next class, alternating
    p3_load_class<hdr_entries(H0), NMAX>(qa, rp, 0);
    p3_static_class<NG, H0, H1, 0, 0, NMAX>(qa, qb, rp, cp, hp, objl, stgl, acc);
    p3_static_class<NG, H1, H2, E1, 1, NMAX>(qb, qa, rp, cp, hp, objl, stgl, acc);
    p3_static_class<NG, H2, H3, E2, 2, NMAX>(qa, qb, rp, cp, hp, objl, stgl, acc);
    p3_static_class<NG, H3, H4, E3, 3, NMAX>(qb, qa, rp, cp, hp, objl, stgl, acc);
    p3_static_class<NG, H4, 0, E4, 4, NMAX>(qa, qb, rp, cp, hp, objl, stgl, acc);
    __syncwarp();
    // the finished jamp of this colour flow, all helicity combinations
    T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
#pragma unroll
    for (int j = 0; j < NH / 32; j++) {
        const int h = lane + 32 * j, pos = posr[j];
        if (pos >= 0) {
            const double2 v = *reinterpret_cast<const double2*>(acc + 16 * acc_swizzle(h));
            const size_t row = (size_t)e * a.nrow_evt + pos;
            if (a.tile_major == 2) {
                // tcgen05 operand layout (csrc/color_sum_tf32.cu, "direct"): per 128-row tile and part, chunks of 24 colours
                // as K-major core matrices [row / 8][colour quad][row % 8][colour % 4], values rounded to TF32
                if constexpr (sizeof(T2) == 4) {
                    const unsigned m = (unsigned)(row & 127);
                    float* __restrict__ o = reinterpret_cast<float*>(out) + (row >> 7) * (size_t)(256 * d.ncolor) +
                                            (size_t)(jamp / 24) * (24 * 128) + (m >> 3) * 192 + ((jamp % 24) >> 2) * 32 + (m & 7) * 4 + (jamp & 3);
                    o[0] = to_tf32((float)v.x); o[(size_t)d.ncolor * 128] = to_tf32((float)v.y);
                }
            } else if (a.tile_major) {
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

template <int NG, typename T2>
__device__ __forceinline__ void p3_flow(const HsDev& d, const HsSmemTabs& tb, const HsLaunch& a, int fl, int e,
                                        const char* __restrict__ objl, const char* __restrict__ stgl, char* __restrict__ accs,
                                        int warp, int lane, const int (&posr)[(1 << HsCfg<NG>::NPAR) / 32])
{
    const int4 fd = tb.p3flow[fl];
#define HS_SIG_CASE(ID, H0, H1, H2, H3, H4) \
    case ID: p3_flow_sig<NG, T2, H0, H1, H2, H3, H4>(d, tb, a, fd, e, objl, stgl, accs, warp, lane, posr); break;
    if constexpr (NG == 4) {
        switch ((fd.y >> 24) & 0x7F) { HS_FLOW_SIGS_4(HS_SIG_CASE) default: break; }
    } else {
        static_assert(NG == 5, "add the process's HS_FLOW_SIGS list here");
        switch ((fd.y >> 24) & 0x7F) { HS_FLOW_SIGS_5(HS_SIG_CASE) default: break; }
    }
#undef HS_SIG_CASE
}

// the phase-2 work of a warp in a step: a contiguous run of chunks; a unit (the chunks of the same 32 (pair object,
// variant) items) starts where rec0 says "first" (accumulators zeroed) and ends at "last" (result stored, p2_chunk).
// The records of the next chunk are in flight while the current one is evaluated.
template <int NG>
__device__ __forceinline__ void p2_run(const HsDev& d, int chunk0, int nchunk, const char* __restrict__ obj,
                                       const char* __restrict__ Ks, char* __restrict__ stage, int lane, uint2 n0, uint2 n1, uint2 n2,
                                       uint2 n3)
{
    using Cfg = HsCfg<NG>;
    constexpr int OBJ_PLANE = Cfg::OBJ_PLANE, STG_PLANE = Cfg::STG_PLANE;
    const uint2* __restrict__ rp = d.p2rec + (size_t)chunk0 * 128 + lane;          // n0 .. n3 = the records of chunk0
    wf<double> acc;
#pragma unroll
    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
    for (int c = 0; c < nchunk; c++) {
        const uint2 r0 = n0, r1 = n1, r2 = n2, r3 = n3;
        rp += 128;                                       // (one chunk past the end of the table: inside the blob)
        n0 = __ldg(rp); n1 = __ldg(rp + 32); n2 = __ldg(rp + 64); n3 = __ldg(rp + 96);
        if (r0.y & 0x1000u) {
#pragma unroll
            for (int q = 0; q < 4; q++) acc.c[q] = mk<double>(0.0, 0.0);
        }
        switch (r0.y & 0xFFFu) {
#define HS_CASE(CT) case CT: p2_chunk<CT, OBJ_PLANE, STG_PLANE>(obj, Ks, stage, r0, r1, r2, r3, acc); break;
            HS_CHUNK_TYPES(HS_CASE)
#undef HS_CASE
            default: break;
        }
    }
}

// T2 = type of the jamps buffer (double: MG_FP64, float: MG_MIXED -- PAPER.md:122 "FPTYPE=m")
template <int NG, typename T2>
__global__ void __launch_bounds__(32 * HsCfg<NG>::NW, HsCfg<NG>::CTAS) hs_diagrams_kernel(const HsDev d, const HsLaunch a)
{
    using Cfg = HsCfg<NG>;
    constexpr int NPAR = Cfg::NPAR, NH = 1 << NPAR, NW = Cfg::NW, NBUF = Cfg::NBUF, NGROUPS = Cfg::NGROUPS;
    constexpr int OBJ_PLANE = Cfg::OBJ_PLANE, STG_PLANE = Cfg::STG_PLANE;
    constexpr int NACC = Cfg::MAX_FLOWS > NW ? NW : Cfg::MAX_FLOWS;
    extern __shared__ __align__(128) char sm[];
    char* __restrict__ obj = sm;
    char* __restrict__ stage0 = sm + 4 * OBJ_PLANE;
    char* __restrict__ accs = stage0 + NBUF * 4 * STG_PLANE;
    char* __restrict__ Ks = accs + NACC * NH * 16;
    double* __restrict__ pm = reinterpret_cast<double*>(Ks + 32 * Cfg::NLEGSETS);
    HsSmemTabs tb;
    {
        int4* t0 = reinterpret_cast<int4*>(pm + 4 * NPAR);
        int* t1 = reinterpret_cast<int*>(t0 + d.nflow);
        uint2* t2 = reinterpret_cast<uint2*>(t1 + ((d.ncls + 1) & ~1));
        unsigned* t3 = reinterpret_cast<unsigned*>(t2 + d.nsched);
        for (int i = threadIdx.x; i < d.nflow; i += blockDim.x) t0[i] = __ldg(d.p3flow + i);
        for (int i = threadIdx.x; i < d.ncls; i += blockDim.x) t1[i] = __ldg(d.p3clsh + i);
        for (int i = threadIdx.x; i < d.nsched; i += blockDim.x) t2[i] = __ldg(d.wsched + i);
        for (int i = threadIdx.x; i < d.nitem; i += blockDim.x) t3[i] = __ldg(d.witem + i);
        tb.p3flow = t0; tb.p3clsh = t1; tb.wsched = t2; tb.witem = t3;
    }
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NTH = 32 * NW;
    const char* __restrict__ objl = obj + (lane & 3) * OBJ_PLANE;             // plane of this lane's fragment component
    int posr[NH / 32];                                  // rows of this lane's helicity combinations (write-out of phase 3)
#pragma unroll
    for (int j = 0; j < NH / 32; j++) posr[j] = a.d_pos[lane + 32 * j];
    // steps of one event: NBUF = 2: step s = phase 3 of group s - 1 together with phase 2 of group s (s = 0 .. NGROUPS);
    //                     NBUF = 1: step 2 g = phase 2 of group g, step 2 g + 1 = phase 3 of group g
    constexpr int NSTEPS = NBUF == 2 ? NGROUPS + 1 : 2 * NGROUPS;
    for (int e = blockIdx.x; e < a.nevt; e += gridDim.x) {
        // a0: momenta (AOS fp64) -> shared; leg-set momenta in the all-incoming convention
        for (int i = tid; i < 4 * NPAR; i += NTH) pm[i] = a.mom[(size_t)e * (4 * NPAR) + i];
        __syncthreads();
        for (int s = tid; s < Cfg::NLEGSETS; s += NTH) {
            const int m = __ldg(d.legset_mask + s);
            double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
#pragma unroll
            for (int p = 0; p < NPAR; p++)
                if ((m >> p) & 1) {
                    const double sg = p < 2 ? 1.0 : -1.0;
                    k0 += sg * pm[4 * p]; k1 += sg * pm[4 * p + 1]; k2 += sg * pm[4 * p + 2]; k3 += sg * pm[4 * p + 3];
                }
            double* K = reinterpret_cast<double*>(Ks + 32 * s);
            K[0] = k0; K[1] = k1; K[2] = k2; K[3] = k3;
        }
        __syncthreads();
        // HsCfg::PRE (measured per process: -6 % for g g -> t tbar g g, +3 % for g g -> t tbar g g g, where it is off): the
        // first records a warp needs in a step are loaded BEFORE the barrier that ends the previous step (the tables do
        // not depend on the event): pa, pb = the four records of the first chunk of a warp that has no colour flow in that step.
        uint4 pa = make_uint4(0u, 0u, 0u, 0u), pb = pa;
        auto preload = [&](int s) {
            if (!Cfg::PRE || s >= NSTEPS) return;
            const uint2 sc = tb.wsched[s * NW + warp];
            if (!(sc.x >> 16) && (sc.y >> 16)) {
                const uint2* __restrict__ rp = d.p2rec + (size_t)(sc.y & 0xFFFFu) * 128 + lane;
                const uint2 r0 = __ldg(rp), r1 = __ldg(rp + 32), r2 = __ldg(rp + 64), r3 = __ldg(rp + 96);
                pa = make_uint4(r0.x, r0.y, r1.x, r1.y); pb = make_uint4(r2.x, r2.y, r3.x, r3.y);
            }
        };
        // phase 1: objects, level by level
        for (int lvl = 0; lvl < 3; lvl++) {
            const int2 ps = d.p1sched[lvl][warp];
            for (int b = 0; b < ps.y; b++) {
                const int it = __ldg(d.p1_items + ps.x + 32 * b + lane);
                if (it < 0) continue;
                const int4 o = __ldg(d.obj + (it >> 8));
                const int var = it & 0xFF;
                wf<double> acc;
                p1_terms<OBJ_PLANE>(d, obj, Ks, pm, o.z, o.w, var, o.y >> 8, a.mt, a.wt, acc);
                st_wf<OBJ_PLANE>(obj, 16u * (unsigned)(o.x + perm(var)), acc);
            }
            if (lvl == 2) preload(0);
            __syncthreads();
        }
        for (int s = 0; s < NSTEPS; s++) {
            // staging buffer the units of this step fill, and the one its colour flows read
            const int b2 = NBUF == 2 ? (s & 1) : 0, b3 = NBUF == 2 ? ((s - 1) & 1) : 0;
            char* __restrict__ stage2 = stage0 + b2 * 4 * STG_PLANE;
            const char* __restrict__ stgl3 = stage0 + b3 * 4 * STG_PLANE + (lane & 3) * STG_PLANE;
            const uint2 sc = tb.wsched[s * NW + warp];
            const unsigned* __restrict__ ip = tb.witem + (sc.x & 0xFFFFu);
            const int nfl = sc.x >> 16, nch = sc.y >> 16;
            uint2 c0 = make_uint2(pa.x, pa.y), c1 = make_uint2(pa.z, pa.w), c2 = make_uint2(pb.x, pb.y), c3 = make_uint2(pb.z, pb.w);
            if (Cfg::PRE && nfl > 0 && nch > 0) {
                // the chunk run's first records travel through the colour flow(s) in registers
                const uint2* __restrict__ rp = d.p2rec + (size_t)(sc.y & 0xFFFFu) * 128 + lane;
                c0 = __ldg(rp); c1 = __ldg(rp + 32); c2 = __ldg(rp + 64); c3 = __ldg(rp + 96);
            }
            for (int k = 0; k < nfl; k++) p3_flow<NG, T2>(d, tb, a, ip[k], e, objl, stgl3, accs, warp, lane, posr);
            if (!Cfg::PRE && nch > 0) {
                const uint2* __restrict__ rp = d.p2rec + (size_t)(sc.y & 0xFFFFu) * 128 + lane;
                c0 = __ldg(rp); c1 = __ldg(rp + 32); c2 = __ldg(rp + 64); c3 = __ldg(rp + 96);
            }
            if (nch) p2_run<NG>(d, sc.y & 0xFFFFu, nch, obj, Ks, stage2, lane, c0, c1, c2, c3);
            preload(s + 1);
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
struct HsContext {
    const HsTables* t = nullptr;
    int ngluon = 0;
    HsDev d;
    void* blob = nullptr;
    size_t smem = 0;
    int threads = 0, ctas = 1, sms = 0;
};

const HsTables* hs_host_tables(const HsContext* c) { return c->t; }
size_t hs_smem_bytes(const HsContext* c) { return c->smem; }

template <int NG> static size_t smem_bytes(const HsTables* t)
{
    using Cfg = HsCfg<NG>;
    constexpr int NACC = Cfg::MAX_FLOWS > Cfg::NW ? Cfg::NW : Cfg::MAX_FLOWS;
    return 4 * (size_t)Cfg::OBJ_PLANE + Cfg::NBUF * 4 * (size_t)Cfg::STG_PLANE + (size_t)NACC * (16u << Cfg::NPAR) +
           32 * (size_t)Cfg::NLEGSETS + 32 * (size_t)Cfg::NPAR +
           16 * (size_t)t->nflow + 4 * (size_t)((t->ncls + 1) & ~1) + 8 * (size_t)t->nsteps * Cfg::NW + 4 * (size_t)t->nitem;
}

template <int NG> static cudaError_t set_smem(size_t smem)
{
    cudaError_t e = cudaFuncSetAttribute(hs_diagrams_kernel<NG, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hs_diagrams_kernel<NG, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e;
}

// Tables are uploaded to the CURRENT device; the per-function shared-memory attribute is set here, per context, so that a
// second handle on another device sets it there too.
cudaError_t hs_create(int ngluon, HsContext** out)
{
    *out = nullptr;
    const HsTables* t = hs_tables(ngluon);
    if (!t) return cudaErrorInvalidValue;
    HsContext* c = new HsContext;
    c->t = t; c->ngluon = ngluon;
    int c_nw = 0;
    switch (ngluon) {
#define HS_NWOF(N) case N: c_nw = HsCfg<N>::NW; break;
        HS_PROCESSES(HS_NWOF)
#undef HS_NWOF
        default: delete c; return cudaErrorInvalidValue;
    }
    // one device blob, every table 256-byte aligned
    struct Part { const void* src; size_t bytes; size_t off; };
    Part parts[11] = { { t->obj, sizeof(int) * 4 * t->nobj, 0 }, { t->term, sizeof(int) * 4 * t->nterm, 0 },
                       { t->p1_items, sizeof(int) * t->np1, 0 }, { t->legset_mask, sizeof(int) * t->nlegsets, 0 },
                       { t->p2rec, sizeof(unsigned) * 256 * (size_t)t->nchunk, 0 }, { t->wsched, sizeof(unsigned) * 2 * (size_t)t->nsteps * (c_nw), 0 },
                       { t->p3rec, sizeof(unsigned) * 32 * (size_t)t->nentry, 0 }, { t->p3cls, sizeof(unsigned) * 64 * (size_t)t->ncls, 0 },
                       { t->p3flow, sizeof(int) * 4 * t->nflow, 0 }, { t->witem, sizeof(unsigned) * (size_t)t->nitem, 0 },
                       { t->p3clsh, sizeof(int) * (size_t)t->ncls, 0 } };
    size_t total = 0;
    for (auto& p : parts) { p.off = total; total += (p.bytes + 255) & ~size_t(255); }
    total += 4096;                                  // the record prefetch may run a few records past the end of a stream
    cudaError_t e = cudaMalloc(&c->blob, total);
    if (e != cudaSuccess) { delete c; return e; }
    e = cudaMemset(c->blob, 0, total);
    for (auto& p : parts)
        if (p.bytes && e == cudaSuccess) e = cudaMemcpy((char*)c->blob + p.off, p.src, p.bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
    char* b = (char*)c->blob;
    HsDev& d = c->d;
    d.obj = (const int4*)(b + parts[0].off); d.term = (const int4*)(b + parts[1].off);
    d.p1_items = (const int*)(b + parts[2].off); d.legset_mask = (const int*)(b + parts[3].off);
    d.p2rec = (const uint2*)(b + parts[4].off); d.wsched = (const uint2*)(b + parts[5].off);
    d.p3rec = (const uint4*)(b + parts[6].off); d.p3cls = (const uint2*)(b + parts[7].off);
    d.p3flow = (const int4*)(b + parts[8].off); d.witem = (const unsigned*)(b + parts[9].off);
    d.p3clsh = (const int*)(b + parts[10].off);
    d.ncolor = t->ncolor; d.nflow = t->nflow; d.ncls = t->ncls; d.nsched = t->nsteps * c_nw; d.nitem = t->nitem;
    {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
    }
    for (int l = 0; l < 3; l++)
        for (int w = 0; w < 16; w++)
            d.p1sched[l][w] = w < c_nw ? make_int2(t->p1sched[2 * (l * c_nw + w)], t->p1sched[2 * (l * c_nw + w) + 1]) : make_int2(0, 0);
    switch (ngluon) {
#define HS_SET(N) case N: c->smem = smem_bytes<N>(t); c->threads = 32 * HsCfg<N>::NW; c->ctas = HsCfg<N>::CTAS; e = set_smem<N>(c->smem); break;
        HS_PROCESSES(HS_SET)
#undef HS_SET
        default: e = cudaErrorInvalidValue;
    }
    if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
    *out = c;
    return cudaSuccess;
}

void hs_destroy(HsContext* c)
{
    if (!c) return;
    cudaFree(c->blob);
    delete c;
}

cudaError_t hs_launch(const HsContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st)
{
    if (a.nevt <= 0) return cudaSuccess;
    const int full = c->sms * c->ctas;                // persistent CTAs: the small tables are staged once per CTA
    const int grid = a.nevt < full ? a.nevt : full;
    switch (c->ngluon) {
#define HS_GO(N)                                                                                           \
    case N:                                                                                                \
        if (jamps_fp64) hs_diagrams_kernel<N, double><<<grid, c->threads, c->smem, st>>>(c->d, a);          \
        else hs_diagrams_kernel<N, float><<<grid, c->threads, c->smem, st>>>(c->d, a);                      \
        break;
        HS_PROCESSES(HS_GO)
#undef HS_GO
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace mg
