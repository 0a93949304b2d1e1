// hsg_kernel.cu -- GENERIC helicity-shared diagram kernel (g g -> t tbar g g g g; Table 2,
// 15 495 diagrams, 720 colour flows, 256 helicities).  Interprets the tables of gen/hsg_tables.py.
//
// Same three phases as the tuned kernel of the smaller processes (hs_kernel.cu): colour-ordered objects of <= 4 legs, every
// helicity variant of their own legs once per event (phase 1); pair objects X = vertex contracted with all branches but the
// largest, Y (phase 2); jamp[sigma][h] = sum over entries of +- sum_c X_c[variant_x(h)] Y_c[variant_y(h)] (phase 3, thread =
// helicity combination).  What changes at this size: one event holds 5 984 object variants (383 KB) and 43 680 pair-object
// variants (2.8 MB) -- they cannot live in shared memory.  Each (persistent) CTA owns a scratch area in GLOBAL memory, written
// and re-read through L1/L2 by the same CTA: the paper's hand-off between diagram-group kernels through global memory
// (PAPER.md:424-444), but inside one kernel and with barriers instead of kernel boundaries.  All pair objects of an event are
// built once (one group of colour flows), so phase 3 runs the 720 flows without a barrier between them.
//
// Scratch layout: four component planes, byte(c, slot) = c * 16 * nslot + 16 * slot, so that the lanes of a warp (consecutive
// variants) read consecutive 16-byte words of one plane.
//
// Phase 3 has two forms (template parameter TENSOR, option "p3_tensor"): thread = helicity combination on the FP64 ALU
// (p3_entry8), which is bound by shared-memory bandwidth -- every lane fetches its own copies of the operands, 24 to 36 16-byte
// loads per entry for 128 DFMA -- and the FP64 tensor path (p3t_entry, default): the entry as 8 tiles of mma.sync.m8n8k4.f64,
// whose fragments are 8 to 10 loads per lane and entry, with the accumulator fragments in registers over a CLASS of entries
// (gen/hsg_tables.py) and one swizzled accumulator per warp in shared memory that collects the classes of a flow.
#include <stdint.h>

#include <vector>

#include "generated/hsg_gen.h"
#include "helas.cuh"
#include "hsg_kernel.cuh"

namespace mg {

struct HsgDev {
    const int4* obj; const int4* term; const int* p1_items; const int* legset_mask;
    const int2* xitem; const int4* entry; const int4* flow; const unsigned short* vtab;
    const int4* dentry; const unsigned* ltab; const unsigned* flowL; const unsigned* flowT;       // tensor path of phase 3
    int npar, ncolor, nslot, nlegsets, nxitem, nflow, nlevel;
    const unsigned char* lut; int nlut;   // sub-variant table [nlut][HSG_LUT_VARS] (copied to shared memory), nlut * HSG_LUT_VARS % 16 == 0
    int nslot_arg;             // slots [0, nslot_arg) = the objects of <= 3 legs: every argument of phases 1 and 2 is one of them
    int p3buf;                 // bytes of one phase-3 operand buffer: max over the entries of 64 (2^|X| + 2^|Y|) + 128
    int p1_level[8];
};

// measured (4096 events, diagrams): 256 threads x 2 CTAs per SM 39.0 ms, 256 x 3 (80 registers, spills) 47.2, 512 x 1 38.0
static constexpr int HSG_THREADS = 512, HSG_CTAS = 1;
// phase 3: operand buffers per warp (entries in flight: the one being evaluated and HSG_P3_STAGES - 1 being copied)
static constexpr int HSG_P3_STAGES = 2;          // (3 stages: 34.7 ms per 4096 events, 2: 33.7 -- the L1 cache left for phases 1 and 2 counts)

// fp32 -> TF32 (10 explicit significand bits), round to nearest: the tensor core would truncate
__device__ __forceinline__ float to_tf32(float x)
{
    unsigned u;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
    return __uint_as_float(u);
}

// variant of an argument object for variant var of its parent: bit j = bit ((code >> 3j) & 7) of var (7 = none).  There are few
// distinct codes (30 at 6 gluons): hsg_create numbers them, writes the number into the device copy of the term records in place
// of the code and tabulates the function -- the kernel reads lut[number][var] from shared memory (one load instead of ~20
// integer instructions per argument).
static int sub_variant4(int var, int code)
{
    return ((var >> (code & 7)) & 1) | (((var >> ((code >> 3) & 7)) & 1) << 1) | (((var >> ((code >> 6) & 7)) & 1) << 2) |
           (((var >> ((code >> 9) & 7)) & 1) << 3);
}
static constexpr int HSG_LUT_VARS = 128;          // variants of a parent: objects have <= 4 legs, pair objects <= 7

__device__ __forceinline__ void ldw(const char* __restrict__ area, size_t plane, int slot, wf<double>& w)
{
#pragma unroll
    for (int c = 0; c < 4; c++) {
        const double2 v = *reinterpret_cast<const double2*>(area + c * plane + 16 * (size_t)slot);
        w.c[c].re = v.x; w.c[c].im = v.y;
    }
}

__device__ __forceinline__ void stw(char* __restrict__ area, size_t plane, int slot, const wf<double>& w)
{
#pragma unroll
    for (int c = 0; c < 4; c++) *reinterpret_cast<double2*>(area + c * plane + 16 * (size_t)slot) = make_double2(w.c[c].re, w.c[c].im);
}

__device__ __forceinline__ p4<double> ldk(const double* __restrict__ Ks, int ls)
{
    p4<double> k = { Ks[4 * ls], Ks[4 * ls + 1], Ks[4 * ls + 2], Ks[4 * ls + 3] };
    return k;
}

__device__ __forceinline__ void axpy(double sg, const wf<double>& r, wf<double>& acc)
{
#pragma unroll
    for (int c = 0; c < 4; c++) { acc.c[c].re = fma(sg, r.c[c].re, acc.c[c].re); acc.c[c].im = fma(sg, r.c[c].im, acc.c[c].im); }
}

// one entry for the 8 helicity combinations q of particles 0, 1, 2 (bit i of q = particle i): XMASK = which of them are legs
// of X, LGX = number of legs of X (npar = 8: Y has 8 - LGX).  The three are the lowest-numbered particles, hence the HIGHEST
// bits of the variant index of whichever object holds them (descending particle order), index bit 0 = the largest of the three.
// bx = the entry's operand buffer in shared memory, [X: 4 components][2^LGX variants] then [Y: 4][2^(8 - LGX)], 16 bytes each;
// vx, vy = this lane's variants (its five helicities): every offset below is a compile-time immediate.
template <int XMASK, int LGX>
__device__ __forceinline__ void p3_entry8(const char* __restrict__ bx, unsigned vx, unsigned vy, double sg, double (&re)[8], double (&im)[8])
{
    constexpr int NFX = ((XMASK >> 0) & 1) + ((XMASK >> 1) & 1) + ((XMASK >> 2) & 1), NX = 1 << NFX, NY = 8 / NX;
    constexpr int LGY = 8 - LGX, LX = LGX - NFX, LY = LGY - (3 - NFX);
    static_assert(LX >= 0 && LY >= 0, "impossible entry kind");
    const char* __restrict__ px = bx + 16 * vx;
    const char* __restrict__ py = bx + (64 << LGX) + 16 * vy;
#pragma unroll
    for (int c = 0; c < 4; c++) {
        double2 x[NX], y[NY];
#pragma unroll
        for (int i = 0; i < NX; i++) {
            x[i] = *reinterpret_cast<const double2*>(px + c * (16 << LGX) + i * (16 << LX));
            if (NX < NY) { x[i].x *= sg; x[i].y *= sg; }
        }
#pragma unroll
        for (int i = 0; i < NY; i++) {
            y[i] = *reinterpret_cast<const double2*>(py + c * (16 << LGY) + i * (16 << LY));
            if (NX >= NY) { y[i].x *= sg; y[i].y *= sg; }
        }
#pragma unroll
        for (int q = 0; q < 8; q++) {
            int xo = 0, yo = 0, nx = 0, ny = 0;
#pragma unroll
            for (int b = 2; b >= 0; b--) {
                if ((XMASK >> b) & 1) { xo |= ((q >> b) & 1) << nx; nx++; }
                else { yo |= ((q >> b) & 1) << ny; ny++; }
            }
            re[q] = fma(x[xo].x, y[yo].x, re[q]); re[q] = fma(-x[xo].y, y[yo].y, re[q]);
            im[q] = fma(x[xo].x, y[yo].y, im[q]); im[q] = fma(x[xo].y, y[yo].x, im[q]);
        }
    }
}

// copy of an entry's operands from the CTA's scratch area (planes of `plane` bytes; xs, ys = first slots of X and Y) into the
// warp's buffer dst (shared-memory address): 4 x 2^LGX + 4 x 2^(8 - LGX) pieces of 16 bytes, lane = piece % 32
template <int LGX>
__device__ __forceinline__ void p3_stage(const char* __restrict__ area, unsigned plane, int xs, int ys, unsigned dst, int lane)
{
    constexpr int LGY = 8 - LGX, NX4 = 4 << LGX, NY4 = 4 << LGY;
#pragma unroll
    for (int t = 0; t < NX4 / 32; t++) {
        const int i = lane + 32 * t;
        const char* src = area + ((unsigned)(i >> LGX) * plane + 16u * (unsigned)(xs + (i & ((1 << LGX) - 1))));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * (unsigned)i), "l"(src) : "memory");
    }
#pragma unroll
    for (int t = 0; t < (NY4 + 31) / 32; t++) {
        const int i = lane + 32 * t;
        if (NY4 % 32 == 0 || i < NY4) {
            const char* src = area + ((unsigned)(i >> LGY) * plane + 16u * (unsigned)(ys + (i & ((1 << LGY) - 1))));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * (unsigned)(NX4 + i)), "l"(src) : "memory");
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// phase 3 on the FP64 tensor path.  One entry = out[hp][hq] += sum_c P_c[hp] Q_c[hq] (complex, c = 4 components) for all 256
// helicity combinations = 8 tiles of mma.sync.m8n8k4.f64: rows = the helicities of the class's three particles R (legs of P),
// column pairs (re, im) = those of its two particles C (legs of Q), tile = those of the remaining three particles T.
// Fragments: a = A[lane / 4][lane % 4] = P_c[row variant] (c = lane % 4; re and im in one 16-byte load), b = B[lane % 4][lane / 4]
// = Re or Im of Q_c[column variant], c0, c1 = C[lane / 4][2 (lane % 4) + {0, 1}].  The two k-steps of a tile, Re P . (Re Q | Im Q)
// and Im P . (-Im Q | Re Q), go to ONE accumulator pair f[2t + {0, 1}] = (re, im): the minus sits on the B fragment of the second
// step (a sign bit in the lanes of the even columns), and the eight first steps are issued before the eight second ones.  (The
// tuned kernel keeps two pairs per tile instead, hs_kernel.cu; here 32 fewer registers and half the flush.)  MASK: tile bits whose particle is a leg of P (they select
// the A fragment, the others the B fragment); d0..d2 = byte distance of the variants that differ in that particle's helicity.
__device__ __forceinline__ void hsg_dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__host__ __device__ constexpr int hsg_popc3(int m) { return (m & 1) + ((m >> 1) & 1) + ((m >> 2) & 1); }
// bits of t selected by mask m, packed
__host__ __device__ constexpr int hsg_pext3(int t, int m)
{
    int r = 0, k = 0;
    for (int b = 0; b < 3; b++)
        if ((m >> b) & 1) { r |= ((t >> b) & 1) << k; k++; }
    return r;
}

__device__ __forceinline__ double hsg_flip(double v, unsigned smask)
{
    return __hiloint2double(__double2hiint(v) ^ (int)smask, __double2loint(v));
}

template <int MASK>
__device__ __forceinline__ void p3t_entry(const char* __restrict__ bx, unsigned aoff, unsigned boff, unsigned d0, unsigned d1,
                                          unsigned d2, unsigned smask, unsigned nmask, double (&f)[16])
{
    constexpr int NA = 1 << hsg_popc3(MASK), NB = 8 / NA;
    const unsigned d[3] = { d0, d1, d2 };
    double2 xa[NA];
    double b0[NB], b1[NB];
#pragma unroll
    for (int a = 0; a < NA; a++) {
        unsigned off = aoff;
        int k = 0;
#pragma unroll
        for (int i = 0; i < 3; i++)
            if ((MASK >> i) & 1) { if ((a >> k) & 1) off += d[i]; k++; }
        xa[a] = *reinterpret_cast<const double2*>(bx + off);
    }
#pragma unroll
    for (int b = 0; b < NB; b++) {
        unsigned off = boff;
        int k = 0;
#pragma unroll
        for (int i = 0; i < 3; i++)
            if (!((MASK >> i) & 1)) { if ((b >> k) & 1) off += d[i]; k++; }
        b0[b] = *reinterpret_cast<const double*>(bx + off);            // even column (re out): Re Q, odd: Im Q
        b1[b] = *reinterpret_cast<const double*>(bx + (off ^ 8u));     // even column: Im Q, odd: Re Q
    }
    // signs: the entry's (smask) on one operand; the minus of Im P . Im Q (nmask: set in the lanes of even columns) on b1 or,
    // where the B fragments are the many, folded into the A side as a second copy of Im P is not worth it: it stays on b1
    if constexpr (NA <= NB) {
#pragma unroll
        for (int a = 0; a < NA; a++) { xa[a].x = hsg_flip(xa[a].x, smask); xa[a].y = hsg_flip(xa[a].y, smask); }
#pragma unroll
        for (int b = 0; b < NB; b++) b1[b] = hsg_flip(b1[b], nmask);
    } else {
#pragma unroll
        for (int b = 0; b < NB; b++) { b0[b] = hsg_flip(b0[b], smask); b1[b] = hsg_flip(b1[b], smask ^ nmask); }
    }
    // all Re P products first, then the Im P ones: the two tensor instructions of a tile are 8 apart
#pragma unroll
    for (int t = 0; t < 8; t++) hsg_dmma884(f[2 * t], f[2 * t + 1], xa[hsg_pext3(t, MASK)].x, b0[hsg_pext3(t, ~MASK & 7)]);
#pragma unroll
    for (int t = 0; t < 8; t++) hsg_dmma884(f[2 * t], f[2 * t + 1], xa[hsg_pext3(t, MASK)].y, b1[hsg_pext3(t, ~MASK & 7)]);
}

// 16-byte slot of helicity combination h in a warp's flow accumulator (gen/hsg_tables.py acc_swz)
__device__ __forceinline__ unsigned acc_swz(unsigned h)
{
    const unsigned hi = h >> 3;
    return h ^ (((hi & 1) * 3) ^ (((hi >> 1) & 1) * 5) ^ (((hi >> 2) & 1) * 6) ^ (((hi >> 3) & 1) * 7) ^ ((hi >> 4) & 1));
}

// Class changes.  The flow's running sum lives in the accumulator fragments: when a class ends they are STORED to the warp's
// accumulator in shared memory (slot of the lane's elements for tile t: L ^ byte t of (tw0, tw1); the swizzle is linear), and the
// next class LOADS them back in its own (lane, tile) order -- the tensor instructions then add onto them.  No FP64 additions: a
// flush by read-add-write put 16 DADDs per class behind the other warps' tensor instructions in the FP64 pipe's queue.
__device__ __forceinline__ void p3t_store(char* __restrict__ acc, unsigned L, unsigned tw0, unsigned tw1, const double (&f)[16])
{
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const unsigned idx = L ^ (((t < 4 ? tw0 : tw1) >> (8 * (t & 3))) & 0xFFu);
        *reinterpret_cast<double2*>(acc + 16u * idx) = make_double2(f[2 * t], f[2 * t + 1]);
    }
}
__device__ __forceinline__ void p3t_load(const char* __restrict__ acc, unsigned L, unsigned tw0, unsigned tw1, double (&f)[16])
{
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const unsigned idx = L ^ (((t < 4 ? tw0 : tw1) >> (8 * (t & 3))) & 0xFFu);
        const double2 v = *reinterpret_cast<const double2*>(acc + 16u * idx);
        f[2 * t] = v.x; f[2 * t + 1] = v.y;
    }
}

// variant index with bits 2 and sw exchanged (sw = 2: unchanged)
__device__ __forceinline__ int swap2(int v, int sw)
{
    const int x = ((v >> 2) ^ (v >> sw)) & 1;
    return v ^ (x << 2) ^ (x << sw);
}

// the tensor path's copy of an entry's operands: component planes of (2^LG + 1) x 16 bytes (X: four planes, then Y), and inside a
// plane the variant index has bits 2 and swx (swy) exchanged.  With that the lanes of one shared-memory access phase of a fragment
// load -- the four components times the helicity of the class's R[0] (16-byte A elements, 8 lanes) or of C[0] and re / im (8-byte
// B elements, 16 lanes) -- fall into different banks (gen/hsg_tables.py staged; checked for every entry: no conflict on A, a
// two-way one on B only where Y has two legs).
template <int LGX>
__device__ __forceinline__ void p3t_stage(const char* __restrict__ area, unsigned plane, int xs, int ys, unsigned dst, int lane,
                                          int swx, int swy)
{
    constexpr int LGY = 8 - LGX, NX4 = 4 << LGX, NY4 = 4 << LGY;
    constexpr unsigned PSX = (16u << LGX) + 16u, PSY = (16u << LGY) + 16u;
#pragma unroll
    for (int t = 0; t < NX4 / 32; t++) {
        const int i = lane + 32 * t, c = i >> LGX, v = i & ((1 << LGX) - 1);
        const char* src = area + ((unsigned)c * plane + 16u * (unsigned)(xs + swap2(v, swx)));
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + (unsigned)c * PSX + 16u * (unsigned)v), "l"(src) : "memory");
    }
#pragma unroll
    for (int t = 0; t < (NY4 + 31) / 32; t++) {
        const int i = lane + 32 * t, c = i >> LGY, v = i & ((1 << LGY) - 1);
        if (NY4 % 32 == 0 || i < NY4) {
            const char* src = area + ((unsigned)c * plane + 16u * (unsigned)(ys + swap2(v, swy)));
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 4u * PSX + (unsigned)c * PSY + 16u * (unsigned)v), "l"(src)
                         : "memory");
        }
    }
}

// T2 = type of the jamps buffer; TENSOR: phase 3 on the FP64 tensor path
template <typename T2, bool TENSOR>
__global__ void __launch_bounds__(HSG_THREADS, HSG_CTAS) hsg_diagrams_kernel(const HsgDev d, const HsLaunch a, char* __restrict__ scratch)
{
    extern __shared__ __align__(16) double smd[];
    double* __restrict__ Ks = smd;                               // [nlegsets][4]
    double* __restrict__ pm = smd + 4 * d.nlegsets;              // [npar][4]
    unsigned char* __restrict__ lut = reinterpret_cast<unsigned char*>(pm + 4 * d.npar);     // [nlut][HSG_LUT_VARS]
    char* __restrict__ p3base = reinterpret_cast<char*>(lut) + d.nlut * HSG_LUT_VARS;        // [warp][HSG_P3_STAGES][p3buf]: operands of phase 3
    // TENSOR: [warp][2^npar][16 B] flow accumulators behind the operand buffers
    char* __restrict__ accbase = p3base + (size_t)(HSG_THREADS / 32) * HSG_P3_STAGES * d.p3buf;
    // TENSOR: [2^npar] element offset of helicity combination h of the current event in the jamps buffer (without the colour's
    // part), -1 = not computed: the write-out of a flow costs one load per element instead of the layout arithmetic
    long long* __restrict__ rofft = reinterpret_cast<long long*>(accbase + (size_t)(HSG_THREADS / 32) * (16u << 8));
    const int tid = threadIdx.x, NT = HSG_THREADS;
    const int npar = d.npar, nh = 1 << npar;
    const size_t plane = 16 * (size_t)d.nslot;
    char* __restrict__ area = scratch + (size_t)blockIdx.x * 4 * plane;
    T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
    int posq[8];                 // rows of this lane's 8 helicity combinations (phase 3; npar = 8: the low five bits = lane)
#pragma unroll
    for (int q = 0; q < 8; q++)
        posq[q] = a.d_pos[(tid & 31) | ((q & 1) << (npar - 1)) | (((q >> 1) & 1) << (npar - 2)) | (((q >> 2) & 1) << (npar - 3))];
    // Arguments of phases 1 and 2 are objects of <= 3 legs only (1 184 slots = 76 KB at 6 gluons; hsg_create checks it): they are
    // kept in SHARED memory, in the area phase 3 uses for its operand buffers afterwards, besides their copy in the scratch area
    // (which phase 3 reads as Y).  With them in the scratch area alone every term of phases 1 and 2 waited for an L2 round trip
    // (L1 hit rate 14 %: the L1 left beside 210 KB of shared memory is small).
    char* __restrict__ argarea = p3base;
    const size_t aplane = 16 * (size_t)d.nslot_arg;
    for (int i = threadIdx.x; i < d.nlut * HSG_LUT_VARS / 4; i += HSG_THREADS)
        reinterpret_cast<unsigned*>(lut)[i] = __ldg(reinterpret_cast<const unsigned*>(d.lut) + i);       // (first use: after a barrier)
    auto arg = [&](int word, int var, wf<double>& w) {
        ldw(argarea, aplane, (word & 0xFFFF) + lut[((word >> 16) & 0xFFF) * HSG_LUT_VARS + var], w);
    };

    for (int e = blockIdx.x; e < a.nevt; e += gridDim.x) {
        // a0: momenta (AOS fp64) -> shared; leg-set momenta in the all-incoming convention
        for (int i = tid; i < 4 * npar; i += NT) pm[i] = a.mom[(size_t)e * (4 * npar) + i];
        if constexpr (TENSOR) {
            for (int h = tid; h < nh; h += NT) {
                const int pos = a.d_pos[h];
                const size_t row = (size_t)e * a.nrow_evt + pos;
                rofft[h] = pos < 0 ? -1ll
                           : a.tile_major == 2 ? (long long)((row >> 7) * (size_t)(256 * d.ncolor) + ((row & 127) >> 3) * 192 + (row & 7) * 4)
                                               : (long long)row;
            }
        }
        __syncthreads();
        for (int s = tid; s < d.nlegsets; s += NT) {
            const int m = __ldg(d.legset_mask + s);
            double k0 = 0, k1 = 0, k2 = 0, k3 = 0;
            for (int p = 0; p < npar; p++)
                if ((m >> p) & 1) {
                    const double sg = p < 2 ? 1.0 : -1.0;
                    k0 += sg * pm[4 * p]; k1 += sg * pm[4 * p + 1]; k2 += sg * pm[4 * p + 2]; k3 += sg * pm[4 * p + 3];
                }
            Ks[4 * s] = k0; Ks[4 * s + 1] = k1; Ks[4 * s + 2] = k2; Ks[4 * s + 3] = k3;
        }
        __syncthreads();
        // phase 1: colour-ordered objects, level by level (an object of L legs reads objects of fewer legs only)
        for (int lvl = 0; lvl < d.nlevel; lvl++) {
            for (int i = d.p1_level[lvl] + tid; i < d.p1_level[lvl + 1]; i += NT) {
                const int it = __ldg(d.p1_items + i);
                const int4 o = __ldg(d.obj + (it >> 8));
                const int var = it & 0xFF;
                const p4<double> K = ldk(Ks, o.y >> 8);
                wf<double> acc;
#pragma unroll
                for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
                for (int t = 0; t < o.w; t++) {
                    const int4 w = __ldg(d.term + o.z + t);
                    const int op = w.x & 0xFF;
                    wf<double> r;
                    if (op <= 2) {
                        const int hel = (var & 1) ? 1 : -1;
                        const double* p = pm + 4 * w.y;
                        if (op == 0) ext_eps(p, hel, w.y >= 2, r);
                        else if (op == 1) ext_ubar(p, a.mt, hel, r);
                        else ext_v(p, a.mt, hel, r);
                    } else {
                        wf<double> A, B;
                        arg(w.y, var, A); arg(w.z, var, B);
                        switch (op) {
                            case 3: v3_off(A, ldk(Ks, (w.x >> 16) & 0xFF), B, ldk(Ks, (w.x >> 24) & 0xFF), 1.0 / m2(K), r); break;
                            case 4: { wf<double> Z; arg(w.w, var, Z); v4_off(A, B, Z, 1.0 / m2(K), r); break; }
                            case 5: ffv_l(A, B, -K, a.mt, inv_prop(m2(K), a.mt, a.wt), r); break;
                            case 6: ffv_r(A, B, K, a.mt, inv_prop(m2(K), a.mt, a.wt), r); break;
                            default: ffv_p(A, B, 1.0 / m2(K), r); break;       // 7
                        }
                    }
                    axpy((w.x >> 8) & 1 ? -1.0 : 1.0, r, acc);
                }
                stw(area, plane, o.x + var, acc);
                if (o.x < d.nslot_arg) stw(argarea, aplane, o.x + var, acc);
            }
            __syncthreads();
        }
        // phase 2: pair objects (raw vertices; vector-valued ones lowered at the store for the plain dot of phase 3)
        for (int i = tid; i < d.nxitem; i += NT) {
            const int2 it = __ldg(d.xitem + i);
            const int t0 = it.x & 0xFFFFFF, nt = (int)((unsigned)it.x >> 24);
            const int slot = it.y & 0xFFFFF, var = (it.y >> 20) & 0xFF;
            wf<double> acc;
#pragma unroll
            for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
            for (int t = 0; t < nt; t++) {
                const int4 w = __ldg(d.term + t0 + t);
                const int op = w.x & 0xFF;
                wf<double> A, B, q;
                arg(w.y, var, A); arg(w.z, var, B);
                switch (op) {
                    case 8: row_slash(A, make_slashed(B), q); break;
                    case 9: slash_col(make_slashed(A), B, q); break;
                    case 10: ffv_p_raw(A, B, q); break;
                    case 11: v3_raw(A, ldk(Ks, (w.x >> 16) & 0xFF), B, ldk(Ks, (w.x >> 24) & 0xFF), q); break;
                    case 12: { wf<double> Z; arg(w.w, var, Z); v4_raw(A, B, Z, q); break; }
                    default: {                                              // 13: 2 (A.Z) B - (B.Z) A - (B.A) Z
                        wf<double> Z; arg(w.w, var, Z);
                        cx<double> xz = dot(A, Z);
                        xz = xz + xz;
                        const cx<double> yz = dot(B, Z), yx = dot(B, A);
#pragma unroll
                        for (int mu = 0; mu < 4; mu++) q.c[mu] = cfms(yx, Z.c[mu], cfms(yz, A.c[mu], xz * B.c[mu]));
                        break;
                    }
                }
                axpy((w.x >> 8) & 1 ? -1.0 : 1.0, q, acc);
            }
            if ((it.y >> 28) & 1) {
#pragma unroll
                for (int c = 1; c < 4; c++) acc.c[c] = -acc.c[c];
            }
            stw(area, plane, slot, acc);
        }
        __syncthreads();
        // phase 3: the colour flows, one warp per flow: lane = helicities of particles 3 .. npar-1 (the low bits of h), and
        // every thread carries the 8 helicity combinations of particles 0, 1, 2 in registers: 2^nx variants of X and 2^(3-nx) of
        // Y serve 8 dot products (9 or 6 wavefunction loads instead of 16), p3_entry8.  Variant indices run over the legs in
        // DESCENDING particle order, so the lanes of the warp read one contiguous run of slots per load.
        // The operands of an entry -- ALL variants of X and of Y, 2 to 4.3 KB -- are copied from the scratch area (L2: the area
        // is 3.2 MB, the L1 hit rate of direct loads was 51 %) into a shared-memory buffer of the warp by cp.async,
        // HSG_P3_STAGES - 1 entries ahead of the one being evaluated: the L2 latency, which bounded the kernel (four dependent
        // batches of loads per entry at 16 warps per SM), is off the critical path.
        if constexpr (TENSOR) {
            // tensor path: one warp per flow; the entries of a flow come class by class (gen/hsg_tables.py).  Staging and
            // prefetching as in the ALU form below: the operands of entry k + 1 are copied while entry k is evaluated, the
            // per-lane fragment offsets (ltab) of entry k + 1 and the records and class tables of the warp's NEXT flow are in
            // flight meanwhile.
            const int lane = tid & 31;
            char* __restrict__ wbuf = p3base + (size_t)(tid >> 5) * (HSG_P3_STAGES * d.p3buf);
            char* __restrict__ acc = accbase + (size_t)(tid >> 5) * (16u << 8);
            const unsigned wbuf_s = (unsigned)__cvta_generic_to_shared(wbuf);
            auto stage = [&](const int4 en, int b) {
                const unsigned dst = wbuf_s + (unsigned)(b * d.p3buf);
                const int xs = en.x & 0xFFFF, ys = (int)((unsigned)en.x >> 16), swx = (en.w >> 16) & 0xF, swy = (en.w >> 20) & 0xF;
                switch ((en.y >> 16) & 0xF) {
                    case 4: p3t_stage<4>(area, (unsigned)plane, xs, ys, dst, lane, swx, swy); break;
                    case 5: p3t_stage<5>(area, (unsigned)plane, xs, ys, dst, lane, swx, swy); break;
                    default: p3t_stage<6>(area, (unsigned)plane, xs, ys, dst, lane, swx, swy); break;
                }
            };
            const int NWARP = NT >> 5;
            auto bcast = [&](const int4 m, int k) {
                return make_int4(__shfl_sync(0xffffffffu, m.x, k), __shfl_sync(0xffffffffu, m.y, k), __shfl_sync(0xffffffffu, m.z, k),
                                 __shfl_sync(0xffffffffu, m.w, k));
            };
            const unsigned* __restrict__ lt = d.ltab + lane;
            int f = tid >> 5;
            int4 fl = make_int4(0, 0, 0, 0), myent = fl;
            unsigned v = 0, myL = 0, myT = 0;
            if (f < d.nflow) {
                fl = __ldg(d.flow + f);
                if (lane < fl.z) myent = __ldg(d.dentry + fl.y + lane);
                myL = __ldg(d.flowL + 32 * f + lane);
                myT = __ldg(d.flowT + 8 * f + (lane & 7));
                v = __ldg(lt + 32 * (size_t)(__shfl_sync(0xffffffffu, myent.y, 0) & 0xFFFF));
            }
            double fr[16];
#pragma unroll
            for (int i = 0; i < 16; i++) fr[i] = 0.0;
            const unsigned nmask = (lane & 4) ? 0u : 0x80000000u;          // lanes of the even columns of the B fragment
            for (; f < d.nflow; f += NWARP) {
                const int fn = f + NWARP;
                int4 fl_n = make_int4(0, 0, 0, 0), myent_n = fl_n;
                unsigned myL_n = 0, myT_n = 0;
                if (fn < d.nflow) fl_n = __ldg(d.flow + fn);
                static_assert(HSG_P3_STAGES == 2, "the record of the entry being copied is kept for the next iteration");
                int4 nxt = bcast(myent, 0);
                if (fl.z > 0) stage(nxt, 0);
                asm volatile("cp.async.commit_group;" ::: "memory");     // one commit group per entry, empty past the end
                int bcur = 0, bnew = 1, cls = 0;
                bool pend = false;
                unsigned pL = 0, ptw0 = 0, ptw1 = 0;
                for (int k = 0; k < fl.z; k++) {
                    const int4 cur = nxt;
                    if (k + 1 < fl.z) { nxt = bcast(myent, k + 1); stage(nxt, bnew); }
                    asm volatile("cp.async.commit_group;" ::: "memory");
                    const unsigned cv = v;
                    if (k == 0 && fn < d.nflow) {
                        if (lane < fl_n.z) myent_n = __ldg(d.dentry + fl_n.y + lane);
                        myL_n = __ldg(d.flowL + 32 * fn + lane);
                        myT_n = __ldg(d.flowT + 8 * fn + (lane & 7));
                    }
                    if (k + 1 < fl.z) v = __ldg(lt + 32 * (size_t)(__shfl_sync(0xffffffffu, myent.y, k + 1) & 0xFFFF));
                    else if (fn < d.nflow) v = __ldg(lt + 32 * (size_t)(__shfl_sync(0xffffffffu, myent_n.y, 0) & 0xFFFF));
                    // the class that ended with the previous entry is stored HERE, behind the copy and the prefetches of this
                    // iteration (its last tensor instructions have ~200 cycles of latency), and the running sum comes back in the
                    // order of this entry's class
                    if (pend) {
                        p3t_store(acc, pL, ptw0, ptw1, fr);
                        __syncwarp();
                        p3t_load(acc, (myL >> (8 * cls)) & 0xFFu, __shfl_sync(0xffffffffu, myT, 2 * cls),
                                 __shfl_sync(0xffffffffu, myT, 2 * cls + 1), fr);           // (cls = the class of entry k)
                        pend = false;
                    }
                    asm volatile("cp.async.wait_group %0;" ::"n"(HSG_P3_STAGES - 1) : "memory");
                    __syncwarp();
                    const char* __restrict__ bx = wbuf + bcur * d.p3buf;
                    const unsigned smask = ((unsigned)cur.y << 8) & 0x80000000u;
                    const unsigned d0 = cur.z & 0xFFFF, d1 = (unsigned)cur.z >> 16, d2 = cur.w & 0xFFFF;
                    switch ((cur.y >> 20) & 7) {
#define HSG_P3T_CASE(M) case M: p3t_entry<M>(bx, cv & 0xFFFFu, cv >> 16, d0, d1, d2, smask, nmask, fr); break;
                        HSG_P3T_MASKS(HSG_P3T_CASE)
#undef HSG_P3T_CASE
                        default: break;                                  // (hsg_create refuses tables with another mask)
                    }
                    if (cur.y & (1 << 24)) {                             // last entry of its class (uniform over the warp)
                        ptw0 = __shfl_sync(0xffffffffu, myT, 2 * cls); ptw1 = __shfl_sync(0xffffffffu, myT, 2 * cls + 1);
                        pL = (myL >> (8 * cls)) & 0xFFu;
                        pend = true;
                        cls++;
                    }
                    __syncwarp();                                        // the buffer is free for the copy of entry k + STAGES
                    bnew = bcur;
                    bcur = bcur + 1 == HSG_P3_STAGES ? 0 : bcur + 1;
                }
                if (pend) { p3t_store(acc, pL, ptw0, ptw1, fr); pend = false; }     // (a flow ends with the end of a class)
#pragma unroll
                for (int i = 0; i < 16; i++) fr[i] = 0.0;                 // the next flow starts from zero
                __syncwarp();
                // the finished jamp of this flow: lane = the helicities of particles 3 .. 7 (low bits of h), q = particles 0, 1, 2
                {
                    const int jc = fl.x;
                    // tcgen05 operand layout (color_sum_tf32_big.cu): per 128-row tile and part, chunks of 24 colours as K-major
                    // core matrices [row / 8][colour quad][row % 8][colour % 4], values rounded to TF32; the row's part is in rofft
                    const size_t joff = a.tile_major == 2 ? (size_t)(jc / 24) * (24 * 128) + ((jc % 24) >> 2) * 32 + (jc & 3)
                                                          : (size_t)jc * a.rows;
#pragma unroll
                    for (int q = 0; q < 8; q++) {
                        const unsigned h = (unsigned)lane | ((q & 1u) << 7) | (((q >> 1) & 1u) << 6) | (((q >> 2) & 1u) << 5);
                        const long long ro = rofft[h];
                        if (ro >= 0) {
                            const double2 val = *reinterpret_cast<const double2*>(acc + 16u * acc_swz(h));
                            if (a.tile_major == 2) {
                                if constexpr (sizeof(T2) == 4) {
                                    float* __restrict__ o = reinterpret_cast<float*>(out) + (size_t)ro + joff;
                                    o[0] = to_tf32((float)val.x); o[(size_t)d.ncolor * 128] = to_tf32((float)val.y);
                                }
                            } else {
                                out[joff + (size_t)ro] = T2(val.x);
                                out[(size_t)d.ncolor * a.rows + joff + (size_t)ro] = T2(val.y);
                            }
                        }
                    }
                }
                __syncwarp();                                            // the next flow's first class overwrites the accumulator
                fl = fl_n; myent = myent_n; myL = myL_n; myT = myT_n;
            }
        } else
        {
            const int lane = tid & 31;
            char* __restrict__ wbuf = p3base + (size_t)(tid >> 5) * (HSG_P3_STAGES * d.p3buf);
            const unsigned wbuf_s = (unsigned)__cvta_generic_to_shared(wbuf);
            auto stage = [&](const int4 en, int b) {
                const unsigned dst = wbuf_s + (unsigned)(b * d.p3buf);
                switch (((en.w >> 4) & 7) + __popc((en.w >> 1) & 7)) {
                    case 4: p3_stage<4>(area, (unsigned)plane, en.x, en.y, dst, lane); break;
                    case 5: p3_stage<5>(area, (unsigned)plane, en.x, en.y, dst, lane); break;
                    default: p3_stage<6>(area, (unsigned)plane, en.x, en.y, dst, lane); break;
                }
            };
            // Nothing a warp needs next may wait for memory: the flow header and the entry records of the warp's NEXT flow are
            // fetched while the current one runs (lane i keeps entry i; an entry's record reaches all lanes by shuffles), and
            // the variant lookup of entry k + 1 is fetched while entry k is evaluated.  (With 143 KB of the SM's memory in use as
            // shared memory the L1 cache is small and mostly holds the operands of phases 1 and 2: a table read is often an L2
            // round trip.)
            const int NWARP = NT >> 5;
            auto bcast = [&](const int4 m, int k) {
                return make_int4(__shfl_sync(0xffffffffu, m.x, k), __shfl_sync(0xffffffffu, m.y, k), __shfl_sync(0xffffffffu, m.z, k),
                                 __shfl_sync(0xffffffffu, m.w, k));
            };
            const unsigned short* __restrict__ vt = d.vtab + lane;
            int f = tid >> 5;
            int4 fl = make_int4(0, 0, 0, 0), myent = fl;
            unsigned v = 0;
            if (f < d.nflow) {
                fl = __ldg(d.flow + f);
                if (lane < fl.z) myent = __ldg(d.entry + fl.y + lane);
                v = __ldg(vt + (size_t)__shfl_sync(0xffffffffu, myent.z, 0) * nh);
            }
            for (; f < d.nflow; f += NWARP) {
                const int fn = f + NWARP;
                int4 fl_n = make_int4(0, 0, 0, 0), myent_n = fl_n;
                if (fn < d.nflow) fl_n = __ldg(d.flow + fn);
                double re[8], im[8];
#pragma unroll
                for (int q = 0; q < 8; q++) re[q] = im[q] = 0.0;
#pragma unroll
                for (int k = 0; k < HSG_P3_STAGES - 1; k++) {            // one commit group per entry, empty past the end
                    if (k < fl.z) stage(bcast(myent, k), k);
                    asm volatile("cp.async.commit_group;" ::: "memory");
                }
                int bcur = 0, bnew = HSG_P3_STAGES - 1;
                for (int k = 0; k < fl.z; k++) {
                    if (k + HSG_P3_STAGES - 1 < fl.z) stage(bcast(myent, k + HSG_P3_STAGES - 1), bnew);
                    asm volatile("cp.async.commit_group;" ::: "memory");
                    const int4 cur = bcast(myent, k);
                    const unsigned cv = v;
                    if (k == 0 && fn < d.nflow && lane < fl_n.z) myent_n = __ldg(d.entry + fl_n.y + lane);
                    if (k + 1 < fl.z) v = __ldg(vt + (size_t)__shfl_sync(0xffffffffu, myent.z, k + 1) * nh);
                    else if (fn < d.nflow) v = __ldg(vt + (size_t)__shfl_sync(0xffffffffu, myent_n.z, 0) * nh);
                    asm volatile("cp.async.wait_group %0;" ::"n"(HSG_P3_STAGES - 1) : "memory");
                    __syncwarp();
                    const char* __restrict__ bx = wbuf + bcur * d.p3buf;
                    const double sg = (cur.w & 1) ? -1.0 : 1.0;
                    const int lgx = ((cur.w >> 4) & 7) + __popc((cur.w >> 1) & 7);
                    switch (((cur.w >> 1) & 7) | (lgx << 3)) {
#define HSG_P3_CASE(M, LG) case (M) | ((LG) << 3): p3_entry8<M, LG>(bx, cv & 0xFFu, cv >> 8, sg, re, im); break;
                        HSG_P3_COMBOS(HSG_P3_CASE)
#undef HSG_P3_CASE
                        default: break;                                  // (hsg_create refuses tables with another kind)
                    }
                    __syncwarp();                                        // the buffer is free for the copy of entry k + STAGES
                    bnew = bcur;
                    bcur = bcur + 1 == HSG_P3_STAGES ? 0 : bcur + 1;
                }
#pragma unroll
                for (int q = 0; q < 8; q++) {
                    const int pos = posq[q];          // q bit i = helicity of particle i = bit npar-1-i of h; the low bits = lane
                    if (pos >= 0) {
                        const size_t row = (size_t)e * a.nrow_evt + pos;
                        if (a.tile_major == 2) {
                            // tcgen05 operand layout (color_sum_tf32_big.cu): per 128-row tile and part, chunks of 24 colours as
                            // K-major core matrices [row / 8][colour quad][row % 8][colour % 4], values rounded to TF32
                            if constexpr (sizeof(T2) == 4) {
                                const unsigned m = (unsigned)(row & 127);
                                const int jc = fl.x;
                                float* __restrict__ o = reinterpret_cast<float*>(out) + (row >> 7) * (size_t)(256 * d.ncolor) +
                                                        (size_t)(jc / 24) * (24 * 128) + (m >> 3) * 192 + ((jc % 24) >> 2) * 32 + (m & 7) * 4 + (jc & 3);
                                o[0] = to_tf32((float)re[q]); o[(size_t)d.ncolor * 128] = to_tf32((float)im[q]);
                            }
                        } else {
                            out[(size_t)fl.x * a.rows + row] = T2(re[q]);
                            out[(size_t)(d.ncolor + fl.x) * a.rows + row] = T2(im[q]);
                        }
                    }
                }
                fl = fl_n; myent = myent_n;
            }
        }
        __syncthreads();                 // the next event overwrites the scratch area
    }
}

// ------------------------------------------------------------------------------------------------------------
struct HsgContext {
    const HsgTables* t = nullptr;
    HsgDev d;
    void* blob = nullptr;
    char* scratch = nullptr;
    int grid = 0;
    size_t smem = 0, smem_alu = 0;   // dynamic shared memory with phase 3 on the tensor path / on the FP64 ALU
    bool tensor = true;              // option "p3_tensor"
    // hsg_launch_static: device address of hsg_static_scratch on this context's device (hsg_static_setup)
    char* static_scratch = nullptr;
    cudaError_t static_err = cudaErrorNotReady;
};

// Scratch areas for callers that cannot allocate (hsg_launch_static; include/mg5_b200.h mg_sigma_batch_noalloc): a file-scope
// array of HSG_STATIC_BYTES = 26 MiB, enough for 8 persistent CTAs of g g -> t tbar g g g g (8 x 3 178 496 B).  Every GPU that
// loads the library holds it until the process exits.  In HOST code this name is a host-side stand-in, not a device address:
// the address a kernel may be given comes from cudaGetSymbolAddress (hsg_static_setup), per device.  All calls share the array
// and it keeps the last call's contents; the kernel writes every slot of an event (phases 1 and 2) before it reads it (phase
// 3), so nothing has to start at zero -- but two such launches that overlap on the GPU race on it.
static constexpr size_t HSG_STATIC_BYTES = (size_t)26 << 20;
static constexpr int HSG_STATIC_CTAS = 8;
static __device__ __align__(256) unsigned char hsg_static_scratch[HSG_STATIC_BYTES];

const HsgTables* hsg_host_tables(const HsgContext* c) { return c->t; }

cudaError_t hsg_create(int ngluon, HsgContext** out)
{
    *out = nullptr;
    const HsgTables* t = hsg_tables(ngluon);
    if (!t) return cudaErrorInvalidValue;
    if (t->npar != 8) return cudaErrorInvalidValue;       // phase 3 maps lane = the helicities of particles 3 .. 7
    HsgContext* c = new HsgContext;
    c->t = t;
    // device copy of the term records: the 12-bit sub-variant code of every argument replaced by its row in the lookup table
    std::vector<int> term(t->term, t->term + 4 * (size_t)t->nterm);
    std::vector<int> codes;
    for (int i = 0; i < t->nterm; i++) {
        const int op = term[4 * i] & 0xFF;
        if (op <= 2) continue;
        const int nargs = (op == 4 || op == 12 || op == 13) ? 3 : 2;
        for (int k = 1; k <= nargs; k++) {
            const int code = (term[4 * i + k] >> 16) & 0xFFF;
            size_t r = 0;
            while (r < codes.size() && codes[r] != code) r++;
            if (r == codes.size()) codes.push_back(code);
            term[4 * i + k] = (term[4 * i + k] & 0xFFFF) | ((int)r << 16);
        }
    }
    while (codes.size() % 4) codes.push_back(0xFFF);                  // (rows of 128 bytes: any count is a multiple of 16 bytes)
    std::vector<unsigned char> lut(codes.size() * HSG_LUT_VARS);
    for (size_t r = 0; r < codes.size(); r++)
        for (int v = 0; v < HSG_LUT_VARS; v++) lut[r * HSG_LUT_VARS + v] = (unsigned char)sub_variant4(v, codes[r]);
    bool vars_ok = codes.size() <= 256;
    for (int i = 0; i < t->nxitem; i++) vars_ok = vars_ok && ((t->xitem[2 * i + 1] >> 20) & 0xFF) < HSG_LUT_VARS;
    if (!vars_ok) { delete c; return cudaErrorInvalidValue; }
    struct Part { const void* src; size_t bytes; size_t off; };
    Part parts[13] = { { t->obj, sizeof(int) * 4 * (size_t)t->nobj, 0 }, { term.data(), sizeof(int) * 4 * (size_t)t->nterm, 0 },
                      { t->p1_items, sizeof(int) * (size_t)t->np1, 0 }, { t->legset_mask, sizeof(int) * (size_t)t->nlegsets, 0 },
                      { t->xitem, sizeof(int) * 2 * (size_t)t->nxitem, 0 }, { t->entry, sizeof(int) * 4 * (size_t)t->nentry, 0 },
                      { t->flow, sizeof(int) * 4 * (size_t)t->nflow, 0 },
                      { t->vtab, sizeof(unsigned short) * ((size_t)t->nvrow << t->npar), 0 },
                      { t->dentry, sizeof(int) * 4 * (size_t)t->nentry, 0 }, { t->ltab, sizeof(unsigned) * 32 * (size_t)t->nlrow, 0 },
                      { t->flowL, sizeof(unsigned) * 32 * (size_t)t->nflow, 0 }, { t->flowT, sizeof(unsigned) * 8 * (size_t)t->nflow, 0 },
                      { lut.data(), lut.size(), 0 } };
    size_t total = 0;
    for (auto& p : parts) { p.off = total; total += (p.bytes + 255) & ~size_t(255); }
    cudaError_t e = cudaMalloc(&c->blob, total);
    if (e != cudaSuccess) { delete c; return e; }
    for (auto& p : parts)
        if (p.bytes && e == cudaSuccess) e = cudaMemcpy((char*)c->blob + p.off, p.src, p.bytes, cudaMemcpyHostToDevice);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    c->grid = HSG_CTAS * sms;                                 // persistent CTAs: one scratch area each
    if (e == cudaSuccess) e = cudaMalloc(&c->scratch, (size_t)c->grid * 64 * (size_t)t->nslot);
    if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
    char* b = (char*)c->blob;
    HsgDev& d = c->d;
    d.obj = (const int4*)(b + parts[0].off); d.term = (const int4*)(b + parts[1].off);
    d.p1_items = (const int*)(b + parts[2].off); d.legset_mask = (const int*)(b + parts[3].off);
    d.xitem = (const int2*)(b + parts[4].off); d.entry = (const int4*)(b + parts[5].off);
    d.flow = (const int4*)(b + parts[6].off); d.vtab = (const unsigned short*)(b + parts[7].off);
    d.dentry = (const int4*)(b + parts[8].off); d.ltab = (const unsigned*)(b + parts[9].off);
    d.flowL = (const unsigned*)(b + parts[10].off); d.flowT = (const unsigned*)(b + parts[11].off);
    d.lut = (const unsigned char*)(b + parts[12].off); d.nlut = (int)codes.size();
    d.npar = t->npar; d.ncolor = t->ncolor; d.nslot = t->nslot; d.nlegsets = t->nlegsets; d.nxitem = t->nxitem;
    d.nflow = t->nflow; d.nlevel = t->nlevel;
    for (int l = 0; l < 8; l++) d.p1_level[l] = l <= t->nlevel ? t->p1_level[l] : 0;
    // objects are sorted by their number of legs: the arguments' area ends where the first object of more than 3 legs starts
    d.nslot_arg = t->ns_obj;
    for (int i = 0; i < t->nobj; i++)
        if ((t->obj[4 * i + 1] & 0xFF) > 3 && t->obj[4 * i] < d.nslot_arg) d.nslot_arg = t->obj[4 * i];
    bool args_ok = true;
    for (int i = 0; i < t->nterm; i++) {
        const int op = t->term[4 * i] & 0xFF;
        if (op <= 2) continue;
        const int nargs = (op == 4 || op == 12 || op == 13) ? 3 : 2;
        for (int k = 1; k <= nargs; k++) args_ok = args_ok && (t->term[4 * i + k] & 0xFFFF) < d.nslot_arg;
    }
    for (int i = 0; i < t->nobj; i++)        // ... and an object of <= 3 legs lies below it entirely
        if ((t->obj[4 * i + 1] & 0xFF) <= 3) args_ok = args_ok && t->obj[4 * i] + (1 << (t->obj[4 * i + 1] & 0xFF)) <= d.nslot_arg;
    if (!args_ok) { cudaFree(c->blob); cudaFree(c->scratch); delete c; return cudaErrorInvalidValue; }
    int p3buf = 0;
    for (int i = 0; i < t->nentry; i++) {
        const int w = t->entry[4 * i + 3];
        const int lgx = ((w >> 4) & 7) + __builtin_popcount((w >> 1) & 7), lgy = t->npar - lgx;
        bool known = false;
#define HSG_P3_KNOWN(M, LG) known = known || (((w >> 1) & 7) == (M) && lgx == (LG));
        HSG_P3_COMBOS(HSG_P3_KNOWN)
#undef HSG_P3_KNOWN
        if (!known || lgx < 4 || lgx > 6) { cudaFree(c->blob); cudaFree(c->scratch); delete c; return cudaErrorInvalidValue; }
        const int b = 64 * ((1 << lgx) + (1 << lgy)) + 128;      // (+ 128: the tensor path's planes are 16 bytes longer)
        if (b > p3buf) p3buf = b;
        // tensor path: the record's mask must be one the kernel is instantiated for, its leg count the entry's
        const int w1 = t->dentry[4 * i + 1], m = (w1 >> 20) & 7;
        bool kmask = false;
#define HSG_P3T_KNOWN(M) kmask = kmask || m == (M);
        HSG_P3T_MASKS(HSG_P3T_KNOWN)
#undef HSG_P3T_KNOWN
        if (!kmask || ((w1 >> 16) & 0xF) != lgx) { cudaFree(c->blob); cudaFree(c->scratch); delete c; return cudaErrorInvalidValue; }
    }
    d.p3buf = p3buf;
    c->smem_alu = sizeof(double) * 4 * (size_t)(t->nlegsets + t->npar) + lut.size() + (size_t)(HSG_THREADS / 32) * HSG_P3_STAGES * p3buf;
    if (64 * (size_t)d.nslot_arg > (size_t)(HSG_THREADS / 32) * HSG_P3_STAGES * p3buf) { cudaFree(c->blob); cudaFree(c->scratch); delete c; return cudaErrorInvalidValue; }
    c->smem = c->smem_alu + (size_t)(HSG_THREADS / 32) * (16u << t->npar) + (sizeof(long long) << t->npar);
    e = cudaFuncSetAttribute(hsg_diagrams_kernel<double, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_alu);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hsg_diagrams_kernel<float, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem_alu);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hsg_diagrams_kernel<double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hsg_diagrams_kernel<float, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
    if (e != cudaSuccess) { cudaFree(c->blob); cudaFree(c->scratch); delete c; return e; }
    *out = c;
    return cudaSuccess;
}

void hsg_set_tensor(HsgContext* c, bool on) { c->tensor = on; }
bool hsg_get_tensor(const HsgContext* c) { return c->tensor; }

static cudaError_t launch_any(const HsgContext* c, bool jamps_fp64, const HsLaunch& a, int grid, char* scratch, cudaStream_t st)
{
    if (c->tensor) {
        if (jamps_fp64) hsg_diagrams_kernel<double, true><<<grid, HSG_THREADS, c->smem, st>>>(c->d, a, scratch);
        else hsg_diagrams_kernel<float, true><<<grid, HSG_THREADS, c->smem, st>>>(c->d, a, scratch);
    } else {
        if (jamps_fp64) hsg_diagrams_kernel<double, false><<<grid, HSG_THREADS, c->smem_alu, st>>>(c->d, a, scratch);
        else hsg_diagrams_kernel<float, false><<<grid, HSG_THREADS, c->smem_alu, st>>>(c->d, a, scratch);
    }
    return cudaGetLastError();
}

// once per context, with the context's device current: the device address of the static scratch array on THAT device
cudaError_t hsg_static_setup(HsgContext* c)
{
    void* ptr = nullptr;
    c->static_err = cudaGetSymbolAddress(&ptr, hsg_static_scratch);
    c->static_scratch = c->static_err == cudaSuccess ? (char*)ptr : nullptr;
    return c->static_err;
}

// persistent CTAs the static array has room for (0: the process's scratch area does not fit at all)
int hsg_static_ctas(const HsgContext* c)
{
    const size_t per_cta = 64 * (size_t)c->t->nslot;
    const size_t n = HSG_STATIC_BYTES / per_cta;
    return (int)(n < (size_t)HSG_STATIC_CTAS ? n : (size_t)HSG_STATIC_CTAS);
}

// the same kernel as hsg_launch with its scratch areas in the static array: allocates nothing, at most HSG_STATIC_CTAS CTAs
cudaError_t hsg_launch_static(const HsgContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st)
{
    if (a.nevt <= 0) return cudaSuccess;
    if (!c->static_scratch) return c->static_err != cudaSuccess ? c->static_err : cudaErrorNotReady;
    const int ctas = hsg_static_ctas(c);
    if (ctas < 1) return cudaErrorInvalidValue;
    const int grid = a.nevt < ctas ? a.nevt : ctas;
    return launch_any(c, jamps_fp64, a, grid, c->static_scratch, st);
}

void hsg_destroy(HsgContext* c)
{
    if (!c) return;
    cudaFree(c->blob);
    cudaFree(c->scratch);
    delete c;
}

cudaError_t hsg_launch(const HsgContext* c, bool jamps_fp64, const HsLaunch& a, cudaStream_t st)
{
    if (a.nevt <= 0) return cudaSuccess;
    const int grid = a.nevt < c->grid ? a.nevt : c->grid;
    return launch_any(c, jamps_fp64, a, grid, c->scratch, st);
}

}  // namespace mg
