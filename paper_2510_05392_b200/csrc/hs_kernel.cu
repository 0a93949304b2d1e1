// hs_kernel.cu -- helicity-shared diagram kernel: one CTA = one event, one thread =
// one helicity combination; interprets the tables of gen/co_program.py (layout: hs_tables.h).
//
// Why this shape on B200: the paper keeps one thread per (event, helicity) and lets
// every helicity recompute every wavefunction, with up to 121 wavefunctions + 120 jamps of per-thread state
// -- 12 KB per thread, i.e. local-memory traffic.  Here the state that depends on
// few helicities lives once per event in shared memory (<= 8 variants per object), the per-helicity work is a
// stream of 4-component complex dot products whose operands are broadcast reads of shared memory, and every
// jamp is finished in registers and written once, coalesced, to the jamps buffer [2][ncolor][rows]
// with rows ordered (event, helicity).
#include <stdint.h>

#include "helas.cuh"
#include "hs_kernel.cuh"

namespace mg {

struct HsDev {
    const int4* obj; const int4* term; const int* p1_items; const int* legset_mask; const int4* group;
    const int4* xobj; const int* x_items; const int4* sigma; const int4* entry; const unsigned short* vtab;
    int npar, ncolor, ngroups, obj_area, stage_area, nlegsets;
    int p1_level[4];
};

__device__ __forceinline__ int pext8(int v, int mask)
{
    int out = 0, j = 0;
#pragma unroll
    for (int b = 0; b < 5; b++) {
        if ((mask >> b) & 1) { out |= ((v >> b) & 1) << j; j++; }
    }
    return out;
}

__device__ __forceinline__ void load_obj(const double2* __restrict__ area, int off, int nv, int var, wf<double>& w)
{
    const double2* p = area + off + var;
#pragma unroll
    for (int c = 0; c < 4; c++) { const double2 v = p[c * nv]; w.c[c].re = v.x; w.c[c].im = v.y; }
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

// sum of the terms [t0, t0+nt) for helicity variant `var` of an object whose leg set has total momentum kout
__device__ __noinline__ void run_terms(const HsDev& d, const double2* __restrict__ area, const double* __restrict__ Ks,
                                       const double* __restrict__ pm, int t0, int nt, int var, int ls_out, double mt,
                                       double wt, wf<double>& acc)
{
#pragma unroll
    for (int c = 0; c < 4; c++) acc.c[c] = mk<double>(0.0, 0.0);
    for (int t = t0; t < t0 + nt; t++) {
        const int4 w = __ldg(d.term + t);
        const int op = w.x & 0xFF, neg = (w.x >> 8) & 1;
        const int a0 = w.y & 0xFFFF, a1 = (w.y >> 16) & 0xFFFF, a2 = w.z & 0xFFFF;
        wf<double> r;
        if (op <= 2) {
            const int hel = (var & 1) ? 1 : -1;
            const double* p = pm + 4 * a0;
            if (op == 0) ext_eps(p, hel, a0 >= 2, r);
            else if (op == 1) ext_ubar(p, mt, hel, r);
            else ext_v(p, mt, hel, r);
        } else {
            const int4 oa = __ldg(d.obj + a0), ob = __ldg(d.obj + a1);
            wf<double> A, B;
            load_obj(area, oa.x, 1 << (oa.y & 0xFF), pext8(var, (w.x >> 16) & 0xFF), A);
            load_obj(area, ob.x, 1 << (ob.y & 0xFF), pext8(var, (w.x >> 24) & 0xFF), B);
            switch (op) {
                case 3: v3_off(A, load_k(Ks, oa.y >> 8), B, load_k(Ks, ob.y >> 8), 1.0 / m2(load_k(Ks, ls_out)), r); break;
                case 11: v3_off(A, load_k(Ks, oa.y >> 8), B, load_k(Ks, ob.y >> 8), 1.0, r); lower(r); break;
                case 4: case 12: {
                    const int4 oc = __ldg(d.obj + a2);
                    wf<double> Z;
                    load_obj(area, oc.x, 1 << (oc.y & 0xFF), pext8(var, (w.z >> 16) & 0xFF), Z);
                    v4_off(A, B, Z, op == 4 ? 1.0 / m2(load_k(Ks, ls_out)) : 1.0, r);
                    if (op == 12) lower(r);
                    break;
                }
                case 5: { const p4<double> K = load_k(Ks, ls_out); ffv_l(A, B, -K, mt, inv_prop(m2(K), mt, wt), r); break; }
                case 6: { const p4<double> K = load_k(Ks, ls_out); ffv_r(A, B, K, mt, inv_prop(m2(K), mt, wt), r); break; }
                case 7: ffv_p(A, B, 1.0 / m2(load_k(Ks, ls_out)), r); break;
                case 8: row_slash(A, make_slashed(B), r); break;
                case 9: slash_col(make_slashed(A), B, r); break;
                default: ffv_p(A, B, 1.0, r); lower(r); break;       // 10: x_bil
            }
        }
        if (neg) { for (int c = 0; c < 4; c++) acc.c[c] -= r.c[c]; }
        else { for (int c = 0; c < 4; c++) acc.c[c] += r.c[c]; }
    }
}

// T2 = type of the jamps buffer (double: MG_FP64, float: MG_MIXED -- PAPER.md:122 "FPTYPE=m")
// blockDim.x = 2^npar * nsplit: thread = (sigma split s, helicity combination h)
template <typename T2>
__global__ void __launch_bounds__(256) hs_diagrams_kernel(const HsDev d, const HsLaunch a)
{
    extern __shared__ double2 sm[];
    double2* __restrict__ area = sm;
    double2* __restrict__ stage = sm + d.obj_area;
    double* __restrict__ Ks = reinterpret_cast<double*>(stage + d.stage_area);
    double* __restrict__ pm = Ks + 4 * d.nlegsets;
    const int tid = threadIdx.x, nth = blockDim.x;
    const int nh = 1 << d.npar;
    const int h = tid & (nh - 1), split = tid >> d.npar, nsplit = nth >> d.npar;
    const int pos = a.d_pos[h];                       // row of this helicity inside the event, -1 = not a good helicity
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
        // phase 1: objects, level by level
        for (int lvl = 0; lvl < 3; lvl++) {
            for (int i = d.p1_level[lvl] + tid; i < d.p1_level[lvl + 1]; i += nth) {
                const int it = __ldg(d.p1_items + i);
                const int4 o = __ldg(d.obj + (it >> 8));
                const int var = it & 0xFF, nv = 1 << (o.y & 0xFF);
                wf<double> acc;
                run_terms(d, area, Ks, pm, o.z, o.w, var, o.y >> 8, a.mt, a.wt, acc);
                double2* out = area + o.x + var;
#pragma unroll
                for (int c = 0; c < 4; c++) out[c * nv] = make_double2(acc.c[c].re, acc.c[c].im);
            }
            __syncthreads();
        }
        const size_t row = (size_t)e * a.nrow_evt + pos;
        for (int g = 0; g < d.ngroups; g++) {
            const int4 g0 = __ldg(d.group + 2 * g), g1 = __ldg(d.group + 2 * g + 1);
            // phase 2: pair objects of this group
            for (int i = tid; i < g0.z; i += nth) {
                const int it = __ldg(d.x_items + g0.y + i);
                const int4 x = __ldg(d.xobj + g0.x + (it >> 8));
                const int var = it & 0xFF, nv = 1 << x.y;
                wf<double> acc;
                run_terms(d, area, Ks, pm, x.z, x.w, var, 0, a.mt, a.wt, acc);
                double2* out = stage + x.x + var;
#pragma unroll
                for (int c = 0; c < 4; c++) out[c * nv] = make_double2(acc.c[c].re, acc.c[c].im);
            }
            __syncthreads();
            // phase 3: the jamps of this group, one colour flow at a time
            if (pos >= 0) {
                for (int s = split; s < g1.x; s += nsplit) {
                    const int4 sg = __ldg(d.sigma + g0.w + s);
                    double re = 0.0, im = 0.0;
#pragma unroll 2
                    for (int k = 0; k < sg.z; k++) {
                        const int4 en = __ldg(d.entry + sg.y + k);
                        const int vv = __ldg(d.vtab + en.z * nh + h);
                        const int nvx = en.x >> 16, nvy = en.y >> 16;
                        const double2* __restrict__ X = stage + (en.x & 0xFFFF) + (vv & 0xFF);
                        const double2* __restrict__ Y = area + (en.y & 0xFFFF) + (vv >> 8);
                        double tr = 0.0, ti = 0.0;
#pragma unroll
                        for (int c = 0; c < 4; c++) {
                            const double2 x = X[c * nvx], y = Y[c * nvy];
                            tr = fma(x.x, y.x, tr); tr = fma(-x.y, y.y, tr);
                            ti = fma(x.x, y.y, ti); ti = fma(x.y, y.x, ti);
                        }
                        const double sgn = (double)en.w;
                        re = fma(sgn, tr, re); im = fma(sgn, ti, im);
                    }
                    T2* __restrict__ out = reinterpret_cast<T2*>(a.d_jamps);
                    out[(size_t)sg.x * a.rows + row] = T2(re);
                    out[(size_t)(d.ncolor + sg.x) * a.rows + row] = T2(im);
                }
            }
            __syncthreads();
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
struct HsContext {
    const HsTables* t = nullptr;
    HsDev d;
    void* blob = nullptr;
    size_t smem = 0;
    int sms = 148;
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
    Part parts[10] = { { t->obj, sizeof(int) * 4 * t->nobj, 0 }, { t->term, sizeof(int) * 4 * t->nterm, 0 },
                       { t->p1_items, sizeof(int) * t->np1, 0 }, { t->legset_mask, sizeof(int) * t->nlegsets, 0 },
                       { t->group, sizeof(int) * 8 * t->ngroups, 0 }, { t->xobj, sizeof(int) * 4 * t->nxobj, 0 },
                       { t->x_items, sizeof(int) * t->nxitems, 0 }, { t->sigma, sizeof(int) * 4 * t->nsigma, 0 },
                       { t->entry, sizeof(int) * 4 * t->nentry, 0 }, { t->vtab, sizeof(unsigned short) * nh * t->nvrow, 0 } };
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
    d.npar = t->npar; d.ncolor = t->ncolor; d.ngroups = t->ngroups; d.obj_area = t->obj_area; d.stage_area = t->stage_area;
    d.nlegsets = t->nlegsets;
    for (int i = 0; i < 4; i++) d.p1_level[i] = t->p1_level[i];
    c->smem = sizeof(double2) * ((size_t)t->obj_area + t->stage_area) + sizeof(double) * 4 * (t->nlegsets + t->npar);
    e = cudaFuncSetAttribute(hs_diagrams_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(hs_diagrams_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem);
    if (e != cudaSuccess) { cudaFree(c->blob); delete c; return e; }
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
    *out = c;
    return cudaSuccess;
}

void hs_destroy(HsContext* c)
{
    if (!c) return;
    cudaFree(c->blob);
    delete c;
}

cudaError_t hs_launch(const HsContext* c, bool jamps_fp64, const HsLaunch& a, int nsplit, cudaStream_t st)
{
    if (a.nevt <= 0) return cudaSuccess;
    const int threads = (1 << c->t->npar) * nsplit;
    if (nsplit < 1 || threads > 256) return cudaErrorInvalidValue;
    const int grid = a.nevt;                         // one CTA per event; the hardware scheduler keeps every SM full
    if (jamps_fp64) hs_diagrams_kernel<double><<<grid, threads, c->smem, st>>>(c->d, a);
    else hs_diagrams_kernel<float><<<grid, threads, c->smem, st>>>(c->d, a);
    return cudaGetLastError();
}

}  // namespace mg
