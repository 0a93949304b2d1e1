// api.cu -- the C ABI of include/mg5_b200.h: handle, parameters, helicity filter, batch scheduling.
//
// Host-side flow of one batch:
//   [first call] helicity filter on a probe batch, every helicity combination in ONE launch
//   diagram kernel(s): helicity as grid.y (MG_SCHED_GRID) or one launch per helicity on a library stream
//   colour sum: fused in the diagram kernel (MG_CS_FUSED) or ONE tensor-core contraction over the
//               nGoodHel*nevt rows of the jamps buffer (MG_CS_TENSOR; csrc/color_sum.cu)
//   helicity sum kernel: me[e] = sum_h me_h[h][e]  (fixed order: deterministic)
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <string>
#include <vector>

#include "../../include/mg5_b200.h"
#include "color_sum.cuh"
#include "hs_kernel.cuh"
#include "hsg_kernel.cuh"
#include "mg_internal.cuh"

using namespace mg;

static thread_local std::string g_init_error;

struct mg_process {
    const ProcessDesc* d = nullptr;
    int precision = MG_FP64;
    int device = 0;
    // parameters (BASELINE.json card)
    double aEWM1 = 132.507, mZ = 91.188, wZ = 2.4414, mW = 80.419, mT = 173.0, wT = 1.4915, aS = 0.118;
    // options
    int color_sum = MG_CS_FUSED, schedule = MG_SCHED_GRID, block = 64, timing = 0;       // (block: 64 measured best for g g -> t tbar (g))
    int diagrams = MG_DIAG_THREAD, hs_color_alu = 0, tf32_direct = 1;
    int max_streams = 0;       // MG_SCHED_STREAMS: helicity h runs on stream h % max_streams (0 = one stream per helicity)
    int graph = 0;             // replay the launch sequence of a batch as a CUDA graph
    // the captured batch: valid for exactly these arguments and this state of the handle (epoch)
    struct GraphKey {
        const double* mom = nullptr; double* me = nullptr; void* ws = nullptr; int nevt = 0; cudaStream_t st = nullptr;
        const void* ex[5] = { nullptr, nullptr, nullptr, nullptr, nullptr };
        long epoch = -1;
        bool operator==(const GraphKey& o) const
        {
            return mom == o.mom && me == o.me && ws == o.ws && nevt == o.nevt && st == o.st && epoch == o.epoch &&
                   !memcmp(ex, o.ex, sizeof ex);
        }
    } gkey;
    cudaGraphExec_t gexec = nullptr;
    cudaStream_t gstream = nullptr;          // capture / replay stream when the caller passes the legacy default stream
    cudaEvent_t gev_in = nullptr, gev_out = nullptr;
    long epoch = 0;            // bumped by every call that changes what a batch launches
    int graph_replays = 0;
    HsContext* hs = nullptr;   // helicity-shared program (gg processes)
    HsgContext* hsg = nullptr; // generic helicity-shared kernel (g g -> t tbar g g g g: the only diagram kernel it has)
    int* d_pos = nullptr;      // DEVICE [ncomb]: position of helicity h in the good list, -1 = not good
    long jamp_chunk_bytes = 16L << 30;     // one chunk for every BASELINE.json batch (180 GB of HBM3e); smaller via "jamp_chunk_mib"
    // good helicities
    std::vector<int> good;
    int* d_good = nullptr;     // DEVICE [ncomb]
    int* d_all = nullptr;      // DEVICE [ncomb] = 0..ncomb-1
    void* d_cmat = nullptr;    // DEVICE [ncolor^2] numerators as the colour-sum type
    void* d_cmat64 = nullptr;  // DEVICE [ncolor^2] numerators in fp64 (helicity filter; = d_cmat in MG_FP64)
    void* d_chol64 = nullptr;  // DEVICE fp64 factor for the helicity filter of the generic kernel when d_chol is the TF32 image (else = d_chol)
    void* d_chol = nullptr;    // DEVICE Cholesky factor of the numerators for the tensor colour sum: fp64 [ncp^2] (MG_FP64) or its TF32 image
    // helicity streams
    std::vector<cudaStream_t> streams;
    cudaEvent_t ev_fork = nullptr;
    std::vector<cudaEvent_t> ev_join;
    // host-buffer path
    double* d_mom_own = nullptr; double* d_me_own = nullptr; void* d_ws_own = nullptr;
    int own_nevt = 0; size_t own_ws = 0;
    // timing
    std::vector<cudaEvent_t> ev_pool;     // timing marks of the last batch: mark k closes stage ev_stage[k]
    std::vector<int> ev_stage;
    int ev_n = 0;
    bool timed = false;
    int launches = 0;          // kernels launched by the last mg_sigma_batch
    std::string err;
};

static int fail(mg_process* p, int code, const std::string& msg)
{
    if (p) p->err = msg; else g_init_error = msg;
    return code;
}
#define CUDA_TRY(p, call)                                                                        \
    do {                                                                                         \
        cudaError_t e_ = (call);                                                                 \
        if (e_ != cudaSuccess)                                                                   \
            return fail(p, e_ == cudaErrorMemoryAllocation ? MG_ENOMEM : MG_ECUDA,               \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                     \
    } while (0)

static size_t cs_elem(const mg_process* p) { return p->precision == MG_FP64 ? 8 : 4; }
static size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

static phys<double> make_phys(const mg_process* p)
{
    phys<double> ph;
    ph.mt = p->mT; ph.wt = p->wT; ph.mz = p->mZ; ph.wz = p->wZ;
    const double ee = sqrt(4.0 * M_PI / p->aEWM1);
    const double sw2 = 1.0 - p->mW * p->mW / (p->mZ * p->mZ);
    const double sw = sqrt(sw2), cw = sqrt(1.0 - sw2);
    ph.ee = ee; ph.gl = ee * (-0.5 + sw2) / (sw * cw); ph.gr = ee * sw / cw;
    return ph;
}

static double make_norm(const mg_process* p)
{
    const double g2 = 4.0 * M_PI * p->aS;
    return pow(g2, p->d->coupling_order) / (p->d->denom * p->d->cden);
}

// g g -> t tbar g g g g (Table 2): no thread-per-(event, helicity) kernel (launch =
// NULL), the generic helicity-shared kernel only.  The colour matrix is expanded from its first row:
// C[s][s'] = row0[rank(s^-1 o s')], permutations in lexicographic order (gen/colour.py colour_matrix).
static const ProcessDesc* desc_gg_ttxgggg()
{
    static ProcessDesc d;
    static std::vector<int> cmat;
    static bool done = false;
    if (done) return &d;
    const HsgTables* t = hsg_tables(6);
    if (!t) return nullptr;
    const int n = 6, np = t->ncolor;
    std::vector<std::vector<int>> perms;
    std::vector<int> a(n);
    for (int i = 0; i < n; i++) a[i] = i;
    do perms.push_back(a); while (std::next_permutation(a.begin(), a.end()));
    auto rank = [&](const std::vector<int>& q) {            // lexicographic rank
        int r = 0;
        for (int i = 0; i < n; i++) {
            int smaller = 0;
            for (int j = i + 1; j < n; j++) smaller += q[j] < q[i];
            int f = 1;
            for (int k = 2; k <= n - 1 - i; k++) f *= k;
            r += smaller * f;
        }
        return r;
    };
    cmat.assign((size_t)np * np, 0);
    for (int i = 0; i < np; i++) {
        int inv[6];
        for (int pos = 0; pos < n; pos++) inv[perms[i][pos]] = pos;
        for (int j = 0; j < np; j++) {
            std::vector<int> rel(n);
            for (int pos = 0; pos < n; pos++) rel[pos] = inv[perms[j][pos]];
            cmat[(size_t)i * np + j] = t->cmat_row0[rank(rel)];
        }
    }
    d.name = "gg_ttxgggg"; d.ngluon = 6; d.npar = 8; d.ncomb = 256; d.ncolor = np; d.ndiagrams = t->ndiagrams;
    d.namps = 0; d.ncurrents = t->nobj; d.ngroups = 1;
    d.denom = 256.0 * 24.0;            // 2*2 spins, 8*8 colours of the beams, 4! identical final gluons (reading A3)
    d.cden = t->cden; d.cmat = cmat.data();
    d.flops = (t->flops_p1 + t->flops_p2) / 256.0 + t->flops_p3;
    d.coupling_order = 6; d.has_fp32 = false; d.launch = nullptr;
    done = true;
    return &d;
}

extern "C" const char* mg_last_error(const mg_process* p) { return p ? p->err.c_str() : g_init_error.c_str(); }

static int upload_tables(mg_process* p)
{
    const ProcessDesc* d = p->d;
    const int n2 = d->ncolor * d->ncolor;
    if (p->d_cmat) { cudaFree(p->d_cmat); p->d_cmat = nullptr; }
    CUDA_TRY(p, cudaMalloc(&p->d_cmat, (size_t)n2 * cs_elem(p)));
    if (p->precision == MG_FP64) {
        std::vector<double> h(n2);
        for (int i = 0; i < n2; i++) h[i] = d->cmat[i];
        CUDA_TRY(p, cudaMemcpy(p->d_cmat, h.data(), n2 * sizeof(double), cudaMemcpyHostToDevice));
    } else {
        std::vector<float> h(n2);
        for (int i = 0; i < n2; i++) h[i] = (float)d->cmat[i];
        CUDA_TRY(p, cudaMemcpy(p->d_cmat, h.data(), n2 * sizeof(float), cudaMemcpyHostToDevice));
        std::vector<double> h64(n2);
        for (int i = 0; i < n2; i++) h64[i] = d->cmat[i];
        CUDA_TRY(p, cudaMalloc(&p->d_cmat64, (size_t)n2 * sizeof(double)));
        CUDA_TRY(p, cudaMemcpy(p->d_cmat64, h64.data(), n2 * sizeof(double), cudaMemcpyHostToDevice));
    }
    if (p->precision == MG_FP64) p->d_cmat64 = p->d_cmat;
    if (d->ncolor > 128) {
        // 720 colours: fp64 factor in fragment order (the helicity filter always decides in fp64, reading A5) and, in mixed
        // precision, its TF32 image for the tcgen05 contraction
        std::vector<double> frag; int rank = 0;
        if (!color_cholesky_big(d->ncolor, d->cmat, frag, &rank)) return fail(p, MG_ESTATE, "colour matrix is not positive semi-definite");
        CUDA_TRY(p, cudaMalloc(&p->d_chol64, frag.size() * sizeof(double)));
        CUDA_TRY(p, cudaMemcpy(p->d_chol64, frag.data(), frag.size() * sizeof(double), cudaMemcpyHostToDevice));
        if (p->precision == MG_FP64) p->d_chol = p->d_chol64;
        else {
            std::vector<float> img;
            if (!tf32_big_build_factor_image(d->ncolor, d->cmat, img)) return fail(p, MG_ESTATE, "cannot build the TF32 factor image");
            CUDA_TRY(p, cudaMalloc(&p->d_chol, img.size() * sizeof(float)));
            CUDA_TRY(p, cudaMemcpy(p->d_chol, img.data(), img.size() * sizeof(float), cudaMemcpyHostToDevice));
        }
    } else if (p->precision == MG_FP64) {
        std::vector<double> lp; int ncp = 0;
        if (!color_cholesky_padded(d->ncolor, d->cmat, lp, &ncp)) return fail(p, MG_ESTATE, "colour matrix is not positive definite");
        std::vector<double> frag;
        color_cholesky_fragments(ncp, lp, frag);               // row-major factor, then its fragment-order copy
        lp.insert(lp.end(), frag.begin(), frag.end());
        CUDA_TRY(p, cudaMalloc(&p->d_chol, lp.size() * sizeof(double)));
        CUDA_TRY(p, cudaMemcpy(p->d_chol, lp.data(), lp.size() * sizeof(double), cudaMemcpyHostToDevice));
    } else {
        std::vector<float> img;
        if (!tf32_build_factor_image(d->ncolor, d->cmat, img)) return fail(p, MG_ESTATE, "colour matrix is not positive definite");
        CUDA_TRY(p, cudaMalloc(&p->d_chol, img.size() * sizeof(float)));
        CUDA_TRY(p, cudaMemcpy(p->d_chol, img.data(), img.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    std::vector<int> all(d->ncomb);
    for (int i = 0; i < d->ncomb; i++) all[i] = i;
    CUDA_TRY(p, cudaMalloc(&p->d_all, d->ncomb * sizeof(int)));
    CUDA_TRY(p, cudaMalloc(&p->d_good, d->ncomb * sizeof(int)));
    CUDA_TRY(p, cudaMalloc(&p->d_pos, d->ncomb * sizeof(int)));
    CUDA_TRY(p, cudaMemcpy(p->d_all, all.data(), d->ncomb * sizeof(int), cudaMemcpyHostToDevice));
    return MG_OK;
}

extern "C" int mg_init_process(const char* name, int precision, int device, mg_process** out)
{
    if (!out) return fail(nullptr, MG_EINVAL, "out is NULL");
    *out = nullptr;
    if (!name) return fail(nullptr, MG_EINVAL, "name is NULL");
    if (precision < MG_FP64 || precision > MG_FP32) return fail(nullptr, MG_EINVAL, "bad precision");
    const ProcessDesc* d = nullptr;
    if (!strcmp(name, "epem_mupmum")) d = desc_epem_mupmum();
    else if (!strcmp(name, "gg_ttx")) d = desc_gg_ttx();
    else if (!strcmp(name, "gg_ttxg")) d = desc_gg_ttxg();
    else if (!strcmp(name, "gg_ttxgg")) d = desc_gg_ttxgg();
    else if (!strcmp(name, "gg_ttxggg")) d = desc_gg_ttxggg();
    else if (!strcmp(name, "gg_ttxgggg")) d = desc_gg_ttxgggg();
    else return fail(nullptr, MG_EINVAL, std::string("unknown process ") + name);
    if (!d) return fail(nullptr, MG_EINVAL, std::string("library built without ") + name);
    if (!d->launch && precision == MG_FP32)
        return fail(nullptr, MG_EINVAL, std::string(name) + " runs in MG_FP64 and MG_MIXED only (generic helicity-shared kernel, fp64 amplitudes)");
    if (precision == MG_FP32 && !d->has_fp32)
        return fail(nullptr, MG_EINVAL, std::string("library built without the MG_FP32 instantiation of ") + name);
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev)
        return fail(nullptr, MG_ENODEV, "no such CUDA device");
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return fail(nullptr, MG_ENODEV, "cannot query device");
    if (prop.major != 10) {
        char buf[128];
        snprintf(buf, sizeof buf, "device is sm_%d%d; this library is sm_100a only (no fallback)", prop.major, prop.minor);
        return fail(nullptr, MG_ENODEV, buf);
    }
    if (cudaSetDevice(device) != cudaSuccess) return fail(nullptr, MG_ECUDA, "cudaSetDevice failed");
    mg_process* p = new mg_process;
    p->d = d; p->precision = precision; p->device = device;
    int rc = upload_tables(p);
    if (rc != MG_OK) { g_init_error = p->err; mg_destroy(p); return rc; }
    if (!d->launch) {                                         // the generic helicity-shared kernel is the only diagram kernel
        cudaError_t e = hsg_create(d->ngluon, &p->hsg);
        if (e != cudaSuccess) { g_init_error = std::string("hsg_create: ") + cudaGetErrorString(e); mg_destroy(p); return e == cudaErrorMemoryAllocation ? MG_ENOMEM : MG_ECUDA; }
        p->diagrams = MG_DIAG_SHARED;
        hsg_static_setup(p->hsg);          // mg_sigma_batch_noalloc (a failure is reported by that call, not here)
    } else if (hs_tables(d->ngluon) && precision != MG_FP32) {       // helicity-shared program: g g -> t tbar + >= 2 g
        cudaError_t e = hs_create(d->ngluon, &p->hs);
        if (e != cudaSuccess) { g_init_error = std::string("hs_create: ") + cudaGetErrorString(e); mg_destroy(p); return MG_ECUDA; }
        p->diagrams = MG_DIAG_SHARED;                         // measured default, see DESIGN.md
        if (d->ncolor < 120) p->hs_color_alu = 1;             // 24 x 24: the fp32 ALU kernel beats the 128-row tcgen05 tiles (measured)
    }
    *out = p;
    return MG_OK;
}

extern "C" void mg_destroy(mg_process* p)
{
    if (!p) return;
    cudaSetDevice(p->device);
    hs_destroy(p->hs);
    hsg_destroy(p->hsg);
    cudaFree(p->d_pos);
    if (p->d_cmat64 != p->d_cmat) cudaFree(p->d_cmat64);
    if (p->d_chol64 != p->d_chol) cudaFree(p->d_chol64);
    cudaFree(p->d_good); cudaFree(p->d_all); cudaFree(p->d_cmat); cudaFree(p->d_chol);
    cudaFree(p->d_mom_own); cudaFree(p->d_me_own); cudaFree(p->d_ws_own);
    for (auto s : p->streams) cudaStreamDestroy(s);
    for (auto e : p->ev_join) cudaEventDestroy(e);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    for (auto e : p->ev_pool) cudaEventDestroy(e);
    if (p->gexec) cudaGraphExecDestroy(p->gexec);
    if (p->gstream) cudaStreamDestroy(p->gstream);
    if (p->gev_in) cudaEventDestroy(p->gev_in);
    if (p->gev_out) cudaEventDestroy(p->gev_out);
    delete p;
}

extern "C" int mg_process_info(const mg_process* p, int* npar, int* ncomb, int* ncolor, int* ndiagrams, int* ngroups)
{
    if (!p) return MG_EINVAL;
    if (npar) *npar = p->d->npar;
    if (ncomb) *ncomb = p->d->ncomb;
    if (ncolor) *ncolor = p->d->ncolor;
    if (ndiagrams) *ndiagrams = p->d->ndiagrams;
    if (ngroups) *ngroups = p->d->ngroups;
    return MG_OK;
}

extern "C" int mg_process_flops(const mg_process* p, double* diagram_flops, double* color_flops)
{
    if (!p) return MG_EINVAL;
    if (diagram_flops) {
        *diagram_flops = p->d->flops;
        if (p->hsg) {
            const HsgTables* t = hsg_host_tables(p->hsg);
            *diagram_flops = (t->flops_p1 + t->flops_p2) / p->d->ncomb + t->flops_p3;
        } else if (p->diagrams == MG_DIAG_SHARED && p->hs) {
            const HsTables* t = hs_host_tables(p->hs);
            *diagram_flops = (t->flops_p1 + t->flops_p2) / p->d->ncomb + t->flops_p3;
        }
    }
    if (color_flops) *color_flops = 4.0 * p->d->ncolor * p->d->ncolor + 4.0 * p->d->ncolor;
    return MG_OK;
}

extern "C" int mg_set_parameters(mg_process* p, const char* const* keys, const double* values, int n)
{
    if (!p || (n > 0 && (!keys || !values))) return fail(p, MG_EINVAL, "bad arguments");
    mg_process tmp;      // validate everything before changing anything
    tmp.aEWM1 = p->aEWM1; tmp.mZ = p->mZ; tmp.wZ = p->wZ; tmp.mW = p->mW; tmp.mT = p->mT; tmp.wT = p->wT; tmp.aS = p->aS;
    for (int i = 0; i < n; i++) {
        const char* k = keys[i];
        if (!k) return fail(p, MG_EINVAL, "NULL key");
        if (!strcmp(k, "aEWM1")) tmp.aEWM1 = values[i];
        else if (!strcmp(k, "mZ")) tmp.mZ = values[i];
        else if (!strcmp(k, "wZ")) tmp.wZ = values[i];
        else if (!strcmp(k, "mW")) tmp.mW = values[i];
        else if (!strcmp(k, "mT")) tmp.mT = values[i];
        else if (!strcmp(k, "wT")) tmp.wT = values[i];
        else if (!strcmp(k, "aS")) tmp.aS = values[i];
        else return fail(p, MG_EINVAL, std::string("unknown parameter ") + k);
    }
    if (!(tmp.aEWM1 > 0) || !(tmp.mZ > 0) || !(tmp.mW > 0) || !(tmp.mW < tmp.mZ) || !(tmp.mT >= 0) || !(tmp.aS > 0) ||
        !(tmp.wZ >= 0) || !(tmp.wT >= 0))
        return fail(p, MG_EINVAL, "parameter out of range");
    p->epoch++;
    p->aEWM1 = tmp.aEWM1; p->mZ = tmp.mZ; p->wZ = tmp.wZ; p->mW = tmp.mW; p->mT = tmp.mT; p->wT = tmp.wT; p->aS = tmp.aS;
    return MG_OK;
}

extern "C" int mg_set_option(mg_process* p, const char* key, int value)
{
    if (!p || !key) return MG_EINVAL;
    if (!strcmp(key, "color_sum")) {
        if (value != MG_CS_FUSED && value != MG_CS_TENSOR) return fail(p, MG_EINVAL, "bad color_sum");
        p->color_sum = value;
    } else if (!strcmp(key, "schedule")) {
        if (value != MG_SCHED_GRID && value != MG_SCHED_STREAMS) return fail(p, MG_EINVAL, "bad schedule");
        if (value == MG_SCHED_STREAMS && p->diagrams == MG_DIAG_SHARED)
            return fail(p, MG_EINVAL, "helicity streams apply to the MG_DIAG_THREAD kernel only (set diagrams = 0 first)");
        p->schedule = value;
    } else if (!strcmp(key, "block")) {
        if (value < 32 || value > 256 || value % 32) return fail(p, MG_EINVAL, "bad block");
        p->block = value;
    } else if (!strcmp(key, "diagrams")) {
        if (value != MG_DIAG_THREAD && value != MG_DIAG_SHARED) return fail(p, MG_EINVAL, "bad diagrams");
        if (value == MG_DIAG_THREAD && !p->d->launch) return fail(p, MG_EINVAL, "this process has the helicity-shared kernel only");
        if (value == MG_DIAG_SHARED && !p->hs && !p->hsg) return fail(p, MG_EINVAL, "this process/precision has no helicity-shared program");
        if (value == MG_DIAG_SHARED && p->schedule == MG_SCHED_STREAMS)
            return fail(p, MG_EINVAL, "the helicity-shared kernel has no helicity streams (set schedule = 0 first)");
        p->diagrams = value;
    } else if (!strcmp(key, "hs_color_alu")) {
        p->hs_color_alu = value != 0;
    } else if (!strcmp(key, "tf32_direct")) {
        p->tf32_direct = value != 0;
    } else if (!strcmp(key, "timing")) {
        p->timing = value != 0;
    } else if (!strcmp(key, "jamp_chunk_mib")) {
        if (value < 1) return fail(p, MG_EINVAL, "bad jamp_chunk_mib");
        p->jamp_chunk_bytes = (long)value << 20;
    } else if (!strcmp(key, "max_streams")) {
        if (value < 0 || value > 1024) return fail(p, MG_EINVAL, "bad max_streams");
        p->max_streams = value;
    } else if (!strcmp(key, "graph")) {
        p->graph = value != 0;
    } else if (!strcmp(key, "p3_tensor")) {
        if (!p->hsg) return fail(p, MG_EINVAL, "p3_tensor applies to the generic helicity-shared kernel only (gg_ttxgggg)");
        hsg_set_tensor(p->hsg, value != 0);
    } else return fail(p, MG_EINVAL, std::string("unknown option ") + key);
    p->epoch++;
    return MG_OK;
}

extern "C" int mg_get_option(const mg_process* p, const char* key, int* value)
{
    if (!p || !key || !value) return MG_EINVAL;
    if (!strcmp(key, "color_sum")) *value = p->color_sum;
    else if (!strcmp(key, "schedule")) *value = p->schedule;
    else if (!strcmp(key, "block")) *value = p->block;
    else if (!strcmp(key, "diagrams")) *value = p->diagrams;
    else if (!strcmp(key, "hs_color_alu")) *value = p->hs_color_alu;
    else if (!strcmp(key, "tf32_direct")) *value = p->tf32_direct;
    else if (!strcmp(key, "timing")) *value = p->timing;
    else if (!strcmp(key, "jamp_chunk_mib")) *value = (int)(p->jamp_chunk_bytes >> 20);
    else if (!strcmp(key, "max_streams")) *value = p->max_streams;
    else if (!strcmp(key, "graph")) *value = p->graph;
    else if (!strcmp(key, "graph_replays")) *value = p->graph_replays;
    else if (!strcmp(key, "p3_tensor")) *value = p->hsg ? (int)hsg_get_tensor(p->hsg) : 0;
    else if (!strcmp(key, "probe_events")) *value = p->d->launch ? 1024 : 16;      // events the automatic helicity filter uses at most
    else return MG_EINVAL;
    return MG_OK;
}

// events per jamps chunk in MG_CS_TENSOR mode
static int chunk_events(const mg_process* p, int nevt, int nhel)
{
    const size_t per_evt = (size_t)nhel * p->d->ncolor * 2 * cs_elem(p);
    long ce = (long)(p->jamp_chunk_bytes / per_evt);
    ce = (ce / 128) * 128;
    if (ce < 128) ce = 128;
    if (ce > nevt) ce = nevt;
    return (int)ce;
}

// optional inputs / outputs of mg_sigma_batch_ex (all DEVICE, any may be NULL)
struct Extras {
    const double* alphas = nullptr; const double* rndhel = nullptr; const double* rndcol = nullptr;
    int* selhel = nullptr; int* selcol = nullptr;
};

static size_t ws_bytes_for(const mg_process* p, int nevt, int nhel, bool need_jamps = false)
{
    size_t b = align256((size_t)nhel * nevt * sizeof(double)) + align256((size_t)nevt * sizeof(double));   // me_h, coupling factors
    if ((p->color_sum == MG_CS_TENSOR || p->diagrams == MG_DIAG_SHARED || need_jamps) && nevt > 0) {
        const int ce = chunk_events(p, nevt, nhel);
        b += align256(color_sum_padded_rows((long)nhel * ce) * p->d->ncolor * 2 * cs_elem(p));
    }
    return b;
}

// events of the first batch the helicity filter looks at (the generic kernel's probe goes through the jamps buffer:
// 2.9 MB per event at 6 gluons)
static int probe_events(const mg_process* p, int nevt)
{
    const int cap = p->d->launch ? 1024 : 16;
    return nevt < cap ? nevt : cap;
}

static size_t filter_bytes(const mg_process* p, int nprobe)
{
    size_t b = align256((size_t)p->d->ncomb * nprobe * sizeof(double));                           // filter uses FUSED
    if (!p->d->launch) b += align256(color_sum_padded_rows((long)p->d->ncomb * nprobe) * p->d->ncolor * 2 * sizeof(double));
    return b;
}

static size_t workspace_bytes(const mg_process* p, int nevt, bool need_jamps)
{
    if (!p || nevt < 0) return 0;
    size_t a = ws_bytes_for(p, nevt, p->good.empty() ? p->d->ncomb : (int)p->good.size(), need_jamps);
    size_t b = p->good.empty() ? filter_bytes(p, probe_events(p, nevt)) : 0;
    return a > b ? a : b;
}

extern "C" size_t mg_workspace_bytes(const mg_process* p, int nevt) { return workspace_bytes(p, nevt, false); }
extern "C" size_t mg_workspace_bytes_ex(const mg_process* p, int nevt, int want_selcol)
{
    return workspace_bytes(p, nevt, want_selcol != 0 && p && p->d->ncolor > 1);
}

__global__ void helicity_sum_kernel(const double* __restrict__ meh, int nhel, int nevt, double* __restrict__ me)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nevt) return;
    double s = 0.0;
    for (int h = 0; h < nhel; h++) s += meh[(size_t)h * nevt + e];
    me[e] = s;
}

// alpha_s-dependent couplings, one thread per event ("an event-by-event running QCD coupling constant
// alpha_s(Q^2)"; the dependent couplings are computed in a kernel of their own): G = sqrt(4 pi alpha_s(e));
// every diagram of these processes carries G^order, so the squared amplitude scales by (G(e)^2 / G_card^2)^order
__global__ void couplings_kernel(const double* __restrict__ alphas, int nevt, int order, double g2_card, double* __restrict__ gfac)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nevt) return;
    const double g2 = 4.0 * 3.14159265358979323846 * alphas[e];
    double f = 1.0;
    for (int k = 0; k < order; k++) f *= g2 / g2_card;
    gfac[e] = f;
}

// helicity sum with the per-event coupling factor and the helicity selection ("Randomly select a color and
// a helicity for event ievt"; reading A15): the first good helicity k (increasing h) with rnd * sum < cum_k
__global__ void helicity_sum_select_kernel(const double* __restrict__ meh, int nhel, int nevt, const double* __restrict__ gfac,
                                           const double* __restrict__ rndhel, const int* __restrict__ good,
                                           double* __restrict__ me, int* __restrict__ selhel)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nevt) return;
    double s = 0.0;
    for (int h = 0; h < nhel; h++) s += meh[(size_t)h * nevt + e];
    me[e] = gfac ? gfac[e] * s : s;
    if (selhel) {
        const double target = rndhel[e] * s;
        double c = 0.0;
        int k = 0;
        for (; k < nhel - 1; k++) {
            c += meh[(size_t)k * nevt + e];
            if (target < c) break;
        }
        selhel[e] = good[k];
    }
}

// colour selection: weight of colour flow c = sum over good helicities of |J_c|^2; the first c with rnd * sum < cum_c.
// One warp per event; lanes stride over the event's rows.  LAYOUT 0: [2][nc][rows], row = el * nhel + ih (event-major);
// 1: [2][nc][rows], row = ih * ne + el (helicity-major); 2: tile-major [row / 128][2][nc][128], row = el * nhel + ih;
// 3: the tcgen05 operand layout of csrc/color_sum_tf32.cu (per tile and part: chunks of 24 colours as K-major core matrices)
template <typename T, int LAYOUT>
__global__ void __launch_bounds__(128) select_color_kernel(const T* __restrict__ J, int nc, int nhel, int ne, long rows,
                                                            const double* __restrict__ rndcol, int e0, int* __restrict__ selcol)
{
    extern __shared__ double wsm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int el = blockIdx.x * (blockDim.x >> 5) + warp;
    if (el >= ne) return;
    double* w = wsm + (size_t)warp * nc;
    for (int c = 0; c < nc; c++) {
        double s = 0.0;
        for (int ih = lane; ih < nhel; ih += 32) {
            double re, im;
            if (LAYOUT == 3) {
                const long row = (long)el * nhel + ih;
                const unsigned m = (unsigned)(row & 127);
                const T* t = J + (row >> 7) * (256L * nc) + (long)(c / 24) * (24 * 128) + (m >> 3) * 192 + ((c % 24) >> 2) * 32 + (m & 7) * 4 + (c & 3);
                re = (double)t[0]; im = (double)t[128L * nc];
            } else if (LAYOUT == 2) {
                const long row = (long)el * nhel + ih;
                const T* t = J + (row >> 7) * (256L * nc) + (long)c * 128 + (row & 127);
                re = (double)t[0]; im = (double)t[128L * nc];
            } else {
                const long row = LAYOUT == 0 ? (long)el * nhel + ih : (long)ih * ne + el;
                re = (double)J[(long)c * rows + row]; im = (double)J[(long)(nc + c) * rows + row];
            }
            s += re * re + im * im;
        }
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) w[c] = s;
    }
    __syncwarp();
    if (lane == 0) {
        double tot = 0.0;
        for (int c = 0; c < nc; c++) tot += w[c];
        const double target = rndcol[e0 + el] * tot;
        double cum = 0.0;
        int c = 0;
        for (; c < nc - 1; c++) {
            cum += w[c];
            if (target < cum) break;
        }
        selcol[e0 + el] = c;
    }
}

template <typename T>
static cudaError_t launch_select_color(int layout, const void* J, int nc, int nhel, int ne, long rows, const double* rnd, int e0,
                                       int* sel, cudaStream_t st)
{
    const int warps = 4;
    const unsigned grid = (unsigned)((ne + warps - 1) / warps);
    const size_t sm = sizeof(double) * warps * nc;
    if (layout == 0) select_color_kernel<T, 0><<<grid, 32 * warps, sm, st>>>((const T*)J, nc, nhel, ne, rows, rnd, e0, sel);
    else if (layout == 1) select_color_kernel<T, 1><<<grid, 32 * warps, sm, st>>>((const T*)J, nc, nhel, ne, rows, rnd, e0, sel);
    else if (layout == 3) select_color_kernel<T, 3><<<grid, 32 * warps, sm, st>>>((const T*)J, nc, nhel, ne, rows, rnd, e0, sel);
    else select_color_kernel<T, 2><<<grid, 32 * warps, sm, st>>>((const T*)J, nc, nhel, ne, rows, rnd, e0, sel);
    return cudaGetLastError();
}

static int set_good(mg_process* p, const std::vector<int>& good)
{
    p->good = good;
    p->epoch++;
    if (!good.empty()) {
        CUDA_TRY(p, cudaMemcpy(p->d_good, good.data(), good.size() * sizeof(int), cudaMemcpyHostToDevice));
        std::vector<int> pos(p->d->ncomb, -1);
        for (size_t i = 0; i < good.size(); i++) pos[good[i]] = (int)i;
        CUDA_TRY(p, cudaMemcpy(p->d_pos, pos.data(), pos.size() * sizeof(int), cudaMemcpyHostToDevice));
    }
    return MG_OK;
}

extern "C" int mg_set_good_helicities(mg_process* p, const unsigned char* h_mask)
{
    if (!p || !h_mask) return fail(p, MG_EINVAL, "bad arguments");
    CUDA_TRY(p, cudaSetDevice(p->device));
    std::vector<int> g;
    for (int h = 0; h < p->d->ncomb; h++) if (h_mask[h]) g.push_back(h);
    if (g.empty()) return fail(p, MG_EINVAL, "empty helicity mask");
    return set_good(p, g);
}

static DiagLaunch base_launch(const mg_process* p, const double* d_mom, int nevt)
{
    DiagLaunch a;
    memset(&a, 0, sizeof a);
    a.mom = d_mom; a.nevt = nevt; a.evt_stride = nevt; a.evt_offset = 0;
    a.ph = make_phys(p); a.norm = make_norm(p); a.d_cmat = p->d_cmat; a.block = p->block;
    return a;
}

extern "C" int mg_helicity_filter(mg_process* p, const double* d_momenta, int nprobe, void* d_workspace, size_t ws_bytes,
                                  void* cuda_stream, unsigned char* h_mask, int* ngood)
{
    if (!p || !d_momenta || nprobe <= 0 || !d_workspace) return fail(p, MG_EINVAL, "bad arguments");
    const int ncomb = p->d->ncomb;
    const size_t need = (size_t)ncomb * nprobe * sizeof(double);
    if (ws_bytes < filter_bytes(p, nprobe)) return fail(p, MG_EINVAL, "workspace too small for the helicity filter");
    CUDA_TRY(p, cudaSetDevice(p->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (!p->d->launch) {
        // generic helicity-shared kernel: every helicity combination is a row of its event (d_all = identity), then the
        // colour sum over the probe's rows
        const long rows = (long)ncomb * nprobe;
        HsLaunch a;
        a.mom = d_momenta; a.nevt = nprobe; a.d_pos = p->d_all; a.nrow_evt = ncomb;
        a.d_jamps = (char*)d_workspace + align256(need); a.rows = color_sum_padded_rows(rows); a.mt = p->mT; a.wt = p->wT; a.tile_major = 0;
        CUDA_TRY(p, hsg_launch(p->hsg, true, a, st));
        RowMap map;
        map.rows_valid = rows; map.hel_minor = ncomb; map.evt_stride = nprobe; map.e0 = 0; map.norm = make_norm(p);
        CUDA_TRY(p, color_sum_tensor(true, p->d->ncolor, p->d_cmat64, p->d_chol64, a.d_jamps, a.rows, map, (double*)d_workspace, st));
    } else {
        DiagLaunch a = base_launch(p, d_momenta, nprobe);
        a.d_hel = p->d_all; a.hel_base = 0; a.nhel = ncomb; a.d_meh = (double*)d_workspace; a.mode = MG_CS_FUSED;
        a.d_cmat = p->d_cmat64;
        CUDA_TRY(p, p->d->launch(MG_FP64, a, st));      // both sides decide in fp64 whatever the handle's precision (reading A5)
    }
    std::vector<double> h(need / sizeof(double));
    CUDA_TRY(p, cudaMemcpyAsync(h.data(), d_workspace, need, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(p, cudaStreamSynchronize(st));
    std::vector<int> good;
    std::vector<double> tot(nprobe, 0.0);
    for (int hh = 0; hh < ncomb; hh++)
        for (int e = 0; e < nprobe; e++) tot[e] += h[(size_t)hh * nprobe + e];
    for (int hh = 0; hh < ncomb; hh++) {
        bool ok = false;
        for (int e = 0; e < nprobe && !ok; e++)
            if (tot[e] > 0 && h[(size_t)hh * nprobe + e] > 1e-8 * tot[e]) ok = true;
        if (h_mask) h_mask[hh] = ok ? 1 : 0;
        if (ok) good.push_back(hh);
    }
    if (ngood) *ngood = (int)good.size();
    if (good.empty()) return fail(p, MG_ESTATE, "helicity filter found no contributing helicity");
    return set_good(p, good);
}

static int ensure_streams(mg_process* p, int n)
{
    while ((int)p->streams.size() < n) {
        cudaStream_t s; cudaEvent_t e;
        CUDA_TRY(p, cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking));
        CUDA_TRY(p, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        p->streams.push_back(s); p->ev_join.push_back(e);
    }
    if (!p->ev_fork) CUDA_TRY(p, cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
    return MG_OK;
}

// timing mark: the work enqueued since the previous mark belongs to `stage` (-1 = start of the batch)
static int mark(mg_process* p, int stage, cudaStream_t st)
{
    if (!p->timing) return MG_OK;
    if (p->ev_n == (int)p->ev_pool.size()) {
        cudaEvent_t e;
        CUDA_TRY(p, cudaEventCreate(&e));
        p->ev_pool.push_back(e); p->ev_stage.push_back(0);
    }
    p->ev_stage[p->ev_n] = stage;
    CUDA_TRY(p, cudaEventRecord(p->ev_pool[p->ev_n], st));
    p->ev_n++;
    return MG_OK;
}
#define MARK(stage) do { int rc_ = mark(p, stage, st); if (rc_ != MG_OK) return rc_; } while (0)

// diagram stage for events [e0, e0+ne) of the batch, all good helicities
static int run_diagrams(mg_process* p, DiagLaunch a, cudaStream_t st)
{
    const int nhel = (int)p->good.size();
    if (p->schedule == MG_SCHED_GRID) {
        a.hel_base = 0; a.nhel = nhel;
        CUDA_TRY(p, p->d->launch(p->precision, a, st));
        p->launches++;
    } else {
        // one stream per good helicity, or a fixed number of them shared round robin ("study how
        // many streams are actually useful, and limit them to a fixed number")
        const int ns = p->max_streams > 0 && p->max_streams < nhel ? p->max_streams : nhel;
        int rc = ensure_streams(p, ns);
        if (rc != MG_OK) return rc;
        CUDA_TRY(p, cudaEventRecord(p->ev_fork, st));
        for (int s_ = 0; s_ < ns; s_++) CUDA_TRY(p, cudaStreamWaitEvent(p->streams[s_], p->ev_fork, 0));
        for (int h = 0; h < nhel; h++) {
            a.hel_base = h; a.nhel = 1;
            CUDA_TRY(p, p->d->launch(p->precision, a, p->streams[h % ns]));
            p->launches++;
        }
        for (int s_ = 0; s_ < ns; s_++) {
            CUDA_TRY(p, cudaEventRecord(p->ev_join[s_], p->streams[s_]));
            CUDA_TRY(p, cudaStreamWaitEvent(st, p->ev_join[s_], 0));
        }
    }
    return MG_OK;
}

static int sigma_batch_impl(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace,
                            size_t ws_bytes, void* cuda_stream, const Extras& ex)
{
    if (!p || nevt < 0) return fail(p, MG_EINVAL, "bad arguments");
    if (nevt == 0) return MG_OK;
    if (!d_momenta || !d_me || !d_workspace) return fail(p, MG_EINVAL, "NULL buffer");
    if (((size_t)d_workspace & 255) != 0) return fail(p, MG_EINVAL, "workspace must be 256-byte aligned");
    CUDA_TRY(p, cudaSetDevice(p->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((ex.selhel != nullptr) != (ex.rndhel != nullptr) || (ex.selcol != nullptr) != (ex.rndcol != nullptr))
        return fail(p, MG_EINVAL, "a selection output needs its random-number input and vice versa");
    const bool want_col = ex.selcol != nullptr && p->d->ncolor > 1;
    if (ws_bytes < workspace_bytes(p, nevt, want_col)) return fail(p, MG_EINVAL, "workspace too small");
    if (p->good.empty()) {
        const int nprobe = probe_events(p, nevt);
        int rc = mg_helicity_filter(p, d_momenta, nprobe, d_workspace, ws_bytes, cuda_stream, nullptr, nullptr);
        if (rc != MG_OK) return rc;
        if (ws_bytes < workspace_bytes(p, nevt, want_col)) return fail(p, MG_EINVAL, "workspace too small");
    }
    const int nhel = (int)p->good.size();
    double* d_meh = (double*)d_workspace;
    double* d_gfac = (double*)((char*)d_workspace + align256((size_t)nhel * nevt * sizeof(double)));
    char* d_j = (char*)d_gfac + align256((size_t)nevt * sizeof(double));
    // colour selection reads the jamps: the thread kernel then takes its jamps-buffer path whatever "color_sum" says
    const int color_sum = want_col ? MG_CS_TENSOR : p->color_sum;
    auto select_color = [&](int layout, const void* J, int ne, long rows, int e0) -> cudaError_t {
        if (!want_col) return cudaSuccess;
        p->launches++;
        return p->precision == MG_FP64 ? launch_select_color<double>(layout, J, p->d->ncolor, nhel, ne, rows, ex.rndcol, e0, ex.selcol, st)
                                       : launch_select_color<float>(layout, J, p->d->ncolor, nhel, ne, rows, ex.rndcol, e0, ex.selcol, st);
    };
    p->timed = false; p->ev_n = 0; p->launches = 0;
    MARK(-1);
    if (p->diagrams == MG_DIAG_SHARED) {
        // helicity-shared diagram kernel -> jamps [2][ncolor][rows], rows (event, helicity) -> colour-sum kernel
        const int ce = chunk_events(p, nevt, nhel);
        for (int e0 = 0; e0 < nevt; e0 += ce) {
            const int ne = nevt - e0 < ce ? nevt - e0 : ce;
            const long rows = (long)nhel * ne;
            HsLaunch a;
            a.mom = d_momenta + (size_t)e0 * p->d->npar * 4; a.nevt = ne; a.d_pos = p->d_pos; a.nrow_evt = nhel;
            a.d_jamps = d_j; a.rows = color_sum_padded_rows(rows); a.mt = p->mT; a.wt = p->wT;
            // tcgen05 colour sum: one contiguous block per 128-row tile, so that a chunk of colours is ONE bulk copy
            // (2: straight in the operand layout, TF32-rounded -- the contraction then needs neither converter warps nor the
            //  low term of the jamps; needs chunks of 24 colours)
            // (the generic kernel has the operand layout only: options "hs_color_alu" / "tf32_direct" do not apply to it)
            const bool alu = p->hs_color_alu && !p->hsg;
            const int tile_major = p->precision != MG_FP64 && !alu ? (p->hsg || (p->d->ncolor % 24 == 0 && p->tf32_direct) ? 2 : 1) : 0;
            a.tile_major = tile_major;
            if (p->hsg) CUDA_TRY(p, hsg_launch(p->hsg, p->precision == MG_FP64, a, st));
            else CUDA_TRY(p, hs_launch(p->hs, p->precision == MG_FP64, a, st));
            p->launches += 2;                      // + the colour-sum kernel below
            MARK(0);
            RowMap map;
            map.rows_valid = rows; map.hel_minor = nhel; map.evt_stride = nevt; map.e0 = e0; map.norm = make_norm(p);
            cudaError_t ce_;
            // tensor-core contraction (DMMA in MG_FP64, tcgen05 kind::tf32 otherwise) unless the ALU kernel is asked for
            if (alu && p->precision != MG_FP64)
                ce_ = color_sum_alu(false, p->d->ncolor, p->d_cmat, d_j, a.rows, d_meh, st, &map);
            else
                ce_ = color_sum_tensor(p->precision == MG_FP64, p->d->ncolor, p->d_cmat, p->d_chol, d_j, a.rows, map, d_meh, st, tile_major);
            if (ce_ != cudaSuccess) return fail(p, MG_ECUDA, std::string("colour sum: ") + cudaGetErrorString(ce_));
            CUDA_TRY(p, select_color(tile_major == 2 ? 3 : (tile_major ? 2 : 0), d_j, ne, a.rows, e0));
            MARK(1);
        }
    } else if (color_sum == MG_CS_FUSED) {
        DiagLaunch a = base_launch(p, d_momenta, nevt);
        a.d_hel = p->d_good; a.d_meh = d_meh; a.mode = MG_CS_FUSED;
        int rc = run_diagrams(p, a, st);
        if (rc != MG_OK) return rc;
        MARK(0);
    } else {
        const int ce = chunk_events(p, nevt, nhel);
        for (int e0 = 0; e0 < nevt; e0 += ce) {
            const int ne = nevt - e0 < ce ? nevt - e0 : ce;
            const long rows = (long)nhel * ne;
            DiagLaunch a = base_launch(p, d_momenta + (size_t)e0 * p->d->npar * 4, ne);
            a.d_hel = p->d_good; a.mode = MG_CS_TENSOR; a.d_jamps = d_j; a.rows = color_sum_padded_rows(rows);
            int rc = run_diagrams(p, a, st);
            if (rc != MG_OK) return rc;
            MARK(0);
            // rows are (helicity-major, event-minor); the contraction writes norm * J^T C J per row into me_h
            RowMap map;
            map.rows_valid = rows; map.ne = ne; map.evt_stride = nevt; map.e0 = e0; map.norm = make_norm(p);
            cudaError_t ce_ = color_sum_tensor(p->precision == MG_FP64, p->d->ncolor, p->d_cmat, p->d_chol, d_j, a.rows, map, d_meh, st);
            if (ce_ != cudaSuccess) return fail(p, MG_ECUDA, std::string("color_sum_tensor: ") + cudaGetErrorString(ce_));
            p->launches++;
            CUDA_TRY(p, select_color(1, d_j, ne, a.rows, e0));
            MARK(1);
        }
    }
    if (ex.selcol && !want_col) CUDA_TRY(p, cudaMemsetAsync(ex.selcol, 0, (size_t)nevt * sizeof(int), st));      // one colour flow
    if (ex.alphas || ex.selhel) {
        if (ex.alphas) {
            couplings_kernel<<<(nevt + 255) / 256, 256, 0, st>>>(ex.alphas, nevt, p->d->coupling_order, 4.0 * M_PI * p->aS, d_gfac);
            CUDA_TRY(p, cudaGetLastError());
            p->launches++;
        }
        helicity_sum_select_kernel<<<(nevt + 255) / 256, 256, 0, st>>>(d_meh, nhel, nevt, ex.alphas ? d_gfac : nullptr, ex.rndhel,
                                                                       p->d_good, d_me, ex.selhel);
    } else
        helicity_sum_kernel<<<(nevt + 255) / 256, 256, 0, st>>>(d_meh, nhel, nevt, d_me);
    CUDA_TRY(p, cudaGetLastError());
    p->launches++;
    MARK(2);
    p->timed = p->timing != 0;
    return MG_OK;
}

// option "graph": the launch sequence of a batch (diagram kernels on their helicity streams, colour sums, selections, helicity
// sum) is captured into a CUDA graph on its first execution and replayed while the arguments and the handle's state stay
// the same -- the paper's gpuDiagrams wrapper ("configures graphs on its first execution ... on
// subsequent executions it runs kernels via graphs rather than launching them individually")
static int sigma_batch_graph(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace, size_t ws_bytes,
                             void* cuda_stream, const Extras& ex)
{
    if (!p) return MG_EINVAL;
    if (!p->graph || p->timing || nevt <= 0)
        return sigma_batch_impl(p, d_momenta, nevt, d_me, d_workspace, ws_bytes, cuda_stream, ex);
    CUDA_TRY(p, cudaSetDevice(p->device));
    cudaStream_t user = (cudaStream_t)cuda_stream;
    if (p->good.empty()) {          // the filter synchronises: not capturable, and it changes what a batch launches
        if (!d_momenta || !d_workspace) return fail(p, MG_EINVAL, "NULL buffer");
        int rc = mg_helicity_filter(p, d_momenta, nevt < 1024 ? nevt : 1024, d_workspace, ws_bytes, cuda_stream, nullptr, nullptr);
        if (rc != MG_OK) return rc;
    }
    // the legacy default stream cannot be captured: run on a library stream ordered after / before it with events
    cudaStream_t st = user;
    if (user == nullptr || user == cudaStreamLegacy) {
        if (!p->gstream) {
            CUDA_TRY(p, cudaStreamCreateWithFlags(&p->gstream, cudaStreamNonBlocking));
            CUDA_TRY(p, cudaEventCreateWithFlags(&p->gev_in, cudaEventDisableTiming));
            CUDA_TRY(p, cudaEventCreateWithFlags(&p->gev_out, cudaEventDisableTiming));
        }
        st = p->gstream;
        CUDA_TRY(p, cudaEventRecord(p->gev_in, user));
        CUDA_TRY(p, cudaStreamWaitEvent(st, p->gev_in, 0));
    }
    mg_process::GraphKey key;
    key.mom = d_momenta; key.me = d_me; key.ws = d_workspace; key.nevt = nevt; key.st = st; key.epoch = p->epoch;
    key.ex[0] = ex.alphas; key.ex[1] = ex.rndhel; key.ex[2] = ex.rndcol; key.ex[3] = ex.selhel; key.ex[4] = ex.selcol;
    if (!(p->gexec && key == p->gkey)) {
        if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }
        CUDA_TRY(p, cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed));
        const int rc = sigma_batch_impl(p, d_momenta, nevt, d_me, d_workspace, ws_bytes, st, ex);
        cudaGraph_t g = nullptr;
        const cudaError_t ce = cudaStreamEndCapture(st, &g);          // always leave capture mode
        if (rc != MG_OK) { if (g) cudaGraphDestroy(g); return rc; }
        if (ce != cudaSuccess) return fail(p, MG_ECUDA, std::string("cudaStreamEndCapture: ") + cudaGetErrorString(ce));
        const cudaError_t ci = cudaGraphInstantiate(&p->gexec, g, 0);
        cudaGraphDestroy(g);
        if (ci != cudaSuccess) { p->gexec = nullptr; return fail(p, MG_ECUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ci)); }
        p->gkey = key;
        p->graph_replays = 0;
    } else
        p->graph_replays++;
    CUDA_TRY(p, cudaGraphLaunch(p->gexec, st));
    if (st != user) {
        CUDA_TRY(p, cudaEventRecord(p->gev_out, st));
        CUDA_TRY(p, cudaStreamWaitEvent(user, p->gev_out, 0));
    }
    return MG_OK;
}

extern "C" int mg_sigma_batch(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace,
                              size_t ws_bytes, void* cuda_stream)
{
    return sigma_batch_graph(p, d_momenta, nevt, d_me, d_workspace, ws_bytes, cuda_stream, Extras());
}

extern "C" int mg_sigma_batch_ex(mg_process* p, const double* d_momenta, int nevt, const double* d_alphas, const double* d_rndhel,
                                 const double* d_rndcol, double* d_me, int* d_selhel, int* d_selcol, void* d_workspace,
                                 size_t ws_bytes, void* cuda_stream)
{
    Extras ex;
    ex.alphas = d_alphas; ex.rndhel = d_rndhel; ex.rndcol = d_rndcol; ex.selhel = d_selhel; ex.selcol = d_selcol;
    return sigma_batch_graph(p, d_momenta, nevt, d_me, d_workspace, ws_bytes, cuda_stream, ex);
}

extern "C" int mg_last_launch_count(const mg_process* p, int* launches)
{
    if (!p || !launches) return MG_EINVAL;
    *launches = p->launches;
    return MG_OK;
}

extern "C" int mg_last_stage_ms(mg_process* p, float ms[3])
{
    if (!p || !ms) return MG_EINVAL;
    if (!p->timed) return fail(p, MG_ESTATE, "no timed batch (set option timing=1 first)");
    CUDA_TRY(p, cudaEventSynchronize(p->ev_pool[p->ev_n - 1]));
    ms[0] = ms[1] = ms[2] = 0.f;
    for (int k = 1; k < p->ev_n; k++) {
        float t = 0.f;
        CUDA_TRY(p, cudaEventElapsedTime(&t, p->ev_pool[k - 1], p->ev_pool[k]));
        ms[p->ev_stage[k]] += t;
    }
    return MG_OK;
}

extern "C" int mg_last_helicity_terms(mg_process* p, int nevt, const void* d_workspace, double* d_out, void* cuda_stream)
{
    if (!p || !d_workspace || !d_out || nevt <= 0 || p->good.empty()) return fail(p, MG_EINVAL, "bad arguments");
    CUDA_TRY(p, cudaMemcpyAsync(d_out, d_workspace, p->good.size() * (size_t)nevt * sizeof(double), cudaMemcpyDeviceToDevice,
                                (cudaStream_t)cuda_stream));
    return MG_OK;
}

extern "C" int mg_sigma_batch_host(mg_process* p, const double* h_momenta, int nevt, double* h_me)
{
    if (!p || nevt < 0) return fail(p, MG_EINVAL, "bad arguments");
    if (nevt == 0) return MG_OK;
    if (!h_momenta || !h_me) return fail(p, MG_EINVAL, "NULL buffer");
    CUDA_TRY(p, cudaSetDevice(p->device));
    const size_t mom_bytes = (size_t)nevt * p->d->npar * 4 * sizeof(double);
    if (nevt > p->own_nevt) {
        cudaFree(p->d_mom_own); cudaFree(p->d_me_own); p->d_mom_own = nullptr; p->d_me_own = nullptr; p->own_nevt = 0;
        CUDA_TRY(p, cudaMalloc(&p->d_mom_own, mom_bytes));
        CUDA_TRY(p, cudaMalloc(&p->d_me_own, (size_t)nevt * sizeof(double)));
        p->own_nevt = nevt;
    }
    size_t ws = mg_workspace_bytes(p, nevt);
    size_t ws_all = ws_bytes_for(p, nevt, p->d->ncomb);      // enough for whatever the filter decides
    if (ws_all > ws) ws = ws_all;
    if (ws > p->own_ws) {
        cudaFree(p->d_ws_own); p->d_ws_own = nullptr; p->own_ws = 0;
        CUDA_TRY(p, cudaMalloc(&p->d_ws_own, ws));
        p->own_ws = ws;
    }
    CUDA_TRY(p, cudaMemcpyAsync(p->d_mom_own, h_momenta, mom_bytes, cudaMemcpyHostToDevice, 0));
    int rc = mg_sigma_batch(p, p->d_mom_own, nevt, p->d_me_own, p->d_ws_own, p->own_ws, nullptr);
    if (rc != MG_OK) return rc;
    CUDA_TRY(p, cudaMemcpyAsync(h_me, p->d_me_own, (size_t)nevt * sizeof(double), cudaMemcpyDeviceToHost, 0));
    CUDA_TRY(p, cudaStreamSynchronize(0));
    return MG_OK;
}

extern "C" int mg_color_matrix(const mg_process* p, int* h_numerators, int* denominator)
{
    if (!p) return MG_EINVAL;
    if (h_numerators) memcpy(h_numerators, p->d->cmat, sizeof(int) * p->d->ncolor * p->d->ncolor);
    if (denominator) *denominator = p->d->cden;
    return MG_OK;
}

// The entry point that allocates nothing (include/mg5_b200.h): diagram kernel with its scratch areas in the static __device__
// array of csrc/hsg_kernel.cu, colour sum, helicity sum -- the launch sequence of sigma_batch_impl for the generic
// helicity-shared kernel, written out here so that no existing path changes.  No cudaMalloc / cudaFree / allocating library
// call, no host-side containers on the success path, no synchronisation, no helicity filter.
extern "C" int mg_sigma_batch_noalloc(mg_process* p, const double* d_momenta, int nevt, double* d_me, void* d_workspace,
                                      size_t ws_bytes, void* cuda_stream)
{
    if (!p || nevt < 0) return fail(p, MG_EINVAL, "bad arguments");
    if (!p->hsg) return fail(p, MG_EINVAL, "mg_sigma_batch_noalloc: this process has no kernel that uses scratch memory (gg_ttxgggg only)");
    if (nevt > MG_NOALLOC_MAX_EVENTS) {
        char buf[160];
        snprintf(buf, sizeof buf, "mg_sigma_batch_noalloc: nevt = %d, at most %d events per call (static scratch: 26 MiB, %d CTAs)",
                 nevt, MG_NOALLOC_MAX_EVENTS, hsg_static_ctas(p->hsg));
        return fail(p, MG_EINVAL, buf);
    }
    if (nevt == 0) return MG_OK;
    if (!d_momenta || !d_me || !d_workspace) return fail(p, MG_EINVAL, "NULL buffer");
    if (((size_t)d_workspace & 255) != 0) return fail(p, MG_EINVAL, "workspace must be 256-byte aligned");
    if (p->good.empty())
        return fail(p, MG_ESTATE, "mg_sigma_batch_noalloc: no good-helicity list (call mg_helicity_filter or mg_set_good_helicities first)");
    if (hsg_static_ctas(p->hsg) < 1) return fail(p, MG_ESTATE, "mg_sigma_batch_noalloc: the static scratch array is too small for this process");
    CUDA_TRY(p, cudaSetDevice(p->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nhel = (int)p->good.size();
    const long rows = (long)nhel * nevt, rows_p = color_sum_padded_rows(rows);
    const size_t meh_b = align256((size_t)nhel * nevt * sizeof(double)), gfac_b = align256((size_t)nevt * sizeof(double));
    if (ws_bytes < meh_b + gfac_b + align256((size_t)rows_p * p->d->ncolor * 2 * cs_elem(p)))
        return fail(p, MG_EINVAL, "workspace too small (mg_workspace_bytes)");
    double* d_meh = (double*)d_workspace;
    char* d_j = (char*)d_workspace + meh_b + gfac_b;
    HsLaunch a;
    a.mom = d_momenta; a.nevt = nevt; a.d_pos = p->d_pos; a.nrow_evt = nhel;
    a.d_jamps = d_j; a.rows = rows_p; a.mt = p->mT; a.wt = p->wT;
    a.tile_major = p->precision != MG_FP64 ? 2 : 0;
    CUDA_TRY(p, hsg_launch_static(p->hsg, p->precision == MG_FP64, a, st));
    RowMap map;
    map.rows_valid = rows; map.hel_minor = nhel; map.evt_stride = nevt; map.e0 = 0; map.norm = make_norm(p);
    CUDA_TRY(p, color_sum_tensor(p->precision == MG_FP64, p->d->ncolor, p->d_cmat, p->d_chol, d_j, rows_p, map, d_meh, st, a.tile_major));
    helicity_sum_kernel<<<(nevt + 255) / 256, 256, 0, st>>>(d_meh, nhel, nevt, d_me);
    CUDA_TRY(p, cudaGetLastError());
    p->timed = false; p->launches = 3;
    return MG_OK;
}

extern "C" int mg_color_sum(mg_process* p, int impl, const void* d_jamps, long nrows, double* d_out, void* cuda_stream)
{
    if (!p || !d_jamps || !d_out || nrows <= 0) return fail(p, MG_EINVAL, "bad arguments");
    CUDA_TRY(p, cudaSetDevice(p->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (impl == MG_CS_FUSED) e = color_sum_alu(p->precision == MG_FP64, p->d->ncolor, p->d_cmat, d_jamps, nrows, d_out, st);
    else if (impl == MG_CS_TENSOR) {
        if (nrows != color_sum_padded_rows(nrows)) return fail(p, MG_EINVAL, "nrows must be a multiple of 128 for the tensor kernel");
        RowMap map;
        map.rows_valid = nrows;
        e = color_sum_tensor(p->precision == MG_FP64, p->d->ncolor, p->d_cmat, p->d_chol, d_jamps, nrows, map, d_out, st);
    } else return fail(p, MG_EINVAL, "bad impl");
    if (e != cudaSuccess) return fail(p, MG_ECUDA, std::string("color sum: ") + cudaGetErrorString(e));
    return MG_OK;
}
