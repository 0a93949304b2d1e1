// eemumu.cu -- e+ e- -> mu+ mu- (BASELINE.json config 1; not in the paper): two diagrams,
// s-channel photon and Z, one colour, hand-written.  Particle order e+ e- mu+ mu-.
//   M_h = [vbar(e+) gamma^mu G_V u(e-)] [ubar(mu-) gamma_mu G_V v(mu+)] P_V summed over V = photon, Z
//   G_photon = -e, P_photon = 1/s;  G_Z = gL PL + gR PR, P_Z = 1/(s - mZ^2 + i mZ wZ)
// (FFV2/FFV4-like chiral currents of helas.cuh; the k^mu k^nu/mZ^2 term vanishes for massless leptons).
#include "proc_kernels.cuh"

namespace mg {
namespace epem_mupmum {
constexpr int NGLUON = 0, NPAR = 4, NCOMB = 16, NCOLOR = 1, NDIAGRAMS = 2, NAMPS = 2, NCURRENTS = 6;
constexpr double DENOM = 4.0;
constexpr int CDEN = 1;
constexpr double FLOPS_PER_EVENT_HELICITY = 4 * 40 + 2 * (2 * 70 + 30) + 20;
static const int CMAT[1] = { 1 };

template <typename T>
__device__ __forceinline__ void jamps(const double* __restrict__ pe, int ihel, const phys<T>& ph, cx<T>* __restrict__ jamp)
{
    T p[4][4];
    for (int i = 0; i < 4; i++)
        for (int mu = 0; mu < 4; mu++) p[i][mu] = T(pe[4 * i + mu]);
    const int l0 = ((ihel >> 3) & 1) ? 1 : -1, l1 = ((ihel >> 2) & 1) ? 1 : -1;
    const int l2 = ((ihel >> 1) & 1) ? 1 : -1, l3 = (ihel & 1) ? 1 : -1;
    wf<T> vbar_ep, u_em, v_mup, ubar_mum;
    ext_vbar(p[0], T(0), l0, vbar_ep);
    ext_u(p[1], T(0), l1, u_em);
    ext_v(p[2], T(0), l2, v_mup);
    ext_ubar(p[3], T(0), l3, ubar_mum);
    const T q[4] = { p[0][0] + p[1][0], p[0][1] + p[1][1], p[0][2] + p[1][2], p[0][3] + p[1][3] };
    const T s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3];
    // diagram 1: photon
    wf<T> je, jm;
    ffv_lr_current(vbar_ep, u_em, -ph.ee, -ph.ee, je);
    ffv_lr_current(ubar_mum, v_mup, -ph.ee, -ph.ee, jm);
    cx<T> amp = (T(1) / s) * dot(je, jm);
    // diagram 2: Z
    ffv_lr_current(vbar_ep, u_em, ph.gl, ph.gr, je);
    ffv_lr_current(ubar_mum, v_mup, ph.gl, ph.gr, jm);
    amp += inv_prop(s, ph.mz, ph.wz) * dot(je, jm);
    jamp[0] = amp;
}
}  // namespace epem_mupmum

struct P_epem_mupmum {
    static constexpr int NPAR = 4, NCOLOR = 1;
    template <typename T>
    static __device__ __forceinline__ void jamps(const double* pe, int ihel, const phys<T>& ph, cx<T>* j)
    {
        epem_mupmum::jamps<T>(pe, ihel, ph, j);
    }
    static cudaError_t launch_f32(const DiagLaunch& a, cudaStream_t st) { return launch_t<P_epem_mupmum, float, float>(a, st); }
};

const ProcessDesc* desc_epem_mupmum()
{
    using namespace epem_mupmum;
    static const ProcessDesc d = { "epem_mupmum", NGLUON, NPAR, NCOMB, NCOLOR, NDIAGRAMS, NAMPS, NCURRENTS, 1,
                                   DENOM, CDEN, CMAT, FLOPS_PER_EVENT_HELICITY, 0, true, &launch_any<P_epem_mupmum> };
    return &d;
}
}  // namespace mg
