// helas.cuh -- helicity-amplitude building blocks (external wavefunctions, off-shell currents, amplitudes).
//
// Roles follow the HELAS/ALOHA routines the paper names ("wavefunctions of external
// particles, via functions like VXXXXX; the wavefunctions of internal propagators, e.g. via VVV1P0_1; the
// dual amplitudes ..., e.g. via FFV1_0"), but the code is written from the Feynman rules, not from those
// sources (which are not available here):
//   metric (+,-,-,-), chiral (Weyl) representation  gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s_i],[-s_i,0]],
//   a wavefunction is 4 complex numbers (spinor components or the contravariant vector components);
//   momenta are NOT carried inside the wavefunction as in HELAS (PAPER.md:141 fn 2: 6 complex): they are
//   sums of external momenta and are kept per leg set.
// All-incoming momentum convention: k = +p for the two beams, -p for final-state particles.
// Couplings and the common phase are factored out of every routine: each vertex
// below is the bare Lorentz structure, so that a diagram term is colour(bare commutators) x Lorentz(bare).
//
// Everything is templated on the real type T (double, float) and usable on the host (tests compile this
// header with g++ to check the routines on CPU; the library itself only instantiates device code).
#pragma once

#include <math.h>

#if defined(__CUDACC__)
#define MG_HD __host__ __device__ __forceinline__
#else
#define MG_HD inline
#endif

namespace mg {

template <typename T>
struct cx {
    T re, im;
};

template <typename T> MG_HD cx<T> mk(T re, T im) { cx<T> r; r.re = re; r.im = im; return r; }
template <typename T> MG_HD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> MG_HD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> MG_HD cx<T> operator-(cx<T> a) { return mk<T>(-a.re, -a.im); }
template <typename T> MG_HD cx<T> operator*(cx<T> a, cx<T> b) { return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <typename T> MG_HD cx<T> operator*(T a, cx<T> b) { return mk<T>(a * b.re, a * b.im); }
template <typename T> MG_HD cx<T> operator*(cx<T> b, T a) { return mk<T>(a * b.re, a * b.im); }
template <typename T> MG_HD cx<T>& operator+=(cx<T>& a, cx<T> b) { a.re += b.re; a.im += b.im; return a; }
template <typename T> MG_HD cx<T>& operator-=(cx<T>& a, cx<T> b) { a.re -= b.re; a.im -= b.im; return a; }
template <typename T> MG_HD cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <typename T> MG_HD cx<T> times_i(cx<T> a) { return mk<T>(-a.im, a.re); }      //  i * a
template <typename T> MG_HD cx<T> times_mi(cx<T> a) { return mk<T>(a.im, -a.re); }     // -i * a
// a + b*c  (complex multiply-add, 4 FMAs)
template <typename T> MG_HD cx<T> cfma(cx<T> b, cx<T> c, cx<T> a)
{
    return mk<T>(a.re + b.re * c.re - b.im * c.im, a.im + b.re * c.im + b.im * c.re);
}

// a - b*c  (4 FMAs)
template <typename T> MG_HD cx<T> cfms(cx<T> b, cx<T> c, cx<T> a)
{
    return mk<T>(a.re - b.re * c.re + b.im * c.im, a.im - b.re * c.im - b.im * c.re);
}

template <typename T>
struct p4 {            // real four-vector (E, x, y, z)
    T e, x, y, z;
};
template <typename T> MG_HD p4<T> operator+(p4<T> a, p4<T> b) { p4<T> r = { a.e + b.e, a.x + b.x, a.y + b.y, a.z + b.z }; return r; }
template <typename T> MG_HD p4<T> operator-(p4<T> a, p4<T> b) { p4<T> r = { a.e - b.e, a.x - b.x, a.y - b.y, a.z - b.z }; return r; }
template <typename T> MG_HD p4<T> operator-(p4<T> a) { p4<T> r = { -a.e, -a.x, -a.y, -a.z }; return r; }
template <typename T> MG_HD T m2(p4<T> a) { return a.e * a.e - a.x * a.x - a.y * a.y - a.z * a.z; }

template <typename T>
struct wf {            // wavefunction: 4 complex components
    cx<T> c[4];
};

// Minkowski products (no complex conjugation)
template <typename T> MG_HD cx<T> dot(const wf<T>& a, const wf<T>& b)
{
    return cfms(a.c[3], b.c[3], cfms(a.c[2], b.c[2], cfms(a.c[1], b.c[1], a.c[0] * b.c[0])));     // FMA chain
}
template <typename T> MG_HD cx<T> dot(p4<T> k, const wf<T>& a)
{
    return mk<T>(k.e * a.c[0].re - k.x * a.c[1].re - k.y * a.c[2].re - k.z * a.c[3].re,
                 k.e * a.c[0].im - k.x * a.c[1].im - k.y * a.c[2].im - k.z * a.c[3].im);
}

template <typename T> MG_HD T rsqrt_(T x) { return T(1) / sqrt(x); }

// ------------------------------------------------------------------------------------------------
// external wavefunctions (the hard-coded, branchy routines of PAPER.md:135: ixxxxx/oxxxxx/vxxxxx)

// two-component helicity eigenstate chi_lambda(p^), lambda = +-1; p along -z (or at rest) handled explicitly
template <typename T> MG_HD void chi2(T px, T py, T pz, T pp, int lambda, cx<T>& x0, cx<T>& x1)
{
    const T ppz = pp + pz;
    if (pp == T(0)) {                       // at rest: quantise along +z
        x0 = mk<T>(lambda > 0 ? T(1) : T(0), T(0));
        x1 = mk<T>(lambda > 0 ? T(0) : T(1), T(0));
    } else if (ppz <= pp * T(1e-7) * T(1e-7)) {   // along -z: azimuth := 0
        x0 = mk<T>(lambda > 0 ? T(0) : T(-1), T(0));
        x1 = mk<T>(lambda > 0 ? T(1) : T(0), T(0));
    } else {
        const T nrm = rsqrt_(T(2) * pp * ppz);
        if (lambda > 0) { x0 = mk<T>(ppz * nrm, T(0)); x1 = mk<T>(px * nrm, py * nrm); }
        else            { x0 = mk<T>(-px * nrm, py * nrm); x1 = mk<T>(ppz * nrm, T(0)); }
    }
}

// u(p, lambda) = (sqrt(E - lambda|p|) chi_lambda, sqrt(E + lambda|p|) chi_lambda): incoming fermion ("ixxxxx", nsf=+1)
template <typename T> MG_HD void ext_u(const T p[4], T m, int lambda, wf<T>& u)
{
    const T pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
    const T sp = sqrt(p[0] + pp);
    const T sm = m > T(0) ? m / sp : T(0);          // sqrt(E - |p|) = m / sqrt(E + |p|)
    cx<T> x0, x1;
    chi2(p[1], p[2], p[3], pp, lambda, x0, x1);
    const T lo = lambda > 0 ? sm : sp, hi = lambda > 0 ? sp : sm;
    u.c[0] = lo * x0; u.c[1] = lo * x1; u.c[2] = hi * x0; u.c[3] = hi * x1;
}

// v(p, lambda) = (sqrt(E + lambda|p|) chi_{-lambda}, -sqrt(E - lambda|p|) chi_{-lambda}): outgoing antifermion
// of physical helicity lambda ("ixxxxx", nsf=-1)
template <typename T> MG_HD void ext_v(const T p[4], T m, int lambda, wf<T>& v)
{
    const T pp = sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
    const T sp = sqrt(p[0] + pp);
    const T sm = m > T(0) ? m / sp : T(0);
    cx<T> x0, x1;
    chi2(p[1], p[2], p[3], pp, -lambda, x0, x1);
    const T up = lambda > 0 ? sp : sm, dn = lambda > 0 ? -sm : -sp;
    v.c[0] = up * x0; v.c[1] = up * x1; v.c[2] = dn * x0; v.c[3] = dn * x1;
}

// Dirac adjoint as a row: psibar = psi^dagger gamma^0 = (conj psi_2, conj psi_3, conj psi_0, conj psi_1)
template <typename T> MG_HD void dirac_bar(const wf<T>& s, wf<T>& b)
{
    b.c[0] = conj(s.c[2]); b.c[1] = conj(s.c[3]); b.c[2] = conj(s.c[0]); b.c[3] = conj(s.c[1]);
}

// ubar(p, lambda): outgoing fermion ("oxxxxx", nsf=+1);  vbar(p, lambda): incoming antifermion ("oxxxxx", nsf=-1)
template <typename T> MG_HD void ext_ubar(const T p[4], T m, int lambda, wf<T>& o)
{
    wf<T> u; ext_u(p, m, lambda, u); dirac_bar(u, o);
}
template <typename T> MG_HD void ext_vbar(const T p[4], T m, int lambda, wf<T>& o)
{
    wf<T> v; ext_v(p, m, lambda, v); dirac_bar(v, o);
}

// polarisation vector of a massless vector boson, helicity lambda = +-1 ("vxxxxx"):
//   eps = (0, (-lambda e1 - i e2)/sqrt2), e1 = (ct cf, ct sf, -st), e2 = (-sf, cf, 0);
//   outgoing particles take the complex conjugate.  pT = 0 (the beams): azimuth := 0.
template <typename T> MG_HD void ext_eps(const T p[4], int lambda, bool outgoing, wf<T>& e)
{
    const T pt2 = p[1] * p[1] + p[2] * p[2];
    const T pp = sqrt(pt2 + p[3] * p[3]);
    const T pt = sqrt(pt2);
    T ct, st, cf, sf;
    if (pt > pp * T(1e-7) * T(1e-7)) { ct = p[3] / pp; st = pt / pp; cf = p[1] / pt; sf = p[2] / pt; }
    else { ct = p[3] > T(0) ? T(1) : T(-1); st = T(0); cf = T(1); sf = T(0); }
    const T r = T(0.70710678118654752440);
    const T l = T(lambda);
    const T s = outgoing ? T(-1) : T(1);          // sign of the imaginary part
    e.c[0] = mk<T>(T(0), T(0));
    e.c[1] = mk<T>(-l * ct * cf * r, s * sf * r);
    e.c[2] = mk<T>(-l * ct * sf * r, -s * cf * r);
    e.c[3] = mk<T>(l * st * r, T(0));
}

// ------------------------------------------------------------------------------------------------
// slashed vector in the chiral representation:  Vslash = [[0, A], [B, 0]],
//   A = V0 - V.sigma = [[vm, -vl], [-vr, vp]],  B = V0 + V.sigma = [[vp, vl], [vr, vm]],
//   vp = V0 + V3, vm = V0 - V3, vr = V1 + i V2, vl = V1 - i V2
template <typename T>
struct slashed {
    cx<T> vp, vm, vr, vl;
};
template <typename T> MG_HD slashed<T> make_slashed(const wf<T>& v)
{
    slashed<T> s;
    s.vp = v.c[0] + v.c[3];
    s.vm = v.c[0] - v.c[3];
    s.vr = v.c[1] + times_i(v.c[2]);
    s.vl = v.c[1] - times_i(v.c[2]);
    return s;
}

// row spinor times Vslash
template <typename T> MG_HD void row_slash(const wf<T>& a, const slashed<T>& s, wf<T>& r)
{
    r.c[0] = cfma(a.c[3], s.vr, a.c[2] * s.vp);
    r.c[1] = cfma(a.c[3], s.vm, a.c[2] * s.vl);
    r.c[2] = cfms(a.c[1], s.vr, a.c[0] * s.vm);
    r.c[3] = cfms(a.c[0], s.vl, a.c[1] * s.vp);
}
// Vslash times column spinor
template <typename T> MG_HD void slash_col(const slashed<T>& s, const wf<T>& b, wf<T>& w)
{
    w.c[0] = cfms(s.vl, b.c[3], s.vm * b.c[2]);
    w.c[1] = cfms(s.vr, b.c[2], s.vp * b.c[3]);
    w.c[2] = cfma(s.vl, b.c[1], s.vp * b.c[0]);
    w.c[3] = cfma(s.vm, b.c[1], s.vr * b.c[0]);
}

// FFV1_0: amplitude  psibar Vslash psi
template <typename T> MG_HD cx<T> ffv_0(const wf<T>& fo, const wf<T>& v, const wf<T>& fi)
{
    wf<T> r;
    row_slash(fo, make_slashed(v), r);
    return r.c[0] * fi.c[0] + r.c[1] * fi.c[1] + r.c[2] * fi.c[2] + r.c[3] * fi.c[3];
}

// inverse of the propagator denominator q^2 - m^2 + i m w
template <typename T> MG_HD cx<T> inv_prop(T q2, T m, T w)
{
    const T dr = q2 - m * m, di = m * w;
    const T n = T(1) / (dr * dr + di * di);
    return mk<T>(dr * n, -di * n);
}

// FFV1_2-like: off-shell row spinor  psibar' = psibar Vslash (qslash + m) / (q^2 - m^2 + i m w),
// q = momentum along the fermion arrow (real)
template <typename T> MG_HD void ffv_l(const wf<T>& fo, const wf<T>& v, p4<T> q, T m, cx<T> invd, wf<T>& out)
{
    wf<T> r;
    row_slash(fo, make_slashed(v), r);
    const T qp = q.e + q.z, qm = q.e - q.z;
    const cx<T> qr = mk<T>(q.x, q.y), ql = mk<T>(q.x, -q.y);
    wf<T> t;
    t.c[0] = m * r.c[0] + qp * r.c[2] + r.c[3] * qr;
    t.c[1] = m * r.c[1] + r.c[2] * ql + qm * r.c[3];
    t.c[2] = qm * r.c[0] - r.c[1] * qr + m * r.c[2];
    t.c[3] = qp * r.c[1] - r.c[0] * ql + m * r.c[3];
    for (int i = 0; i < 4; i++) out.c[i] = t.c[i] * invd;
}

// FFV1_1-like: off-shell column spinor  psi' = (qslash + m) Vslash psi / (q^2 - m^2 + i m w)
template <typename T> MG_HD void ffv_r(const wf<T>& v, const wf<T>& fi, p4<T> q, T m, cx<T> invd, wf<T>& out)
{
    wf<T> w;
    slash_col(make_slashed(v), fi, w);
    const T qp = q.e + q.z, qm = q.e - q.z;
    const cx<T> qr = mk<T>(q.x, q.y), ql = mk<T>(q.x, -q.y);
    wf<T> t;
    t.c[0] = m * w.c[0] + qm * w.c[2] - ql * w.c[3];
    t.c[1] = m * w.c[1] - qr * w.c[2] + qp * w.c[3];
    t.c[2] = qp * w.c[0] + ql * w.c[1] + m * w.c[2];
    t.c[3] = qr * w.c[0] + qm * w.c[1] + m * w.c[3];
    for (int i = 0; i < 4; i++) out.c[i] = t.c[i] * invd;
}

// FFV1P0_3-like: off-shell vector  J^mu = psibar gamma^mu psi / K^2
template <typename T> MG_HD void ffv_p(const wf<T>& a, const wf<T>& b, T invk2, wf<T>& out)
{
    const cx<T> t02 = a.c[0] * b.c[2], t13 = a.c[1] * b.c[3], t20 = a.c[2] * b.c[0], t31 = a.c[3] * b.c[1];
    const cx<T> t03 = a.c[0] * b.c[3], t12 = a.c[1] * b.c[2], t21 = a.c[2] * b.c[1], t30 = a.c[3] * b.c[0];
    out.c[0] = invk2 * (t02 + t13 + t20 + t31);
    out.c[1] = invk2 * (t03 + t12 - t21 - t30);
    out.c[2] = invk2 * times_i((t12 - t03) + (t21 - t30));
    out.c[3] = invk2 * (t02 - t13 - t20 + t31);
}

// psibar gamma^mu psi without the propagator factor (raw vertex), FMA chains
template <typename T> MG_HD void ffv_p_raw(const wf<T>& a, const wf<T>& b, wf<T>& out)
{
    const cx<T> u = cfma(a.c[3], b.c[1], a.c[0] * b.c[2]);      // t02 + t31
    const cx<T> v = cfma(a.c[2], b.c[0], a.c[1] * b.c[3]);      // t13 + t20
    out.c[0] = u + v;
    out.c[1] = cfms(a.c[3], b.c[0], cfms(a.c[2], b.c[1], cfma(a.c[1], b.c[2], a.c[0] * b.c[3])));            // t03 + t12 - t21 - t30
    out.c[2] = times_i(cfms(a.c[3], b.c[0], cfms(a.c[0], b.c[3], cfma(a.c[2], b.c[1], a.c[1] * b.c[2]))));   // i (t12 + t21 - t03 - t30)
    out.c[3] = u - v;
}

// VVV1P0_1-like: off-shell gluon from two gluon currents, all momenta incoming:
//   J = [ (A.B)(kA-kB) + ((2kB+kA).A) B - ((2kA+kB).B) A ] / K^2,  K = kA + kB
template <typename T> MG_HD void v3_off(const wf<T>& A, p4<T> kA, const wf<T>& B, p4<T> kB, T invk2, wf<T>& out)
{
    const cx<T> ab = invk2 * dot(A, B);                 // 1/K^2 folded into the three scalar factors
    p4<T> ea = { T(2) * kB.e + kA.e, T(2) * kB.x + kA.x, T(2) * kB.y + kA.y, T(2) * kB.z + kA.z };
    p4<T> eb = { T(2) * kA.e + kB.e, T(2) * kA.x + kB.x, T(2) * kA.y + kB.y, T(2) * kA.z + kB.z };
    const cx<T> xa = invk2 * dot(ea, A), xb = invk2 * dot(eb, B);
    const p4<T> d = kA - kB;
    const T dd[4] = { d.e, d.x, d.y, d.z };
    for (int mu = 0; mu < 4; mu++) out.c[mu] = cfms(xb, A.c[mu], cfma(xa, B.c[mu], dd[mu] * ab));
}
// the same without the propagator factor (raw vertex)
template <typename T> MG_HD void v3_raw(const wf<T>& A, p4<T> kA, const wf<T>& B, p4<T> kB, wf<T>& out)
{
    const cx<T> ab = dot(A, B);
    p4<T> ea = { T(2) * kB.e + kA.e, T(2) * kB.x + kA.x, T(2) * kB.y + kA.y, T(2) * kB.z + kA.z };
    p4<T> eb = { T(2) * kA.e + kB.e, T(2) * kA.x + kB.x, T(2) * kA.y + kB.y, T(2) * kA.z + kB.z };
    const cx<T> xa = dot(ea, A), xb = dot(eb, B);
    const p4<T> d = kA - kB;
    const T dd[4] = { d.e, d.x, d.y, d.z };
    for (int mu = 0; mu < 4; mu++) out.c[mu] = cfms(xb, A.c[mu], cfma(xa, B.c[mu], dd[mu] * ab));
}

// VVVV1/3/4P0_1-like: one colour/Lorentz term of the four-gluon vertex, (x y | z out):
//   J = [ (X.Z) Y - (Y.Z) X ] / K^2
template <typename T> MG_HD void v4_off(const wf<T>& X, const wf<T>& Y, const wf<T>& Z, T invk2, wf<T>& out)
{
    const cx<T> xz = invk2 * dot(X, Z), yz = invk2 * dot(Y, Z);
    for (int mu = 0; mu < 4; mu++) out.c[mu] = cfms(yz, X.c[mu], xz * Y.c[mu]);
}
template <typename T> MG_HD void v4_raw(const wf<T>& X, const wf<T>& Y, const wf<T>& Z, wf<T>& out)
{
    const cx<T> xz = dot(X, Z), yz = dot(Y, Z);
    for (int mu = 0; mu < 4; mu++) out.c[mu] = cfms(yz, X.c[mu], xz * Y.c[mu]);
}

// VVV1_0: (A.B)((kA-kB).C) + (B.C)((kB-kC).A) + (C.A)((kC-kA).B), all momenta incoming
template <typename T> MG_HD cx<T> vvv_0(const wf<T>& A, p4<T> kA, const wf<T>& B, p4<T> kB, const wf<T>& C, p4<T> kC)
{
    return dot(A, B) * dot(kA - kB, C) + dot(B, C) * dot(kB - kC, A) + dot(C, A) * dot(kC - kA, B);
}

// VVVV_0 term (x y | z w): (X.Z)(Y.W) - (X.W)(Y.Z)
template <typename T> MG_HD cx<T> vvvv_0(const wf<T>& X, const wf<T>& Y, const wf<T>& Z, const wf<T>& W)
{
    return dot(X, Z) * dot(Y, W) - dot(X, W) * dot(Y, Z);
}

// chiral vector couplings for e+e- -> mu+mu- (FFV2/FFV4-like): psibar gamma^mu (gL PL + gR PR) psi
//   PL picks the upper two components of the column spinor (chiral representation), PR the lower two
template <typename T> MG_HD void ffv_lr_current(const wf<T>& a, const wf<T>& b, T gl, T gr, wf<T>& out)
{
    // gamma^mu PL psi couples row components 2,3 (sigma-bar block) to column 0,1; PR: row 0,1 to column 2,3
    const cx<T> t02 = a.c[0] * b.c[2], t13 = a.c[1] * b.c[3], t20 = a.c[2] * b.c[0], t31 = a.c[3] * b.c[1];
    const cx<T> t03 = a.c[0] * b.c[3], t12 = a.c[1] * b.c[2], t21 = a.c[2] * b.c[1], t30 = a.c[3] * b.c[0];
    out.c[0] = gr * (t02 + t13) + gl * (t20 + t31);
    out.c[1] = gr * (t03 + t12) - gl * (t21 + t30);
    out.c[2] = times_i(gr * (t12 - t03) + gl * (t21 - t30));
    out.c[3] = gr * (t02 - t13) - gl * (t20 - t31);
}

}  // namespace mg
