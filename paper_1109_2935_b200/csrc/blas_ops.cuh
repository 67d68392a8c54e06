// blas_ops.cuh -- the fused BLAS-1 passes of the solvers:
// BiCGstab (recurrences restated in DESIGN.md "BiCGstab"), GCR (Algorithm 1,
// PAPER.md:260-292) and the per-block MR update of the Schwarz preconditioner.
#pragma once
#include "blas.cuh"

namespace lq {

struct NoCoef {};

// ---- generic ----------------------------------------------------------------------------------
struct OpZero {            // v0 = 0
  static constexpr int NV = 0, READ = 0, WRITE = 1;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R*, R*, R*, R*, double*) {
#pragma unroll
    for (int k = 0; k < 24; ++k) v0[k] = 0;
  }
  LQ_DEV static void finalize(const double*, const BlasArgs&, int) {}
};

struct OpNorm2 {           // S_OUT = ||v0||^2
  static constexpr int NV = 1, READ = 1, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R*, R*, R*, R*, double* red) { site_norm2(v0, red[0]); }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { a.S[S_OUT + a.i0] = s[0]; }
};

struct OpCdot {            // S_OUT..+1 = <v0,v1>, S_OUT+2 = ||v1||^2
  static constexpr int NV = 3, READ = 3, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R* v1, R*, R*, R*, double* red) {
    site_cdot(v0, v1, red[0], red[1]);
    site_norm2(v1, red[2]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    a.S[S_OUT] = s[0]; a.S[S_OUT + 1] = s[1]; a.S[S_OUT + 2] = s[2];
  }
};

struct OpAxpyNorm {        // v1 += c0*v0 ; S_OUT = ||v1||^2     (axpy+norm)
  static constexpr int NV = 1, READ = 3, WRITE = 2;
  struct Coef { double a; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.a = a.c[0]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* v0, R* v1, R*, R*, R*, double* red) {
    const R al = (R)c.a;
#pragma unroll
    for (int k = 0; k < 24; ++k) v1[k] += al * v0[k];
    site_norm2(v1, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { a.S[S_OUT] = s[0]; }
};

struct OpXmyNorm {         // v1 = v0 - v1 ; S_OUT = ||v1||^2      (r = b - M x)
  static constexpr int NV = 1, READ = 3, WRITE = 2;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R* v1, R*, R*, R*, double* red) {
#pragma unroll
    for (int k = 0; k < 24; ++k) v1[k] = v0[k] - v1[k];
    site_norm2(v1, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { a.S[S_OUT] = s[0]; }
};

// ---- BiCGstab -----------------------------------------------------------------------------------
// Device scalars: rho, rho_old, alpha, omega, beta (complex), rr.
struct OpBicgInit {        // v0 = rtilde, v1 = r : rho = <rt,r>, rho_old = alpha = omega = 1, beta = rho; rr = ||r||^2
  static constexpr int NV = 3, READ = 3, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R* v1, R*, R*, R*, double* red) {
    site_cdot(v0, v1, red[0], red[1]);
    site_norm2(v1, red[2]);
  }
  // i0 == 0: fresh start (rho_old = alpha = omega = 1, p = v = 0 so beta is irrelevant but finite)
  // i0 == 1: after a reliable update: r replaced; rho_old, alpha, omega kept; recompute rho, beta
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    if (a.i0 == 0) {
      S[S_RHO_OLD] = 1; S[S_RHO_OLD + 1] = 0; S[S_ALPHA] = 1; S[S_ALPHA + 1] = 0;
      S[S_OMEGA] = 1; S[S_OMEGA + 1] = 0; S[S_FLAG] = 0;
    }
    S[S_RHO] = s[0]; S[S_RHO + 1] = s[1];
    const cd rho = {s[0], s[1]}, rho_old = {S[S_RHO_OLD], S[S_RHO_OLD + 1]};
    const cd al = {S[S_ALPHA], S[S_ALPHA + 1]}, om = {S[S_OMEGA], S[S_OMEGA + 1]};
    const cd beta = cd_mul(cd_div(rho, rho_old), cd_div(al, om));
    S[S_BETA] = beta.re; S[S_BETA + 1] = beta.im;
    S[S_RR] = s[2];
  }
};

struct OpBicgP {           // v0 = p, v1 = r, v2 = v :  p = r + beta (p - omega v)
  static constexpr int NV = 0, READ = 7, WRITE = 1;
  struct Coef { double br, bi, wr, wi; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) {
    c.br = a.S[S_BETA]; c.bi = a.S[S_BETA + 1]; c.wr = a.S[S_OMEGA]; c.wi = a.S[S_OMEGA + 1];
  }
  template <typename R> LQ_DEV static void site(const Coef& c, R* p, R* r, R* v, R*, R*, double*) {
    const R br = (R)c.br, bi = (R)c.bi, wr = (R)c.wr, wi = (R)c.wi;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
      const R tr = p[2 * k] - (wr * v[2 * k] - wi * v[2 * k + 1]);
      const R ti = p[2 * k + 1] - (wr * v[2 * k + 1] + wi * v[2 * k]);
      p[2 * k] = r[2 * k] + br * tr - bi * ti;
      p[2 * k + 1] = r[2 * k + 1] + br * ti + bi * tr;
    }
  }
  LQ_DEV static void finalize(const double*, const BlasArgs&, int) {}
};

struct OpBicgAlpha {       // v0 = rtilde, v1 = v : alpha = rho / <rt,v>
  static constexpr int NV = 2, READ = 3, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* v0, R* v1, R*, R*, R*, double* red) { site_cdot(v0, v1, red[0], red[1]); }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    S[S_RTV] = s[0]; S[S_RTV + 1] = s[1];
    const double d = s[0] * s[0] + s[1] * s[1];
    if (!(d > 0.0)) { S[S_FLAG] = 1; S[S_ALPHA] = 0; S[S_ALPHA + 1] = 0; return; }
    const cd al = cd_div(cd{S[S_RHO], S[S_RHO + 1]}, cd{s[0], s[1]});
    S[S_ALPHA] = al.re; S[S_ALPHA + 1] = al.im;
  }
};

struct OpBicgS {           // v0 = r (becomes s), v1 = v : s = r - alpha v
  static constexpr int NV = 0, READ = 3, WRITE = 1;
  struct Coef { double ar, ai; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.ar = a.S[S_ALPHA]; c.ai = a.S[S_ALPHA + 1]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* r, R* v, R*, R*, R*, double*) {
    site_caxpy<R>((R)(-c.ar), (R)(-c.ai), v, r);
  }
  LQ_DEV static void finalize(const double*, const BlasArgs&, int) {}
};

struct OpBicgOmega {       // v0 = t, v1 = s : omega = <t,s>/<t,t>
  static constexpr int NV = 3, READ = 3, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* t, R* s, R*, R*, R*, double* red) {
    site_cdot(t, s, red[0], red[1]);
    site_norm2(t, red[2]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    S[S_TS] = s[0]; S[S_TS + 1] = s[1]; S[S_TT] = s[2];
    if (!(s[2] > 0.0)) { S[S_OMEGA] = 0; S[S_OMEGA + 1] = 0; S[S_FLAG] = 2; return; }
    S[S_OMEGA] = s[0] / s[2]; S[S_OMEGA + 1] = s[1] / s[2];
  }
};

struct OpBicgXR {          // v0 = x, v1 = p, v2 = s->r, v3 = t, v4 = rtilde
  // x += alpha p + omega s ; r = s - omega t ; rho' = <rt,r> ; rr = ||r||^2 ; beta = (rho'/rho)(alpha/omega)
  static constexpr int NV = 3, READ = 31, WRITE = 5;
  struct Coef { double ar, ai, wr, wi; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) {
    c.ar = a.S[S_ALPHA]; c.ai = a.S[S_ALPHA + 1]; c.wr = a.S[S_OMEGA]; c.wi = a.S[S_OMEGA + 1];
  }
  template <typename R> LQ_DEV static void site(const Coef& c, R* x, R* p, R* s, R* t, R* rt, double* red) {
    site_caxpy<R>((R)c.ar, (R)c.ai, p, x);
    site_caxpy<R>((R)c.wr, (R)c.wi, s, x);
    site_caxpy<R>((R)(-c.wr), (R)(-c.wi), t, s);
    site_cdot(rt, s, red[0], red[1]);
    site_norm2(s, red[2]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { update(s, a); publish(a); }
  LQ_DEV static void update(const double* s, const BlasArgs& a) {
    double* S = a.S;
    const cd rho_old = {S[S_RHO], S[S_RHO + 1]};
    S[S_RHO_OLD] = rho_old.re; S[S_RHO_OLD + 1] = rho_old.im;
    S[S_RHO] = s[0]; S[S_RHO + 1] = s[1];
    S[S_RR] = s[2];
    const cd al = {S[S_ALPHA], S[S_ALPHA + 1]}, om = {S[S_OMEGA], S[S_OMEGA + 1]};
    const double d1 = rho_old.re * rho_old.re + rho_old.im * rho_old.im, d2 = om.re * om.re + om.im * om.im;
    if (!(d1 > 0.0) || !(d2 > 0.0)) { if (s[2] > 0.0) S[S_FLAG] = 3; S[S_BETA] = 0; S[S_BETA + 1] = 0; return; }
    const cd beta = cd_mul(cd_div(cd{s[0], s[1]}, rho_old), cd_div(al, om));
    S[S_BETA] = beta.re; S[S_BETA + 1] = beta.im;
  }
  // publish (||r||^2, breakdown flag) of iteration i0 to the host: values first, then the iteration number the host polls
  LQ_DEV static void publish(const BlasArgs& a) {
    if (!a.hmirror) return;
    volatile double* h = a.hmirror + 4 * (a.i0 & 1);
    h[0] = a.S[S_RR]; h[1] = a.S[S_FLAG];
    __threadfence_system();
    h[2] = (double)a.i0;
  }
};

// ---- CGNR (CG on the normal equations Mhat^dag Mhat x = Mhat^dag bhat) -------------
// Device scalars: zz = <z,z> in S_RHO, alpha in S_ALPHA, beta in S_BETA (all real), rr in S_RR.
struct OpCgInit {          // v0 = z, v1 = p : p = z ; zz = ||z||^2          (start, i0 = 0)
  //                          i0 = 1 (after a reliable update): beta = ||z||^2 / zz_old ; p = z + beta p is done by OpCgP
  //                          i0 = 2: the same when S_RHO and beta were already advanced by OpCgXRB (CGNE, plain CG)
  static constexpr int NV = 1, READ = 1, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* z, R*, R*, R*, R*, double* red) { site_norm2(z, red[0]); }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    if (a.i0 == 0) { S[S_BETA] = 0; S[S_FLAG] = 0; }
    else if (a.i0 == 1) S[S_BETA] = (S[S_RHO] > 0.0) ? s[0] / S[S_RHO] : 0.0;
    else S[S_BETA] *= (S[S_RHO] > 0.0) ? s[0] / S[S_RHO] : 0.0;     // i0 == 2: the residual whose norm gave beta (OpCgXRB:
    S[S_RHO] = s[0];                                                  // beta = rr'/rr, S_RHO = rr') was replaced: beta = rr_new/rr
  }
};

struct OpCgP {             // v0 = p, v1 = z : p = z + beta p
  static constexpr int NV = 0, READ = 3, WRITE = 1;
  struct Coef { double b; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.b = a.S[S_BETA]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* p, R* z, R*, R*, R*, double*) {
    const R b = (R)c.b;
#pragma unroll
    for (int k = 0; k < 24; ++k) p[k] = fma_(b, p[k], z[k]);
  }
  LQ_DEV static void finalize(const double*, const BlasArgs&, int) {}
};

struct OpCgAlpha {         // v0 = w = Mhat p : alpha = zz / ||w||^2
  static constexpr int NV = 1, READ = 1, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* w, R*, R*, R*, R*, double* red) { site_norm2(w, red[0]); }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    if (!(s[0] > 0.0)) { S[S_FLAG] = 1; S[S_ALPHA] = 0; return; }
    S[S_ALPHA] = S[S_RHO] / s[0];
  }
};

struct OpCgXR {            // v0 = x, v1 = p, v2 = r, v3 = w : x += alpha p ; r -= alpha w ; rr = ||r||^2
  static constexpr int NV = 1, READ = 15, WRITE = 5;
  struct Coef { double a; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.a = a.S[S_ALPHA]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* x, R* p, R* r, R* w, R*, double* red) {
    const R al = (R)c.a;
#pragma unroll
    for (int k = 0; k < 24; ++k) { x[k] = fma_(al, p[k], x[k]); r[k] = fma_(-al, w[k], r[k]); }
    site_norm2(r, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { a.S[S_RR] = s[0]; }
};

// ---- CG on a Hermitian positive definite operator, and its multi-shift form (staggered path) -----
// (M^dag M + sigma_i) x_i = b, Eq. 4, solver of PAPER.md:296.  Scalars: rr = <r,r> in
// S_RHO, alpha in S_ALPHA, beta in S_BETA (real).  Multi-shift state (Jegerlehner's recurrences; the
// shifted residuals are zeta_i r): per shift i at S_MS + LQ_MS_STRIDE*i: zeta, zeta_old, alpha_i, beta_i,
// sigma_i - sigma_0; S_MS_AOLD, S_MS_BOLD the previous alpha, beta of the base system; S_MS_N shifts.
enum { S_MS = S_GCR_BETA, LQ_MS_STRIDE = 8, LQ_MS_MAX = 32, S_MS_AOLD = S_MS + LQ_MS_STRIDE * LQ_MS_MAX, S_MS_BOLD, S_MS_N };
static_assert(S_MS_N < S_GCR_GAMMAS, "multi-shift scalars must fit the GCR beta region they reuse");

struct OpCgPAp {           // v0 = p, v1 = A p : alpha = rr / Re<p, A p>
  static constexpr int NV = 1, READ = 3, WRITE = 0;
  typedef NoCoef Coef;
  LQ_DEV static void prepare(Coef&, const BlasArgs&, int) {}
  template <typename R> LQ_DEV static void site(const Coef&, R* p, R* ap, R*, R*, R*, double* red) {
    R s = 0;
#pragma unroll
    for (int k = 0; k < 24; ++k) s = fma_(p[k], ap[k], s);
    red[0] += (double)s;
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    if (!(s[0] > 0.0)) { S[S_FLAG] = 1; S[S_ALPHA] = 0; return; }
    S[S_ALPHA] = S[S_RHO] / s[0];
  }
};

struct OpCgXRB {           // v0 = x, v1 = p, v2 = r, v3 = A p : x += alpha p ; r -= alpha A p ; rr' = ||r||^2 ; beta = rr'/rr
  static constexpr int NV = 1, READ = 15, WRITE = 5;
  struct Coef { double a; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.a = a.S[S_ALPHA]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* x, R* p, R* r, R* ap, R*, double* red) {
    const R al = (R)c.a;
#pragma unroll
    for (int k = 0; k < 24; ++k) { x[k] = fma_(al, p[k], x[k]); r[k] = fma_(-al, ap[k], r[k]); }
    site_norm2(r, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    S[S_BETA] = (S[S_RHO] > 0.0) ? s[0] / S[S_RHO] : 0.0;
    S[S_RHO] = s[0]; S[S_RR] = s[0];
  }
};

struct OpMsR {             // v0 = r, v1 = A p (base system): r -= alpha A p ; rr' ; beta ; all shifted scalars
  static constexpr int NV = 1, READ = 3, WRITE = 1;
  struct Coef { double a; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) { c.a = a.S[S_ALPHA]; }
  template <typename R> LQ_DEV static void site(const Coef& c, R* r, R* ap, R*, R*, R*, double* red) {
    const R al = (R)c.a;
#pragma unroll
    for (int k = 0; k < 24; ++k) r[k] = fma_(-al, ap[k], r[k]);
    site_norm2(r, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) {
    double* S = a.S;
    const double al = S[S_ALPHA], be = (S[S_RHO] > 0.0) ? s[0] / S[S_RHO] : 0.0;
    const double a_old = S[S_MS_AOLD], b_old = S[S_MS_BOLD];
    const int n = (int)S[S_MS_N];
    for (int i = 0; i < n; ++i) {
      double* m = S + S_MS + LQ_MS_STRIDE * i;
      const double z = m[0], zo = m[1], d = m[4];
      // zeta_{n+1} = zeta_n zeta_{n-1} a_{n-1} / ( a_n b_{n-1} (zeta_{n-1} - zeta_n) + zeta_{n-1} a_{n-1} (1 + d a_n) )
      const double den = al * b_old * (zo - z) + zo * a_old * (1.0 + d * al);
      const double zn = (den != 0.0) ? z * zo * a_old / den : 0.0;
      const double ratio = (z != 0.0) ? zn / z : 0.0;
      m[2] = al * ratio;                 // alpha_i of this step
      m[3] = be * ratio * ratio;         // beta_i
      m[1] = z; m[0] = zn;
    }
    S[S_MS_AOLD] = al; S[S_MS_BOLD] = be;
    S[S_BETA] = be; S[S_RHO] = s[0]; S[S_RR] = s[0];
  }
};

// ---- GCR (Algorithm 1) --------------------------------------------------------------------------
struct OpGcrScale {        // v0 = z_k, v1 = rhat : z_k /= gamma ; rhat -= alpha z_k ; rr = ||rhat||^2
  static constexpr int NV = 1, READ = 3, WRITE = 3;
  struct Coef { double ig, ar, ai; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int) {
    const double g = a.S[S_GCR_GAMMA];
    c.ig = g > 0.0 ? 1.0 / g : 0.0; c.ar = a.S[S_GCR_ALPHA]; c.ai = a.S[S_GCR_ALPHA + 1];
  }
  template <typename R> LQ_DEV static void site(const Coef& c, R* z, R* r, R*, R*, R*, double* red) {
    const R ig = (R)c.ig;
#pragma unroll
    for (int k = 0; k < 24; ++k) z[k] *= ig;
    site_caxpy<R>((R)(-c.ar), (R)(-c.ai), z, r);
    site_norm2(r, red[0]);
  }
  LQ_DEV static void finalize(const double* s, const BlasArgs& a, int) { a.S[S_RR] = s[0]; }
};

// ---- Schwarz / MR: one alpha per box ---------------------------------------------
// alpha_b = c0 * <w,rho>_b / <w,w>_b from the Dslash epilogue's per-warp partials: one CTA per box adds the box's
// nchunk partials in a fixed order (deterministic) and writes (re, im) of alpha_b.  A kernel of its own: summing the
// partials at the start of every CTA of the update pass (162 x 4 x 3 doubles per box at 12^3x24, read by 81 CTAs)
// was 80 us of its 350 us at config 5.
LQ_DEV void mr_alpha_box(const double* boxdots, int nchunk, int box, double c0, double* boxalpha) {
  __shared__ double sm[3 * (LQ_BLAS_BLOCK / 32)];
  double s[3] = {0, 0, 0};
  const double* d = boxdots + (long long)box * nchunk * 4;
  for (int i = threadIdx.x; i < nchunk; i += LQ_BLAS_BLOCK) {
    s[0] += __ldcg(d + 4 * i); s[1] += __ldcg(d + 4 * i + 1); s[2] += __ldcg(d + 4 * i + 2);
  }
  cta_reduce<3, LQ_BLAS_BLOCK>(s, sm);
  if (threadIdx.x == 0) {
    const double ww = s[2];
    boxalpha[2 * box] = (ww > 0.0) ? c0 * s[0] / ww : 0.0;
    boxalpha[2 * box + 1] = (ww > 0.0) ? c0 * s[1] / ww : 0.0;
  }
}

// v0 = x, v1 = rho, v2 = w:  x += alpha_b rho;  rho -= alpha_b w
template <bool FIRST, bool LASTSTEP>
struct OpMrUpdate {
  static constexpr int NV = 0, READ = (FIRST ? 0 : 1) | 2 | (LASTSTEP ? 0 : 4), WRITE = 1 | (LASTSTEP ? 0 : 2);
  struct Coef { double ar, ai; };
  LQ_DEV static void prepare(Coef& c, const BlasArgs& a, int box) {
    c.ar = __ldcg(a.boxalpha + 2 * box);
    c.ai = __ldcg(a.boxalpha + 2 * box + 1);
  }
  template <typename R> LQ_DEV static void site(const Coef& c, R* x, R* rho, R* w, R*, R*, double*) {
    if (FIRST) {
#pragma unroll
      for (int k = 0; k < 24; ++k) x[k] = 0;
    }
    site_caxpy<R>((R)c.ar, (R)c.ai, rho, x);
    if (!LASTSTEP) site_caxpy<R>((R)(-c.ar), (R)(-c.ai), w, rho);
  }
  LQ_DEV static void finalize(const double*, const BlasArgs&, int) {}
};

}  // namespace lq
