// ============================================================================
// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product.
//
// Plain, slow, fp64 statement of the improved staggered (asqtad) path of
// arXiv:1109.2935: the matrix M^IS of PAPER.md:114-122 (Sec. 2.3, Eq. 3) acting on
// 3-component colour vectors with a fat (one-hop) and a long (three-hop) gauge
// field, and the shifted systems (M^dag M + sigma_i) x_i = b of PAPER.md:130-134
// (Sec. 3.1, Eq. 4).  SURVEY.md 8(f) NEXT-3.  Shares no code with the CUDA path.
//
// Form: full lattice, lexicographic AoS, complex<double>:
//   site = x + X*(y + Y*(z + Z*t));  chi[site][colour];
//   fat[mu][site][row][col], lng[mu][site][row][col]  (general 3x3 complex: the fat
//   links are sums of paths, not unitary; both are INPUTS, "precalculated before the
//   application of M").
//
// Readings (the paper is silent or garbled; R13-R15):
//   R13 Eq. 3 as printed has the same sign on forward and backward hops and no staggered
//       phases, which contradicts "the staggered fermion matrix is anti-Hermitian"
//       (PAPER.md:130).  Reading (the asqtad operator of ref. [8]):
//         (D chi)(x) = sum_mu eta_mu(x) [ fat_mu(x) chi(x+mu) - fat_mu(x-mu)^dag chi(x-mu)
//                                       + lng_mu(x) chi(x+3mu) - lng_mu(x-3mu)^dag chi(x-3mu) ],
//         eta_x = 1, eta_y = (-1)^x, eta_z = (-1)^(x+y), eta_t = (-1)^(x+y+z),
//       path coefficients (c1, c3 = Naik) are part of the given links.  D is anti-Hermitian.
//   R14 M = -1/2 D + m (Eq. 3 as printed);  M^dag M = m^2 - D^2/4 couples only sites of the
//       same parity ("the even and odd lattices are decoupled").
//   R15 boundary: per direction +1 / -1; the sign multiplies every hop that wraps (a 3-hop
//       wraps when x_mu + 3 >= L_mu, resp. x_mu - 3 < 0).
//   Multi-shift CG is HOW the solutions are obtained; WHAT is computed is
//   x_i = (M^dag M + sigma_i)^-1 b, so the oracle solves every shift on its own with plain CG.
//
// Pins (tests/test_oracle_staggered.py): D anti-Hermitian; D couples opposite parities only;
// free field: M^dag M e^{ipx} = [m^2 + sum_mu (c1 sin p_mu + c3 sin 3p_mu)^2] e^{ipx}; gauge
// covariance; dense LU of (M^dag M + sigma) on 4^4; boundary signs through the closed form
// with half-integer momenta.
// ============================================================================
#include <complex>
#include <vector>
#include <cmath>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

namespace {

struct Lat {
  int L[4], bc[4];
  long V;
  Lat(const int* dims, const int* b) {
    V = 1;
    for (int m = 0; m < 4; ++m) { L[m] = dims[m]; bc[m] = b ? b[m] : 1; V *= dims[m]; }
  }
  void coords(long s, int* c) const { for (int m = 0; m < 4; ++m) { c[m] = (int)(s % L[m]); s /= L[m]; } }
  long site(const int* c) const { return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3])); }
};

// eta_mu(x) of R13
inline double eta(int mu, const int* c) {
  int e = 0;
  for (int nu = 0; nu < mu; ++nu) e += c[nu];
  return (e & 1) ? -1.0 : 1.0;
}

// site reached from c by `step` (+-1, +-3) lattice units in direction mu, and the boundary sign (R15)
inline long hop(const Lat& lat, const int* c, int mu, int step, double* sign) {
  int d[4] = {c[0], c[1], c[2], c[3]};
  int v = c[mu] + step;
  *sign = 1.0;
  if (v >= lat.L[mu] || v < 0) *sign = (double)lat.bc[mu];
  v %= lat.L[mu];
  if (v < 0) v += lat.L[mu];
  d[mu] = v;
  return lat.site(d);
}

// out = D in  (R13)
void stag_dslash(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const Lat& lat) {
#pragma omp parallel for if(lat.V >= 2048) schedule(static)
  for (long s = 0; s < lat.V; ++s) {
    int c[4];
    lat.coords(s, c);
    cplx acc[3] = {0, 0, 0};
    for (int mu = 0; mu < 4; ++mu) {
      const double e = eta(mu, c);
      for (int kind = 0; kind < 2; ++kind) {          // 0: fat, one hop; 1: long, three hops
        const cplx* links = kind ? lng : fat;
        const int step = kind ? 3 : 1;
        double sf, sb;
        const long xf = hop(lat, c, mu, +step, &sf), xb = hop(lat, c, mu, -step, &sb);
        const cplx* Uf = links + ((long)mu * lat.V + s) * 9;      // link at x
        const cplx* Ub = links + ((long)mu * lat.V + xb) * 9;     // link at x - step*mu
        for (int r = 0; r < 3; ++r) {
          cplx f = 0, b = 0;
          for (int k = 0; k < 3; ++k) {
            f += Uf[3 * r + k] * in[xf * 3 + k];
            b += std::conj(Ub[3 * k + r]) * in[xb * 3 + k];
          }
          acc[r] += e * (sf * f - sb * b);
        }
      }
    }
    for (int r = 0; r < 3; ++r) out[s * 3 + r] = acc[r];
  }
}

// out = M in = -1/2 D in + m in ;  dagger: M^dag = +1/2 D + m   (R14, D anti-Hermitian)
void stag_M(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const Lat& lat, double mass, int dagger) {
  stag_dslash(out, in, fat, lng, lat);
  const double h = dagger ? 0.5 : -0.5;
  const long n = lat.V * 3;
#pragma omp parallel for if(n >= 16384) schedule(static)
  for (long i = 0; i < n; ++i) out[i] = h * out[i] + mass * in[i];
}

// out = (M^dag M + sigma) in, written as the two applications it is
void stag_MdagM(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const Lat& lat, double mass, double sigma) {
  const long n = lat.V * 3;
  std::vector<cplx> t(n);
  stag_M(t.data(), in, fat, lng, lat, mass, 0);
  stag_M(out, t.data(), fat, lng, lat, mass, 1);
#pragma omp parallel for if(n >= 16384) schedule(static)
  for (long i = 0; i < n; ++i) out[i] += sigma * in[i];
}

double norm2(const cplx* a, long n) {
  double s = 0;
#pragma omp parallel for if(n >= 16384) reduction(+:s) schedule(static)
  for (long i = 0; i < n; ++i) s += std::norm(a[i]);
  return s;
}
double rdot(const cplx* a, const cplx* b, long n) {       // Re <a,b>
  double s = 0;
#pragma omp parallel for if(n >= 16384) reduction(+:s) schedule(static)
  for (long i = 0; i < n; ++i) s += (std::conj(a[i]) * b[i]).real();
  return s;
}

}  // namespace

extern "C" {

void ors_dslash(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const int* dims, const int* bc) {
  Lat lat(dims, bc);
  stag_dslash(out, in, fat, lng, lat);
}

void ors_M(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const int* dims, const int* bc, double mass, int dagger) {
  Lat lat(dims, bc);
  stag_M(out, in, fat, lng, lat, mass, dagger);
}

void ors_MdagM(cplx* out, const cplx* in, const cplx* fat, const cplx* lng, const int* dims, const int* bc, double mass, double sigma) {
  Lat lat(dims, bc);
  stag_MdagM(out, in, fat, lng, lat, mass, sigma);
}

// Plain CG (Hestenes-Stiefel, ref. [9]) on the Hermitian positive definite (M^dag M + sigma) x = b from x = 0.
// Stops when ||r|| <= tol * ||b||.  Returns 0, or 1 if maxit was reached.
int ors_cg(cplx* x, const cplx* b, const cplx* fat, const cplx* lng, const int* dims, const int* bc,
           double mass, double sigma, double tol, int maxit, int* iters, double* rel_res) {
  Lat lat(dims, bc);
  const long n = lat.V * 3;
  std::vector<cplx> r(b, b + n), p(b, b + n), Ap(n);
  for (long i = 0; i < n; ++i) x[i] = 0;
  const double bn = std::sqrt(norm2(b, n));
  double rr = norm2(r.data(), n);
  int it = 0, status = 0;
  while (std::sqrt(rr) > tol * bn) {
    if (it >= maxit) { status = 1; break; }
    stag_MdagM(Ap.data(), p.data(), fat, lng, lat, mass, sigma);
    const double alpha = rr / rdot(p.data(), Ap.data(), n);
    for (long i = 0; i < n; ++i) { x[i] += alpha * p[i]; r[i] -= alpha * Ap[i]; }
    const double rr1 = norm2(r.data(), n);
    const double beta = rr1 / rr;
    for (long i = 0; i < n; ++i) p[i] = r[i] + beta * p[i];
    rr = rr1;
    ++it;
  }
  // true residual
  stag_MdagM(Ap.data(), x, fat, lng, lat, mass, sigma);
  double d = 0;
  for (long i = 0; i < n; ++i) d += std::norm(b[i] - Ap[i]);
  *iters = it;
  *rel_res = bn > 0 ? std::sqrt(d) / bn : 0.0;
  return status;
}

}  // extern "C"
