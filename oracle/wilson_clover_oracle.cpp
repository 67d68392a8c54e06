// ============================================================================
// CPU ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product.
//
// Plain, slow, fp64 statement of what the hot path of arXiv:1109.2935
// ("Scaling Lattice QCD beyond 100 GPUs", Babich et al., SC11) computes:
// the Wilson-clover Dirac operator (Sec. 2.2, Eq. 2), its
// even-odd (Schur complement) preconditioned form (Sec. 3.1),
// BiCGstab, the non-overlapping additive-Schwarz preconditioner
// with a fixed number of MR steps (PAPER.md:146, Sec. 3.2; :250, Sec. 8.1) and
// the GCR-DD solver (Algorithm 1); plus the multiplicative (SAP) and the overlapping (restricted
// additive) Schwarz variants the paper names.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this file.  It shares no code, header, table
// or constant generator with the CUDA path (paper_1109_2935_b200/csrc).
//
// Form (deliberately different from the GPU path):
//   * full lattice, lexicographic, array-of-structures, complex<double>:
//       site = x + X*(y + Y*(z + Z*t));  psi[site][spin][colour];
//       U[mu][site][row][col],  mu = 0:x 1:y 2:z 3:t,  U_mu(x) multiplies psi(x+mu)
//   * no checkerboard storage: parity operators are obtained by masking
//   * no gauge compression, no spin-projection trick: full 4x4 (1 -/+ gamma_mu)
//   * no blocking, fusion or reordering; OpenMP over the site loop only, and only from 2048 sites up
//     (on the 4^4 pin lattices the thread start-up of ~25,000 tiny calls dominated the CPU test time).
//
// Readings of the paper (it is silent on all of these):
//   R1  P^{+-mu} = 1 +- gamma_mu  (unnormalised; Eq. 2's -1/2 makes it a projector)
//   R2  gamma basis: DeGrand-Rossi chiral basis, gamma5 = diag(1,1,-1,-1)
//   R3  kappa normalisation: kappa = 1/(2(4+m)); M = A(kappa) - kappa*D,
//       A_x(kappa) = 1 + kappa*T_x   (2*kappa*M^WC of Eq. 2)
//   R4  clover term: four-leaf F_munu = (Q - Q^dag)/8, no trace subtraction,
//       T_x = c_sw * sum_{mu<nu} (i sigma_munu) (x) F_munu(x), sigma = (i/2)[g_mu,g_nu]
//   R5  boundary: per-direction +1 periodic / -1 antiperiodic sign on wrapping hops
//   R6  even-odd: asymmetric Schur complement  Mhat = A_pp - kappa^2 D A^-1 D
//   R7  Schwarz: Dirichlet = hops whose ends lie in different blocks are dropped;
//       K = n_MR minimum-residual steps on Mhat_D with one alpha per block
//   R8  Algorithm 1 as restated in DESIGN.md (hats restored, indentation restored)
//
// Parity pins (tests/test_oracle_*.py): gamma algebra; free-field plane waves
// (closed form M(p)); gamma5-hermiticity; gauge covariance; abelian constant-flux
// closed form of the clover term; c_sw=0 => A=1; dense LU on 2^4 and 4^4 for the
// even-odd algebra and both solvers; block-diagonality of Mhat_D; GCR identities.
// Unpinned (reported, never asserted): iteration counts, convergence history.
// ============================================================================
#include <complex>
#include <vector>
#include <cmath>
#include <cstring>
#include <cstdlib>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const cplx I_(0.0, 1.0);

namespace {

struct Lat {
  int L[4];
  long V;
  int bc[4];
  explicit Lat(const int* dims, const int* bc_) {
    V = 1;
    for (int m = 0; m < 4; ++m) { L[m] = dims[m]; V *= dims[m]; bc[m] = bc_ ? bc_[m] : 1; }
  }
  inline void coords(long s, int c[4]) const {
    c[0] = (int)(s % L[0]); s /= L[0];
    c[1] = (int)(s % L[1]); s /= L[1];
    c[2] = (int)(s % L[2]); s /= L[2];
    c[3] = (int)s;
  }
  inline long site(const int c[4]) const {
    return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3]));
  }
  // neighbour of c displaced by d (= +-1) in direction mu, periodic wrap
  inline long shifted(const int c[4], int mu, int d) const {
    int n[4] = {c[0], c[1], c[2], c[3]};
    n[mu] = (c[mu] + d + L[mu]) % L[mu];
    return site(n);
  }
  inline long shifted2(const int c[4], int mu, int dm, int nu, int dn) const {
    int n[4] = {c[0], c[1], c[2], c[3]};
    n[mu] = (c[mu] + dm + L[mu]) % L[mu];
    n[nu] = (n[nu] + dn + L[nu]) % L[nu];
    return site(n);
  }
  inline int parity(const int c[4]) const { return (c[0] + c[1] + c[2] + c[3]) & 1; }
};

// ---- gamma matrices: reading R2 (DeGrand-Rossi) -----------------------------
// gamma[mu][row][col]; gamma[4] = gamma5 = gx*gy*gz*gt.
struct Gamma {
  cplx g[5][4][4];
  Gamma() {
    std::memset((void*)g, 0, sizeof(g));
    const cplx i = I_;
    // gamma_x
    g[0][0][3] = i;   g[0][1][2] = i;   g[0][2][1] = -i;  g[0][3][0] = -i;
    // gamma_y
    g[1][0][3] = -1.; g[1][1][2] = 1.;  g[1][2][1] = 1.;  g[1][3][0] = -1.;
    // gamma_z
    g[2][0][2] = i;   g[2][1][3] = -i;  g[2][2][0] = -i;  g[2][3][1] = i;
    // gamma_t
    g[3][0][2] = 1.;  g[3][1][3] = 1.;  g[3][2][0] = 1.;  g[3][3][1] = 1.;
    cplx t1[4][4], t2[4][4];
    mul(g[0], g[1], t1); mul(t1, g[2], t2); mul(t2, g[3], g[4]);
  }
  static void mul(const cplx a[4][4], const cplx b[4][4], cplx c[4][4]) {
    for (int r = 0; r < 4; ++r) for (int s = 0; s < 4; ++s) {
      cplx acc = 0; for (int k = 0; k < 4; ++k) acc += a[r][k] * b[k][s]; c[r][s] = acc;
    }
  }
};
static const Gamma G;

inline void su3_mul(const cplx* a, const cplx* b, cplx* c) {        // c = a b
  for (int r = 0; r < 3; ++r) for (int s = 0; s < 3; ++s) {
    cplx acc = 0; for (int k = 0; k < 3; ++k) acc += a[3*r+k] * b[3*k+s]; c[3*r+s] = acc;
  }
}
inline void su3_dag(const cplx* a, cplx* c) {                         // c = a^dagger
  for (int r = 0; r < 3; ++r) for (int s = 0; s < 3; ++s) c[3*r+s] = std::conj(a[3*s+r]);
}

// block id of a site for the Schwarz decomposition; blk == nullptr -> one block
inline bool same_block(const int* blk, const int c[4], int mu, int d, const Lat& lat) {
  if (!blk) return true;
  if (blk[mu] >= lat.L[mu]) return true;           // direction not partitioned: wrap kept (R7)
  int n = c[mu] + d;
  if (n < 0 || n >= lat.L[mu]) return false;       // global wrap joins two different blocks
  return (n / blk[mu]) == (c[mu] / blk[mu]);
}

// ---- c.1  Dslash: the hopping part of Eq. 2 ---------------
// (D psi)(x) = sum_mu [ s+ (1 - g_mu) U_mu(x) psi(x+mu) + s- (1 + g_mu) U_mu(x-mu)^dag psi(x-mu) ]
// dagger: (1 -/+ g_mu) exchanged.  blk: Dirichlet cut (R7) or nullptr.
// dom: optional site mask (overlapping Schwarz domains, schwarz_ras below): a hop is kept only if both its ends are
// in the domain.
void dslash(cplx* out, const cplx* in, const cplx* U, const Lat& lat, int dagger, const int* blk,
            const unsigned char* dom = nullptr) {
  const long V = lat.V;
#pragma omp parallel for if(V >= 2048) schedule(static)
  for (long s = 0; s < V; ++s) {
    int c[4]; lat.coords(s, c);
    cplx acc[4][3];
    for (int a = 0; a < 4; ++a) for (int k = 0; k < 3; ++k) acc[a][k] = 0;
    for (int mu = 0; mu < 4; ++mu) {
      for (int dir = +1; dir >= -1; dir -= 2) {
        if (!same_block(blk, c, mu, dir, lat)) continue;
        const long n = lat.shifted(c, mu, dir);
        if (dom && !(dom[s] && dom[n])) continue;
        const bool wraps = (dir > 0) ? (c[mu] == lat.L[mu] - 1) : (c[mu] == 0);
        const double sgn = (wraps && lat.bc[mu] < 0) ? -1.0 : 1.0;
        // colour part: U_mu(x) psi(x+mu)  or  U_mu(x-mu)^dagger psi(x-mu)
        cplx W[9];
        if (dir > 0) std::memcpy((void*)W, (const void*)(U + ((long)mu * V + s) * 9), sizeof(W));
        else su3_dag(U + ((long)mu * V + n) * 9, W);
        cplx cp[4][3];
        for (int a = 0; a < 4; ++a) for (int r = 0; r < 3; ++r) {
          cplx t = 0; for (int k = 0; k < 3; ++k) t += W[3*r+k] * in[(n * 4 + a) * 3 + k];
          cp[a][r] = t;
        }
        // spin part: (1 - dir*g_mu) forward/backward as in Eq. 2; dagger flips the sign
        const double gs = (dagger ? +1.0 : -1.0) * dir;      // coefficient of gamma_mu
        for (int a = 0; a < 4; ++a) for (int r = 0; r < 3; ++r) {
          cplx t = cp[a][r];
          for (int b = 0; b < 4; ++b) t += gs * G.g[mu][a][b] * cp[b][r];
          acc[a][r] += sgn * t;
        }
      }
    }
    for (int a = 0; a < 4; ++a) for (int k = 0; k < 3; ++k) out[(s * 4 + a) * 3 + k] = acc[a][k];
  }
}

// ---- c.2  clover term (reading R4) -------------------------------------------
// T[site][12][12], row index = spin*3 + colour.
void clover_term(cplx* T, const cplx* U, const Lat& lat, double c_sw) {
  const long V = lat.V;
  // i*sigma_munu = i*(i/2)[g_mu,g_nu] = -(1/2)[g_mu,g_nu]
  cplx isig[4][4][4][4];
  for (int mu = 0; mu < 4; ++mu) for (int nu = 0; nu < 4; ++nu) {
    cplx ab[4][4], ba[4][4];
    Gamma::mul(G.g[mu], G.g[nu], ab); Gamma::mul(G.g[nu], G.g[mu], ba);
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b)
      isig[mu][nu][a][b] = I_ * (I_ / 2.0) * (ab[a][b] - ba[a][b]);
  }
#pragma omp parallel for if(V >= 2048) schedule(static)
  for (long s = 0; s < V; ++s) {
    int c[4]; lat.coords(s, c);
    cplx* Ts = T + s * 144;
    for (int i = 0; i < 144; ++i) Ts[i] = 0;
    for (int mu = 0; mu < 4; ++mu) for (int nu = mu + 1; nu < 4; ++nu) {
      auto Ul = [&](int d, long site) { return U + ((long)d * V + site) * 9; };
      const long x    = s;
      const long xpm  = lat.shifted(c, mu, +1);
      const long xpn  = lat.shifted(c, nu, +1);
      const long xmm  = lat.shifted(c, mu, -1);
      const long xmn  = lat.shifted(c, nu, -1);
      const long xmmpn = lat.shifted2(c, mu, -1, nu, +1);
      const long xmmmn = lat.shifted2(c, mu, -1, nu, -1);
      const long xpmmn = lat.shifted2(c, mu, +1, nu, -1);
      cplx Q[9], a[9], b[9], d1[9], d2[9], leaf[9];
      for (int i = 0; i < 9; ++i) Q[i] = 0;
      // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
      su3_mul(Ul(mu, x), Ul(nu, xpm), a); su3_dag(Ul(mu, xpn), d1); su3_dag(Ul(nu, x), d2);
      su3_mul(a, d1, b); su3_mul(b, d2, leaf); for (int i = 0; i < 9; ++i) Q[i] += leaf[i];
      // leaf 2: U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
      su3_dag(Ul(mu, xmmpn), d1); su3_dag(Ul(nu, xmm), d2);
      su3_mul(Ul(nu, x), d1, a); su3_mul(a, d2, b); su3_mul(b, Ul(mu, xmm), leaf);
      for (int i = 0; i < 9; ++i) Q[i] += leaf[i];
      // leaf 3: U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
      su3_dag(Ul(mu, xmm), d1); su3_dag(Ul(nu, xmmmn), d2);
      su3_mul(d1, d2, a); su3_mul(a, Ul(mu, xmmmn), b); su3_mul(b, Ul(nu, xmn), leaf);
      for (int i = 0; i < 9; ++i) Q[i] += leaf[i];
      // leaf 4: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
      su3_dag(Ul(nu, xmn), d1); su3_dag(Ul(mu, x), d2);
      su3_mul(d1, Ul(mu, xmn), a); su3_mul(a, Ul(nu, xpmmn), b); su3_mul(b, d2, leaf);
      for (int i = 0; i < 9; ++i) Q[i] += leaf[i];
      cplx Qd[9], F[9];
      su3_dag(Q, Qd);
      for (int i = 0; i < 9; ++i) F[i] = (Q[i] - Qd[i]) / 8.0;
      for (int sa = 0; sa < 4; ++sa) for (int sb = 0; sb < 4; ++sb) {
        const cplx w = c_sw * isig[mu][nu][sa][sb];
        if (w == cplx(0.0)) continue;
        for (int ca = 0; ca < 3; ++ca) for (int cb = 0; cb < 3; ++cb)
          Ts[(sa * 3 + ca) * 12 + (sb * 3 + cb)] += w * F[3 * ca + cb];
      }
    }
  }
}

// dense 12x12 solve  A y = rhs  by Gaussian elimination with partial pivoting
void solve12(const cplx* A, const cplx* rhs, cplx* y) {
  cplx a[12][13];
  for (int r = 0; r < 12; ++r) { for (int k = 0; k < 12; ++k) a[r][k] = A[12*r+k]; a[r][12] = rhs[r]; }
  for (int col = 0; col < 12; ++col) {
    int piv = col; double best = std::abs(a[col][col]);
    for (int r = col + 1; r < 12; ++r) if (std::abs(a[r][col]) > best) { best = std::abs(a[r][col]); piv = r; }
    if (piv != col) for (int k = 0; k < 13; ++k) std::swap(a[piv][k], a[col][k]);
    for (int r = col + 1; r < 12; ++r) {
      const cplx f = a[r][col] / a[col][col];
      for (int k = col; k < 13; ++k) a[r][k] -= f * a[col][k];
    }
  }
  for (int r = 11; r >= 0; --r) {
    cplx t = a[r][12];
    for (int k = r + 1; k < 12; ++k) t -= a[r][k] * y[k];
    y[r] = t / a[r][r];
  }
}

// out = A in or A^{-1} in with A = 1 + kappa*T  (R3); mask: -1 all sites, else only that parity
void clover_apply(cplx* out, const cplx* in, const cplx* T, const Lat& lat, double kappa, int inverse, int par) {
  const long V = lat.V;
#pragma omp parallel for if(V >= 2048) schedule(static)
  for (long s = 0; s < V; ++s) {
    int c[4]; lat.coords(s, c);
    if (par >= 0 && lat.parity(c) != par) { for (int i = 0; i < 12; ++i) out[s*12+i] = 0; continue; }
    cplx A[144];
    for (int r = 0; r < 12; ++r) for (int k = 0; k < 12; ++k)
      A[12*r+k] = (r == k ? 1.0 : 0.0) + kappa * T[s*144 + 12*r + k];
    if (!inverse) {
      for (int r = 0; r < 12; ++r) { cplx t = 0; for (int k = 0; k < 12; ++k) t += A[12*r+k] * in[s*12+k]; out[s*12+r] = t; }
    } else {
      cplx y[12]; solve12(A, in + s*12, y);
      for (int r = 0; r < 12; ++r) out[s*12+r] = y[r];
    }
  }
}

void mask_parity(cplx* v, const Lat& lat, int keep) {
#pragma omp parallel for if(lat.V >= 2048) schedule(static)
  for (long s = 0; s < lat.V; ++s) {
    int c[4]; lat.coords(s, c);
    if (lat.parity(c) != keep) for (int i = 0; i < 12; ++i) v[s*12+i] = 0;
  }
}

struct Op {                         // everything an operator application needs
  const cplx* U; const cplx* T; Lat lat; double kappa;
  const int* blk;                   // Schwarz block extents or nullptr
  int sym;                          // 0: asymmetric Schur complement (default), 1: symmetric form (c.5 "Optional")
  const unsigned char* dom = nullptr;   // site mask of one overlapping Schwarz domain (schwarz_ras) or nullptr
  Op(const cplx* U_, const cplx* T_, const int* dims, const int* bc, double k, const int* blk_, int sym_ = 0)
    : U(U_), T(T_), lat(dims, bc), kappa(k), blk(blk_), sym(sym_) {}
  long n() const { return lat.V * 12; }
};

// c.3  M = A - kappa D   (2*kappa times Eq. 2; reading R3)
void apply_M(cplx* out, const cplx* in, const Op& op, int dagger) {
  std::vector<cplx> d(op.n());
  dslash(d.data(), in, op.U, op.lat, dagger, op.blk, op.dom);
  clover_apply(out, in, op.T, op.lat, op.kappa, 0, -1);
  const long n = op.n();
#pragma omp parallel for if(n >= 16384) schedule(static)
  for (long i = 0; i < n; ++i) out[i] -= op.kappa * d[i];
}

// c.5  Mhat = A_pp - kappa^2 D_{p pbar} A_{pbar pbar}^{-1} D_{pbar p}   (reading R6), by masking.
// in/out are full-lattice arrays; only parity-p sites of `in` are read, the rest of out is 0.
// Symmetric form (same reference [11]):  Mhat_s = 1 - kappa^2 A_pp^-1 D A_pbar^-1 D = A_pp^-1 Mhat,
// Mhat_s^dag = 1 - kappa^2 D^dag A_pbar^-1 D^dag A_pp^-1 (A is Hermitian).
void apply_matpc_sym(cplx* out, const cplx* in, const Op& op, int p, int dagger) {
  const long n = op.n();
  std::vector<cplx> xin(in, in + n), t1(n), t2(n);
  mask_parity(xin.data(), op.lat, p);
  if (!dagger) {
    dslash(t1.data(), xin.data(), op.U, op.lat, 0, op.blk);
    mask_parity(t1.data(), op.lat, 1 - p);
    clover_apply(t2.data(), t1.data(), op.T, op.lat, op.kappa, 1, 1 - p);
    dslash(t1.data(), t2.data(), op.U, op.lat, 0, op.blk);
    mask_parity(t1.data(), op.lat, p);
    clover_apply(t2.data(), t1.data(), op.T, op.lat, op.kappa, 1, p);
  } else {
    clover_apply(t1.data(), xin.data(), op.T, op.lat, op.kappa, 1, p);
    dslash(t2.data(), t1.data(), op.U, op.lat, 1, op.blk);
    mask_parity(t2.data(), op.lat, 1 - p);
    clover_apply(t1.data(), t2.data(), op.T, op.lat, op.kappa, 1, 1 - p);
    dslash(t2.data(), t1.data(), op.U, op.lat, 1, op.blk);
    mask_parity(t2.data(), op.lat, p);
  }
  const double k2 = op.kappa * op.kappa;
#pragma omp parallel for if(n >= 16384) schedule(static)
  for (long i = 0; i < n; ++i) out[i] = xin[i] - k2 * t2[i];
}

void apply_matpc(cplx* out, const cplx* in, const Op& op, int p, int dagger) {
  if (op.sym) { apply_matpc_sym(out, in, op, p, dagger); return; }
  const long n = op.n();
  std::vector<cplx> xin(in, in + n), t1(n), t2(n);
  mask_parity(xin.data(), op.lat, p);
  dslash(t1.data(), xin.data(), op.U, op.lat, dagger, op.blk, op.dom);     // lives on pbar
  mask_parity(t1.data(), op.lat, 1 - p);
  clover_apply(t2.data(), t1.data(), op.T, op.lat, op.kappa, 1, 1 - p);
  dslash(t1.data(), t2.data(), op.U, op.lat, dagger, op.blk, op.dom);      // back on p
  mask_parity(t1.data(), op.lat, p);
  clover_apply(out, xin.data(), op.T, op.lat, op.kappa, 0, p);
  const double k2 = op.kappa * op.kappa;
#pragma omp parallel for if(n >= 16384) schedule(static)
  for (long i = 0; i < n; ++i) out[i] -= k2 * t1[i];
}

// ---- linear algebra on full-lattice arrays -------------------------------------
cplx cdot(const cplx* a, const cplx* b, long n) {       // <a,b> = sum conj(a) b
  double re = 0, im = 0;
#pragma omp parallel for if(n >= 16384) reduction(+:re,im) schedule(static)
  for (long i = 0; i < n; ++i) { cplx t = std::conj(a[i]) * b[i]; re += t.real(); im += t.imag(); }
  return cplx(re, im);
}
double norm2(const cplx* a, long n) { return cdot(a, a, n).real(); }

// c.7  plain BiCGstab on Mhat (van der Vorst, ref [10]).
// Stops when ||r|| <= stop (absolute).  x is the initial guess on entry.
int bicgstab(cplx* x, const cplx* bhat, const Op& op, int p, double stop, int maxit, int* iters, double* rnorm) {
  const long n = op.n();
  std::vector<cplx> r(n), rt(n), pv(n, 0), v(n, 0), s(n), t(n);
  apply_matpc(r.data(), x, op, p, 0);
  for (long i = 0; i < n; ++i) r[i] = bhat[i] - r[i];
  mask_parity(r.data(), op.lat, p);
  rt = r;
  cplx rho = 1, alpha = 1, omega = 1;
  double rn = std::sqrt(norm2(r.data(), n));
  int it = 0, status = 0;
  while (rn > stop) {
    if (it >= maxit) { status = 1; break; }
    const cplx rho1 = cdot(rt.data(), r.data(), n);
    if (std::abs(rho1) == 0.0) { status = 2; break; }
    const cplx beta = (rho1 / rho) * (alpha / omega);
    for (long i = 0; i < n; ++i) pv[i] = r[i] + beta * (pv[i] - omega * v[i]);
    apply_matpc(v.data(), pv.data(), op, p, 0);
    alpha = rho1 / cdot(rt.data(), v.data(), n);
    for (long i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
    apply_matpc(t.data(), s.data(), op, p, 0);
    const double tt = norm2(t.data(), n);
    if (tt == 0.0) {                 // s is already the zero residual
      for (long i = 0; i < n; ++i) x[i] += alpha * pv[i];
      r = s; rn = std::sqrt(norm2(r.data(), n)); ++it; break;
    }
    omega = cdot(t.data(), s.data(), n) / tt;
    for (long i = 0; i < n; ++i) { x[i] += alpha * pv[i] + omega * s[i]; r[i] = s[i] - omega * t[i]; }
    rho = rho1;
    rn = std::sqrt(norm2(r.data(), n));
    ++it;
  }
  *iters = it; *rnorm = rn;
  return status;
}

// CGNR: conjugate gradients on the normal equations Mhat^dag Mhat x = Mhat^dag bhat (PAPER.md:128,
// Sec. 3.1: "either Conjugate Gradients [9] on the normal equations (CGNE or CGNR) is used, or ...
// BiCGstab").  Textbook form (Hestenes-Stiefel CG applied to A = Mhat^dag Mhat, with the residual of
// the ORIGINAL system r = bhat - Mhat x carried along):  z = Mhat^dag r;  p = z;  repeat
// { w = Mhat p; alpha = <z,z>/<w,w>; x += alpha p; r -= alpha w; z' = Mhat^dag r;
//   beta = <z',z'>/<z,z>; p = z' + beta p }.  Stops when ||r|| <= stop (absolute).
int cgnr(cplx* x, const cplx* bhat, const Op& op, int p, double stop, int maxit, int* iters, double* rnorm) {
  const long n = op.n();
  std::vector<cplx> r(n), z(n), pv(n), w(n);
  apply_matpc(r.data(), x, op, p, 0);
  for (long i = 0; i < n; ++i) r[i] = bhat[i] - r[i];
  mask_parity(r.data(), op.lat, p);
  apply_matpc(z.data(), r.data(), op, p, 1);
  pv = z;
  double zz = norm2(z.data(), n), rn = std::sqrt(norm2(r.data(), n));
  int it = 0, status = 0;
  while (rn > stop) {
    if (it >= maxit) { status = 1; break; }
    apply_matpc(w.data(), pv.data(), op, p, 0);
    const double ww = norm2(w.data(), n);
    if (ww == 0.0) { status = 2; break; }
    const double alpha = zz / ww;
    for (long i = 0; i < n; ++i) { x[i] += alpha * pv[i]; r[i] -= alpha * w[i]; }
    apply_matpc(z.data(), r.data(), op, p, 1);
    const double zz1 = norm2(z.data(), n);
    const double beta = zz1 / zz;
    for (long i = 0; i < n; ++i) pv[i] = z[i] + beta * pv[i];
    zz = zz1;
    rn = std::sqrt(norm2(r.data(), n));
    ++it;
  }
  *iters = it; *rnorm = rn;
  return status;
}

// CGNE (Craig's method): CG on Mhat Mhat^dag y = bhat with x = Mhat^dag y carried directly (PAPER.md:128,
// "CGNE or CGNR").  r = bhat - Mhat x;  p = Mhat^dag r;  repeat { alpha = <r,r>/<p,p>; x += alpha p;
// r -= alpha Mhat p; beta = <r',r'>/<r,r>; p = Mhat^dag r' + beta p }.  Stops when ||r|| <= stop (absolute).
int cgne(cplx* x, const cplx* bhat, const Op& op, int p, double stop, int maxit, int* iters, double* rnorm) {
  const long n = op.n();
  std::vector<cplx> r(n), z(n), pv(n), w(n);
  apply_matpc(r.data(), x, op, p, 0);
  for (long i = 0; i < n; ++i) r[i] = bhat[i] - r[i];
  mask_parity(r.data(), op.lat, p);
  apply_matpc(pv.data(), r.data(), op, p, 1);
  double rr = norm2(r.data(), n);
  int it = 0, status = 0;
  while (std::sqrt(rr) > stop) {
    if (it >= maxit) { status = 1; break; }
    const double pp = norm2(pv.data(), n);
    if (pp == 0.0) { status = 2; break; }
    const double alpha = rr / pp;
    apply_matpc(w.data(), pv.data(), op, p, 0);
    for (long i = 0; i < n; ++i) { x[i] += alpha * pv[i]; r[i] -= alpha * w[i]; }
    const double rr1 = norm2(r.data(), n);
    const double beta = rr1 / rr;
    apply_matpc(z.data(), r.data(), op, p, 1);
    for (long i = 0; i < n; ++i) pv[i] = z[i] + beta * pv[i];
    rr = rr1;
    ++it;
  }
  *iters = it; *rnorm = std::sqrt(rr);
  return status;
}

// c.8  Schwarz preconditioner K: n_mr MR steps on Mhat_D from x = 0,
// one alpha per block, sums over the block's parity-p sites.
void schwarz_K(cplx* out, const cplx* rin, const Op& opD, int p, int n_mr, double omega_mr) {
  const long n = opD.n(), V = opD.lat.V;
  const Lat& lat = opD.lat;
  const int* blk = opD.blk;
  int nb[4], NB = 1;
  for (int m = 0; m < 4; ++m) { nb[m] = blk ? lat.L[m] / blk[m] : 1; NB *= nb[m]; }
  std::vector<int> bid(V);
  for (long s = 0; s < V; ++s) {
    int c[4]; lat.coords(s, c);
    int b = 0;
    for (int m = 3; m >= 0; --m) b = b * nb[m] + (blk ? c[m] / blk[m] : 0);
    bid[s] = b;
  }
  std::vector<cplx> rho(rin, rin + n), w(n);
  mask_parity(rho.data(), lat, p);
  for (long i = 0; i < n; ++i) out[i] = 0;
  for (int step = 0; step < n_mr; ++step) {
    apply_matpc(w.data(), rho.data(), opD, p, 0);
    std::vector<cplx> wr(NB, 0); std::vector<double> ww(NB, 0);
    for (long s = 0; s < V; ++s) for (int i = 0; i < 12; ++i) {
      wr[bid[s]] += std::conj(w[s*12+i]) * rho[s*12+i];
      ww[bid[s]] += std::norm(w[s*12+i]);
    }
    for (long s = 0; s < V; ++s) {
      const int b = bid[s];
      const cplx a = (ww[b] > 0.0) ? omega_mr * wr[b] / ww[b] : cplx(0.0);
      for (int i = 0; i < 12; ++i) { out[s*12+i] += a * rho[s*12+i]; rho[s*12+i] -= a * w[s*12+i]; }
    }
  }
}

// Multiplicative Schwarz (SAP: section 4, "Schwarz alternating procedure" of ref. [20]; multiplicative
// variant named in PAPER.md:146 section 3.2; reading R16 in DESIGN.md).  Blocks are coloured (bx+by+bz+bt) mod 2.
// K_sap r: x = 0; repeat n_cycle times, for colour c = 0, 1:
//   rho = r on the blocks of colour c, 0 elsewhere;  y = (n_mr MR steps on Mhat_D from 0, one alpha per block) rho;
//   x += y;  r -= Mhat y   (the FULL operator: the other colour sees the update).
// One cycle with the update of r dropped between the colours would be the additive K above.
void schwarz_sap(cplx* out, const cplx* rin, const Op& op, const Op& opD, int p, int n_mr, double omega_mr, int n_cycle) {
  const long n = opD.n(), V = opD.lat.V;
  const Lat& lat = opD.lat;
  const int* blk = opD.blk;
  std::vector<int> colour(V);
  for (long s = 0; s < V; ++s) {
    int c[4]; lat.coords(s, c);
    int sum = 0;
    for (int m = 0; m < 4; ++m) sum += blk ? c[m] / blk[m] : 0;
    colour[s] = sum & 1;
  }
  std::vector<cplx> r(rin, rin + n), rho(n), y(n), t(n);
  mask_parity(r.data(), lat, p);
  for (long i = 0; i < n; ++i) out[i] = 0;
  for (int cyc = 0; cyc < n_cycle; ++cyc)
    for (int c = 0; c < 2; ++c) {
      for (long s = 0; s < V; ++s) for (int i = 0; i < 12; ++i) rho[s*12+i] = (colour[s] == c) ? r[s*12+i] : cplx(0.0);
      schwarz_K(y.data(), rho.data(), opD, p, n_mr, omega_mr);
      apply_matpc(t.data(), y.data(), op, p, 0);
      for (long i = 0; i < n; ++i) { out[i] += y[i]; r[i] -= t[i]; }
    }
}

// Overlapping additive Schwarz in its restricted form (PAPER.md:146 "blocks which may or may not overlap", :338
// "overlapping domains"; the restricted variant is the one of the paper's ref. [21]; reading R18 in
// DESIGN.md).  The domain of block b is its box grown by `ovl` sites on both sides of every partitioned direction
// (through the periodic wrap of the lattice; it must stay shorter than the lattice).  For every block, one at a time:
//   rho = r on the domain, 0 elsewhere;  x_b = n_mr MR steps from 0 on Mhat with every hop that leaves the domain
//   dropped, one alpha per domain;  out += x_b on the block's OWN box only (each site is written by exactly one block).
// ovl = 0 is the non-overlapping K above.  only_block >= 0: that block alone (sampling at large sizes).
// Returns 0, or 1 if a domain would reach around the lattice.
int schwarz_ras(cplx* out, const cplx* rin, const Op& op, const int* blk, int ovl, int p, int n_mr, double omega_mr, int only_block) {
  const long n = op.n(), V = op.lat.V;
  const Lat& lat = op.lat;
  int nb[4], NB = 1;
  for (int m = 0; m < 4; ++m) {
    nb[m] = lat.L[m] / blk[m]; NB *= nb[m];
    if (nb[m] > 1 && ovl > 0 && blk[m] + 2 * ovl >= lat.L[m]) return 1;
  }
  for (long i = 0; i < n; ++i) out[i] = 0;
  std::vector<unsigned char> dom(V), own(V);
  std::vector<cplx> rho(n), w(n), xb(n);
  for (int b = 0; b < NB; ++b) {
    if (only_block >= 0 && b != only_block) continue;
    int bc[4], q = b;
    for (int m = 0; m < 4; ++m) { bc[m] = q % nb[m]; q /= nb[m]; }
    for (long s = 0; s < V; ++s) {
      int c[4]; lat.coords(s, c);
      bool in = true, mine = true;
      for (int m = 0; m < 4; ++m) {
        if (nb[m] == 1) continue;                               // unpartitioned direction: the whole extent
        const int d = ((c[m] - bc[m] * blk[m]) % lat.L[m] + lat.L[m]) % lat.L[m];   // distance from the box's first site
        mine = mine && d < blk[m];
        in = in && (d < blk[m] + ovl || d >= lat.L[m] - ovl);
      }
      dom[s] = in; own[s] = mine;
    }
    Op od = op; od.blk = nullptr; od.dom = dom.data();
    for (long s = 0; s < V; ++s) for (int i = 0; i < 12; ++i) { rho[s*12+i] = dom[s] ? rin[s*12+i] : cplx(0.0); xb[s*12+i] = 0; }
    mask_parity(rho.data(), lat, p);
    for (int step = 0; step < n_mr; ++step) {
      apply_matpc(w.data(), rho.data(), od, p, 0);
      cplx wr = 0; double ww = 0;
      for (long i = 0; i < n; ++i) { wr += std::conj(w[i]) * rho[i]; ww += std::norm(w[i]); }
      const cplx a = (ww > 0.0) ? omega_mr * wr / ww : cplx(0.0);
      for (long i = 0; i < n; ++i) { xb[i] += a * rho[i]; rho[i] -= a * w[i]; }
    }
    for (long s = 0; s < V; ++s) if (own[s]) for (int i = 0; i < 12; ++i) out[s*12+i] += xb[s*12+i];
  }
  return 0;
}

// c.9  GCR-DD, Algorithm 1, all in fp64 here (hats kept as names only).
// Stops when ||r0|| <= stop.  precond: 0 = identity (plain GCR), 1 = Schwarz K.
int gcr_dd(cplx* x, const cplx* bhat, const Op& op, const Op& opD, int p, double stop, int maxit,
           int kmax, double delta, int precond, int n_mr, double omega_mr,
           int* iters, int* restarts, double* rnorm, int sap_cycles = 0) {
  const long n = op.n();
  std::vector<cplx> r0(n), rh(n), tmp(n), xh(n);
  std::vector<std::vector<cplx>> ph(kmax, std::vector<cplx>(n)), zh(kmax, std::vector<cplx>(n));
  std::vector<cplx> alpha(kmax), beta(kmax * kmax, 0), chi(kmax);
  std::vector<double> gamma(kmax);
  apply_matpc(tmp.data(), x, op, p, 0);
  for (long i = 0; i < n; ++i) r0[i] = bhat[i] - tmp[i];
  mask_parity(r0.data(), op.lat, p);
  double r0n = std::sqrt(norm2(r0.data(), n));
  rh = r0;
  int k = 0, total = 0, nrest = 0, status = 0;
  while (r0n > stop) {
    if (total >= maxit) { status = 1; break; }
    if (precond && sap_cycles > 0) schwarz_sap(ph[k].data(), rh.data(), op, opD, p, n_mr, omega_mr, sap_cycles);
    else if (precond) schwarz_K(ph[k].data(), rh.data(), opD, p, n_mr, omega_mr);
    else ph[k] = rh;
    apply_matpc(zh[k].data(), ph[k].data(), op, p, 0);
    for (int i = 0; i < k; ++i) {                       // orthogonalisation (modified Gram-Schmidt)
      const cplx b = cdot(zh[i].data(), zh[k].data(), n);
      beta[i * kmax + k] = b;
      for (long j = 0; j < n; ++j) zh[k][j] -= b * zh[i][j];
    }
    gamma[k] = std::sqrt(norm2(zh[k].data(), n));
    for (long j = 0; j < n; ++j) zh[k][j] /= gamma[k];
    alpha[k] = cdot(zh[k].data(), rh.data(), n);
    for (long j = 0; j < n; ++j) rh[j] -= alpha[k] * zh[k][j];
    ++k; ++total;
    const double rhn = std::sqrt(norm2(rh.data(), n));
    if (k == kmax || rhn / r0n < delta || rhn < stop) {  // high precision restart
      for (int l = k - 1; l >= 0; --l) {
        cplx t = alpha[l];
        for (int i = l + 1; i < k; ++i) t -= beta[l * kmax + i] * chi[i];
        chi[l] = t / gamma[l];
      }
      for (long j = 0; j < n; ++j) xh[j] = 0;
      for (int i = 0; i < k; ++i) for (long j = 0; j < n; ++j) xh[j] += chi[i] * ph[i][j];
      for (long j = 0; j < n; ++j) x[j] += xh[j];
      apply_matpc(tmp.data(), x, op, p, 0);
      for (long j = 0; j < n; ++j) r0[j] = bhat[j] - tmp[j];
      mask_parity(r0.data(), op.lat, p);
      r0n = std::sqrt(norm2(r0.data(), n));
      rh = r0; k = 0; ++nrest;
    }
  }
  *iters = total; *restarts = nrest; *rnorm = r0n;
  return status;
}

}  // namespace

// ============================ C entry points (ctypes) ===========================
extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// out16 = gamma_mu (mu = 0..3) or gamma5 (mu = 4), row-major 4x4
void orc_gamma(int mu, cplx* out16) {
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) out16[4*a+b] = G.g[mu][a][b];
}

// Full-lattice hopping term (c.1).  block may be NULL (no Dirichlet cut).
void orc_dslash(cplx* out, const cplx* in, const cplx* U, const int* dims, const int* bc, int dagger, const int* block) {
  Lat lat(dims, bc);
  dslash(out, in, U, lat, dagger, block);
}

// T[site][12][12] of reading R4
void orc_clover_term(cplx* T, const cplx* U, const int* dims, double c_sw) {
  Lat lat(dims, nullptr);
  clover_term(T, U, lat, c_sw);
}

// out = (1 + kappa T) in  or its inverse; parity = -1 (all sites) / 0 / 1 (others zeroed)
void orc_clover_apply(cplx* out, const cplx* in, const cplx* T, const int* dims, double kappa, int inverse, int parity) {
  Lat lat(dims, nullptr);
  clover_apply(out, in, T, lat, kappa, inverse, parity);
}

// out = (A - kappa D) in   (c.3)
void orc_M(cplx* out, const cplx* in, const cplx* U, const cplx* T, const int* dims, const int* bc,
           double kappa, int dagger, const int* block) {
  Op op(U, T, dims, bc, kappa, block);
  apply_M(out, in, op, dagger);
}

// out = Mhat in on parity p (c.5); full-lattice arrays, other parity of out is zero
void orc_matpc(cplx* out, const cplx* in, const cplx* U, const cplx* T, const int* dims, const int* bc,
               double kappa, int parity, int dagger, const int* block) {
  Op op(U, T, dims, bc, kappa, block);
  apply_matpc(out, in, op, parity, dagger);
}

// bhat_p = b_p + kappa D_{p pbar} A^{-1}_{pbar pbar} b_pbar   (c.5); other parity zeroed
void orc_prepare_source(cplx* bhat, const cplx* b, const cplx* U, const cplx* T, const int* dims, const int* bc,
                        double kappa, int parity) {
  Op op(U, T, dims, bc, kappa, nullptr);
  const long n = op.n();
  std::vector<cplx> t1(n), t2(n);
  clover_apply(t1.data(), b, T, op.lat, kappa, 1, 1 - parity);
  dslash(t2.data(), t1.data(), U, op.lat, 0, nullptr);
  for (long i = 0; i < n; ++i) bhat[i] = b[i] + kappa * t2[i];
  mask_parity(bhat, op.lat, parity);
}

// x_pbar = A^{-1}_{pbar pbar} (b_pbar + kappa D_{pbar p} x_p); x_p is kept   (c.5)
void orc_reconstruct(cplx* x, const cplx* b, const cplx* U, const cplx* T, const int* dims, const int* bc,
                     double kappa, int parity) {
  Op op(U, T, dims, bc, kappa, nullptr);
  const long n = op.n();
  std::vector<cplx> xp(x, x + n), t1(n), t2(n);
  mask_parity(xp.data(), op.lat, parity);
  dslash(t1.data(), xp.data(), U, op.lat, 0, nullptr);
  for (long i = 0; i < n; ++i) t1[i] = b[i] + kappa * t1[i];
  clover_apply(t2.data(), t1.data(), T, op.lat, kappa, 1, 1 - parity);
  for (long i = 0; i < n; ++i) x[i] = xp[i] + t2[i];
}

// K r (c.8) on parity p
void orc_schwarz(cplx* out, const cplx* rin, const cplx* U, const cplx* T, const int* dims, const int* bc,
                 double kappa, int parity, const int* block, int n_mr, double omega_mr) {
  Op opD(U, T, dims, bc, kappa, block);
  schwarz_K(out, rin, opD, parity, n_mr, omega_mr);
}

// K_sap r on parity p (multiplicative Schwarz, n_cycle cycles over the two block colours)
int orc_schwarz_ras(cplx* out, const cplx* rin, const cplx* U, const cplx* T, const int* dims, const int* bc,
                    double kappa, int parity, const int* block, int overlap, int n_mr, double omega_mr, int only_block) {
  Op op(U, T, dims, bc, kappa, nullptr);
  return schwarz_ras(out, rin, op, block, overlap, parity, n_mr, omega_mr, only_block);
}

void orc_schwarz_sap(cplx* out, const cplx* rin, const cplx* U, const cplx* T, const int* dims, const int* bc,
                     double kappa, int parity, const int* block, int n_mr, double omega_mr, int n_cycle) {
  Op op(U, T, dims, bc, kappa, nullptr);
  Op opD(U, T, dims, bc, kappa, block);
  schwarz_sap(out, rin, op, opD, parity, n_mr, omega_mr, n_cycle);
}

// GCR preconditioned by K_sap: solve Mhat x = bhat on one parity
int orc_gcr_sap_pc(cplx* x, const cplx* bhat, const cplx* U, const cplx* T, const int* dims, const int* bc,
                   double kappa, int parity, double stop, int maxit, int kmax, double delta,
                   const int* block, int n_mr, double omega_mr, int n_cycle, int* iters, int* restarts, double* rnorm) {
  Op op(U, T, dims, bc, kappa, nullptr);
  Op opD(U, T, dims, bc, kappa, block);
  return gcr_dd(x, bhat, op, opD, parity, stop, maxit, kmax, delta, 1, n_mr, omega_mr, iters, restarts, rnorm, n_cycle);
}

// Parity-system solves: Mhat x_p = bhat.  stop is an ABSOLUTE residual norm.
int orc_bicgstab_pc(cplx* x, const cplx* bhat, const cplx* U, const cplx* T, const int* dims, const int* bc,
                    double kappa, int parity, double stop, int maxit, int* iters, double* rnorm) {
  Op op(U, T, dims, bc, kappa, nullptr);
  return bicgstab(x, bhat, op, parity, stop, maxit, iters, rnorm);
}

int orc_cgnr_pc(cplx* x, const cplx* bhat, const cplx* U, const cplx* T, const int* dims, const int* bc,
                double kappa, int parity, double stop, int maxit, int* iters, double* rnorm) {
  Op op(U, T, dims, bc, kappa, nullptr);
  return cgnr(x, bhat, op, parity, stop, maxit, iters, rnorm);
}

int orc_gcr_pc(cplx* x, const cplx* bhat, const cplx* U, const cplx* T, const int* dims, const int* bc,
               double kappa, int parity, double stop, int maxit, int kmax, double delta,
               int precond, const int* block, int n_mr, double omega_mr,
               int* iters, int* restarts, double* rnorm) {
  Op op(U, T, dims, bc, kappa, nullptr);
  Op opD(U, T, dims, bc, kappa, block);
  return gcr_dd(x, bhat, op, opD, parity, stop, maxit, kmax, delta, precond, n_mr, omega_mr, iters, restarts, rnorm);
}

// Symmetric even-odd form: out = Mhat_s in  (or Mhat_s^dag in)
void orc_matpc_sym(cplx* out, const cplx* in, const cplx* U, const cplx* T, const int* dims, const int* bc,
                   double kappa, int parity, int dagger) {
  Op op(U, T, dims, bc, kappa, nullptr, 1);
  apply_matpc(out, in, op, parity, dagger);
}

// Full solve of M x = b through the SYMMETRIC Schur system Mhat_s x_p = A_pp^-1 bhat (solver 0 BiCGstab,
// 2 CGNR).  ||b - M x|| = ||A_pp r_s|| <= ||A|| ||r_s|| < 2 ||r_s|| (clover eigenvalues within
// 1 +- 6 kappa c_sw, kappa c_sw < 1/6), so iterating to ||r_s|| <= tol ||b|| / 2 meets the full-system criterion.
int orc_invert_sym(cplx* x, const cplx* b, const cplx* U, const cplx* T, const int* dims, const int* bc,
                   double kappa, int parity, double tol, int maxit, int solver, int* iters, double* true_res) {
  Op op(U, T, dims, bc, kappa, nullptr, 1);
  Op opa(U, T, dims, bc, kappa, nullptr, 0);
  const long n = op.n();
  std::vector<cplx> bhat(n), bs(n), xp(n, 0);
  orc_prepare_source(bhat.data(), b, U, T, dims, bc, kappa, parity);
  clover_apply(bs.data(), bhat.data(), T, op.lat, kappa, 1, parity);
  const double bn = std::sqrt(norm2(b, n));
  double rn = 0; int st;
  if (solver == 2) st = cgnr(xp.data(), bs.data(), op, parity, 0.5 * tol * bn, maxit, iters, &rn);
  else st = bicgstab(xp.data(), bs.data(), op, parity, 0.5 * tol * bn, maxit, iters, &rn);
  for (long i = 0; i < n; ++i) x[i] = xp[i];
  orc_reconstruct(x, b, U, T, dims, bc, kappa, parity);
  std::vector<cplx> mx(n);
  apply_M(mx.data(), x, opa, 0);
  double d = 0;
  for (long i = 0; i < n; ++i) d += std::norm(b[i] - mx[i]);
  *true_res = std::sqrt(d) / bn;
  return st;
}

// Full solve of M x = b (Eq. 1): prepare -> parity solve -> reconstruct.
// solver: 0 BiCGstab, 1 GCR-DD, 2 CGNR, 3 CGNE.  Stops on ||bhat - Mhat x_p|| <= tol*||b||  (= ||b - M x||, c.5).
int orc_invert(cplx* x, const cplx* b, const cplx* U, const cplx* T, const int* dims, const int* bc,
               double kappa, int parity, double tol, int maxit, int solver,
               int kmax, double delta, const int* block, int n_mr, double omega_mr,
               int* iters, double* true_res) {
  Op op(U, T, dims, bc, kappa, nullptr);
  const long n = op.n();
  std::vector<cplx> bhat(n), xp(n, 0);
  orc_prepare_source(bhat.data(), b, U, T, dims, bc, kappa, parity);
  const double bn = std::sqrt(norm2(b, n));
  int restarts = 0; double rn = 0; int st;
  if (solver == 0) st = bicgstab(xp.data(), bhat.data(), op, parity, tol * bn, maxit, iters, &rn);
  else if (solver == 2) st = cgnr(xp.data(), bhat.data(), op, parity, tol * bn, maxit, iters, &rn);
  else if (solver == 3) st = cgne(xp.data(), bhat.data(), op, parity, tol * bn, maxit, iters, &rn);
  else {
    Op opD(U, T, dims, bc, kappa, block);
    st = gcr_dd(xp.data(), bhat.data(), op, opD, parity, tol * bn, maxit, kmax, delta, 1, n_mr, omega_mr, iters, &restarts, &rn);
  }
  for (long i = 0; i < n; ++i) x[i] = xp[i];
  orc_reconstruct(x, b, U, T, dims, bc, kappa, parity);
  std::vector<cplx> mx(n);
  apply_M(mx.data(), x, op, 0);
  double d = 0;
  for (long i = 0; i < n; ++i) d += std::norm(b[i] - mx[i]);
  *true_res = std::sqrt(d) / bn;
  return st;
}

}  // extern "C"
