// clover.cu -- the site-local clover term A_x of Eq. 2 (72 reals, fn.1 :138).
//
//   T_x = c_sw * sum_{mu<nu} (i sigma_munu) (x) F_munu(x),  F = (Q - Q^dag)/8, Q = sum of the four
//   plaquette leaves in the mu-nu plane that start and end at x              (reading R4)
//   A_x(kappa) = 1 + kappa T_x                                               (reading R3)
//
// In the chiral basis (R2) i*sigma_munu is block diagonal, so A_x is two Hermitian 6x6 blocks
// (row = (spin mod 2)*3 + colour), each stored as 6 real diagonal entries + 15 complex
// lower-triangle entries.  Setup runs in fp64; A and A^-1 are then written in every storage
// precision (half: int16 with one fp32 norm per site, R9).
#include "host.h"

namespace lq {

__constant__ double c_isig[6 * 2 * 4 * 2];   // [pair(mu<nu)][chirality][s*2+s'][re,im] of i*sigma_munu

// ---- 3x3 complex fp64 helpers (row-major, 18 doubles) ----
template <bool DA, bool DB>
LQ_DEV void mm(const double* a, const double* b, double* c) {   // c = op(a) op(b), op = dagger if flag
#pragma unroll
  for (int r = 0; r < 3; ++r)
#pragma unroll
    for (int s = 0; s < 3; ++s) {
      double re = 0, im = 0;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const double ar = DA ? a[6 * k + 2 * r] : a[6 * r + 2 * k];
        const double ai = DA ? -a[6 * k + 2 * r + 1] : a[6 * r + 2 * k + 1];
        const double br = DB ? b[6 * s + 2 * k] : b[6 * k + 2 * s];
        const double bi = DB ? -b[6 * s + 2 * k + 1] : b[6 * k + 2 * s + 1];
        re += ar * br - ai * bi;
        im += ar * bi + ai * br;
      }
      c[6 * r + 2 * s] = re; c[6 * r + 2 * s + 1] = im;
    }
}

LQ_DEV void link_at(double* u, const double* g64, const Geom& g, const int* c, int mu) {
  const int par = (c[0] + c[1] + c[2] + c[3]) & 1;
  Rec<double, 18>::load(u, (const char*)g64 + (long long)(par * 4 + mu) * 144 * g.ns, g.ns, coords_to_cb(g, c));
}
LQ_DEV void shift(const Geom& g, const int* c, int mu, int dm, int nu, int dn, int* o) {
  o[0] = c[0]; o[1] = c[1]; o[2] = c[2]; o[3] = c[3];
  o[mu] = (o[mu] + dm + g.X[mu]) % g.X[mu];
  o[nu] = (o[nu] + dn + g.X[nu]) % g.X[nu];
}

__global__ void __launch_bounds__(64) clover_term_kernel(double* T72, const double* __restrict__ g64, const Geom g, double c_sw) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.ns) return;
  const int parity = blockIdx.y;
  int c[4];
  cb_to_coords(g, (int)i, parity, c);
  alignas(16) double t[72];
#pragma unroll
  for (int k = 0; k < 72; ++k) t[k] = 0;
  int pair = 0;
  for (int mu = 0; mu < 4; ++mu)
    for (int nu = mu + 1; nu < 4; ++nu, ++pair) {
      double Q[18], a[18], b[18], u1[18], u2[18], u3[18], u4[18];
      int n[4];
#pragma unroll
      for (int k = 0; k < 18; ++k) Q[k] = 0;
      // leaf 1: U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
      link_at(u1, g64, g, c, mu);
      shift(g, c, mu, +1, nu, 0, n); link_at(u2, g64, g, n, nu);
      shift(g, c, mu, 0, nu, +1, n); link_at(u3, g64, g, n, mu);
      link_at(u4, g64, g, c, nu);
      mm<false, false>(u1, u2, a); mm<false, true>(a, u3, b); mm<false, true>(b, u4, a);
#pragma unroll
      for (int k = 0; k < 18; ++k) Q[k] += a[k];
      // leaf 2: U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
      shift(g, c, mu, -1, nu, +1, n); link_at(u2, g64, g, n, mu);
      shift(g, c, mu, -1, nu, 0, n); link_at(u3, g64, g, n, nu); link_at(u1, g64, g, n, mu);
      mm<false, true>(u4, u2, a); mm<false, true>(a, u3, b); mm<false, false>(b, u1, a);
#pragma unroll
      for (int k = 0; k < 18; ++k) Q[k] += a[k];
      // leaf 3: U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
      shift(g, c, mu, -1, nu, -1, n); link_at(u2, g64, g, n, nu); link_at(u3, g64, g, n, mu);
      shift(g, c, mu, 0, nu, -1, n); link_at(u4, g64, g, n, nu);
      mm<true, true>(u1, u2, a); mm<false, false>(a, u3, b); mm<false, false>(b, u4, a);
#pragma unroll
      for (int k = 0; k < 18; ++k) Q[k] += a[k];
      // leaf 4: U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
      link_at(u1, g64, g, n, mu);
      shift(g, c, mu, +1, nu, -1, n); link_at(u2, g64, g, n, nu);
      link_at(u3, g64, g, c, mu);
      mm<true, false>(u4, u1, a); mm<false, false>(a, u2, b); mm<false, true>(b, u3, a);
#pragma unroll
      for (int k = 0; k < 18; ++k) Q[k] += a[k];
      // F = (Q - Q^dag)/8
      double F[18];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int s = 0; s < 3; ++s) {
          F[6 * r + 2 * s] = (Q[6 * r + 2 * s] - Q[6 * s + 2 * r]) * 0.125;
          F[6 * r + 2 * s + 1] = (Q[6 * r + 2 * s + 1] + Q[6 * s + 2 * r + 1]) * 0.125;
        }
      // accumulate the lower triangle of both chiral blocks
#pragma unroll
      for (int ch = 0; ch < 2; ++ch)
#pragma unroll
        for (int s = 0; s < 2; ++s)
#pragma unroll
          for (int sp = 0; sp < 2; ++sp) {
            const double wr = c_sw * c_isig[((pair * 2 + ch) * 4 + s * 2 + sp) * 2];
            const double wi = c_sw * c_isig[((pair * 2 + ch) * 4 + s * 2 + sp) * 2 + 1];
#pragma unroll
            for (int ca = 0; ca < 3; ++ca)
#pragma unroll
              for (int cb = 0; cb < 3; ++cb) {
                const int ii = s * 3 + ca, jj = sp * 3 + cb;
                if (ii < jj) continue;
                const double re = wr * F[6 * ca + 2 * cb] - wi * F[6 * ca + 2 * cb + 1];
                const double im = wr * F[6 * ca + 2 * cb + 1] + wi * F[6 * ca + 2 * cb];
                if (ii == jj) t[36 * ch + ii] += re;
                else { t[36 * ch + 6 + 2 * (ii * (ii - 1) / 2 + jj)] += re; t[36 * ch + 6 + 2 * (ii * (ii - 1) / 2 + jj) + 1] += im; }
              }
          }
    }
  Rec<double, 72>::store(t, (char*)T72 + (long long)parity * 576 * g.ns, g.ns, i);
}

cudaError_t run_clover_term(double* T72, const double* g64, const Geom& nat, double c_sw, cudaStream_t s) {
  // i*sigma_munu = -(1/2)[g_mu, g_nu] from this library's own statement of the DeGrand-Rossi basis
  typedef double C2[2];
  static const int gj[4][4] = {{3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}, {2, 3, 0, 1}};        // column of the non-zero in row a
  static const double gv[4][4][2] = {                                                           // its value
      {{0, 1}, {0, 1}, {0, -1}, {0, -1}}, {{-1, 0}, {1, 0}, {1, 0}, {-1, 0}},
      {{0, 1}, {0, -1}, {0, -1}, {0, 1}}, {{1, 0}, {1, 0}, {1, 0}, {1, 0}}};
  double gm[4][4][4][2] = {};
  for (int mu = 0; mu < 4; ++mu) for (int a = 0; a < 4; ++a) { gm[mu][a][gj[mu][a]][0] = gv[mu][a][0]; gm[mu][a][gj[mu][a]][1] = gv[mu][a][1]; }
  double h[6 * 2 * 4 * 2];
  int pair = 0;
  for (int mu = 0; mu < 4; ++mu) for (int nu = mu + 1; nu < 4; ++nu, ++pair) {
    double comm[4][4][2] = {};
    for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b) for (int k = 0; k < 4; ++k) {
      const double *x = gm[mu][a][k], *y = gm[nu][k][b], *p = gm[nu][a][k], *q = gm[mu][k][b];
      comm[a][b][0] += (x[0] * y[0] - x[1] * y[1]) - (p[0] * q[0] - p[1] * q[1]);
      comm[a][b][1] += (x[0] * y[1] + x[1] * y[0]) - (p[0] * q[1] + p[1] * q[0]);
    }
    for (int ch = 0; ch < 2; ++ch) for (int s = 0; s < 2; ++s) for (int sp = 0; sp < 2; ++sp) {
      h[((pair * 2 + ch) * 4 + s * 2 + sp) * 2] = -0.5 * comm[2 * ch + s][2 * ch + sp][0];
      h[((pair * 2 + ch) * 4 + s * 2 + sp) * 2 + 1] = -0.5 * comm[2 * ch + s][2 * ch + sp][1];
    }
  }
  (void)sizeof(C2);
  cudaError_t e = cudaMemcpyToSymbolAsync(c_isig, h, sizeof(h), 0, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return e;
  e = cudaStreamSynchronize(s);       // h is a stack array
  if (e != cudaSuccess) return e;
  dim3 grid((unsigned)((nat.ns + 63) / 64), 2), block(64);
  clover_term_kernel<<<grid, block, 0, s>>>(T72, g64, nat, c_sw);
  return cudaGetLastError();
}

// A = 1 + kappa T and A^-1 (6x6 Gauss-Jordan per chiral block, fp64) written in precision P
template <class P>
__global__ void __launch_bounds__(64) clover_make_kernel(char* A, char* Ainv, const double* __restrict__ T72, const BlockMap bm, int blocked, double kappa) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long ns_d = blocked ? bm.blk.ns : bm.nat.ns;      // block-major copies have their own size with overlapping domains (host.h)
  if (i >= ns_d) return;
  const int parity = blockIdx.y;
  long long is = i;
  if (blocked) is = block_to_natural(bm, (int)(i / bm.blk.vh), (int)(i % bm.blk.vh), parity);
  alignas(16) double t[72];
  Rec<double, 72>::load(t, (const char*)T72 + (long long)parity * 576 * bm.nat.ns, bm.nat.ns, is);
  double inv[72];
  for (int ch = 0; ch < 2; ++ch) {
    double* b = t + 36 * ch;
    for (int k = 0; k < 6; ++k) b[k] = 1.0 + kappa * b[k];
    for (int k = 6; k < 36; ++k) b[k] *= kappa;
    double mr[6][6], mi[6][6];
    for (int r = 0; r < 6; ++r) {
      mr[r][r] = b[r]; mi[r][r] = 0;
      for (int s = 0; s < r; ++s) {
        const double re = b[6 + 2 * (r * (r - 1) / 2 + s)], im = b[6 + 2 * (r * (r - 1) / 2 + s) + 1];
        mr[r][s] = re; mi[r][s] = im; mr[s][r] = re; mi[s][r] = -im;
      }
    }
    for (int k = 0; k < 6; ++k) {
      const double d = mr[k][k] * mr[k][k] + mi[k][k] * mi[k][k];
      const double pr = mr[k][k] / d, pi = -mi[k][k] / d;        // 1/pivot
      mr[k][k] = 1; mi[k][k] = 0;
      for (int s = 0; s < 6; ++s) {
        const double xr = mr[k][s], xi = mi[k][s];
        mr[k][s] = xr * pr - xi * pi; mi[k][s] = xr * pi + xi * pr;
      }
      for (int r = 0; r < 6; ++r) {
        if (r == k) continue;
        const double fr = mr[r][k], fi = mi[r][k];
        mr[r][k] = 0; mi[r][k] = 0;
        for (int s = 0; s < 6; ++s) {
          mr[r][s] -= fr * mr[k][s] - fi * mi[k][s];
          mi[r][s] -= fr * mi[k][s] + fi * mr[k][s];
        }
      }
    }
    double* o = inv + 36 * ch;
    for (int r = 0; r < 6; ++r) {
      o[r] = mr[r][r];
      for (int s = 0; s < r; ++s) { o[6 + 2 * (r * (r - 1) / 2 + s)] = mr[r][s]; o[6 + 2 * (r * (r - 1) / 2 + s) + 1] = mi[r][s]; }
    }
  }
  typename P::real v[72];
  const long long pb = (long long)parity * site_bytes<P>(72, true) * ns_d;
#pragma unroll
  for (int k = 0; k < 72; ++k) v[k] = (typename P::real)t[k];
  store_site<P, 72>(v, A + pb, ns_d, i);
#pragma unroll
  for (int k = 0; k < 72; ++k) v[k] = (typename P::real)inv[k];
  store_site<P, 72>(v, Ainv + pb, ns_d, i);
}

cudaError_t run_clover_make(int prec, char* A, char* Ainv, const double* T72, const BlockMap& bm, int blocked, double kappa, cudaStream_t s) {
  dim3 grid((unsigned)(((blocked ? bm.blk.ns : bm.nat.ns) + 63) / 64), 2), block(64);
  switch (prec) {
    case 0: clover_make_kernel<PrecD><<<grid, block, 0, s>>>(A, Ainv, T72, bm, blocked, kappa); break;
    case 1: clover_make_kernel<PrecS><<<grid, block, 0, s>>>(A, Ainv, T72, bm, blocked, kappa); break;
    case 2: clover_make_kernel<PrecH><<<grid, block, 0, s>>>(A, Ainv, T72, bm, blocked, kappa); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

// out = C in on one parity (C = A or A^-1): 504 flop per site
template <class P>
__global__ void __launch_bounds__(128) clover_apply_kernel(char* out, const char* in, const char* clov, const Geom g, int parity) {
  typedef typename P::real R;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.ns) return;
  R x[24], y[24];
  load_site<P, 24>(x, in, g.ns, i);
  clover_site<P>(y, x, clov + (long long)parity * site_bytes<P>(72, true) * g.ns, g.ns, i);
  store_site<P, 24>(y, out, g.ns, i);
}

cudaError_t run_clover_apply(int prec, char* out, const char* in, const char* clov, const Geom& g, int parity, cudaStream_t s) {
  dim3 grid((unsigned)((g.ns + 127) / 128)), block(128);
  switch (prec) {
    case 0: clover_apply_kernel<PrecD><<<grid, block, 0, s>>>(out, in, clov, g, parity); break;
    case 1: clover_apply_kernel<PrecS><<<grid, block, 0, s>>>(out, in, clov, g, parity); break;
    case 2: clover_apply_kernel<PrecH><<<grid, block, 0, s>>>(out, in, clov, g, parity); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace lq
