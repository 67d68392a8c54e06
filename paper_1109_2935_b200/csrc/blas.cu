// blas.cu -- launchers for the fused BLAS-1 passes (blas_ops.cuh), the multi-vector GCR
// orthogonalisation kernels (Algorithm 1) and the mixed-precision
// convert / accumulate kernels used at reliable updates and GCR restarts.
#include "blas_ops.cuh"
#include "host.h"

namespace lq {

template <class Op>
cudaError_t run_blas(int prec, const BlasArgs& a, int max_ctas, cudaStream_t s, int nrhs) {
  int gx = (a.vh + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK;
  if (gx > max_ctas) gx = max_ctas;
  if (gx < 1) gx = 1;
  if (nrhs > 1 && (a.nb != 1 || !a.rhs_bytes)) return cudaErrorInvalidValue;
  dim3 grid(gx, a.nb, nrhs), block(LQ_BLAS_BLOCK);
  switch (prec) {
    case 0: blas_kernel<PrecD, Op><<<grid, block, 0, s>>>(a); break;
    case 1: blas_kernel<PrecS, Op><<<grid, block, 0, s>>>(a); break;
    case 2: blas_kernel<PrecH, Op><<<grid, block, 0, s>>>(a); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

#define LQ_INST(OP) template cudaError_t run_blas<OP>(int, const BlasArgs&, int, cudaStream_t, int);
LQ_INST(OpZero) LQ_INST(OpNorm2) LQ_INST(OpCdot) LQ_INST(OpAxpyNorm) LQ_INST(OpXmyNorm)
LQ_INST(OpBicgInit) LQ_INST(OpBicgP) LQ_INST(OpBicgAlpha) LQ_INST(OpBicgS) LQ_INST(OpBicgOmega) LQ_INST(OpBicgXR)
LQ_INST(OpGcrScale)
LQ_INST(OpCgInit) LQ_INST(OpCgP) LQ_INST(OpCgAlpha) LQ_INST(OpCgXR)
LQ_INST(OpCgPAp) LQ_INST(OpCgXRB) LQ_INST(OpMsR)
typedef OpMrUpdate<true, false> OpMrFirst;
typedef OpMrUpdate<false, false> OpMrMid;
typedef OpMrUpdate<false, true> OpMrLast;
typedef OpMrUpdate<true, true> OpMrOnly;
LQ_INST(OpMrFirst) LQ_INST(OpMrMid) LQ_INST(OpMrLast) LQ_INST(OpMrOnly)
#undef LQ_INST

// alpha_b of the MR step for boxes [box0, box0 + nbox) (blas_ops.cuh)
__global__ void __launch_bounds__(LQ_BLAS_BLOCK) mr_alpha_kernel(const double* boxdots, int nchunk, int box0, double c0, double* boxalpha) {
  mr_alpha_box(boxdots, nchunk, box0 + blockIdx.x, c0, boxalpha);
}

cudaError_t run_mr_alpha(const BlasArgs& a, cudaStream_t s) {
  mr_alpha_kernel<<<a.nb, LQ_BLAS_BLOCK, 0, s>>>(a.boxdots, a.nchunk, a.box0, a.c[0], const_cast<double*>(a.boxalpha));
  return cudaGetLastError();
}

// ---------------------------------------------------------------- GCR multi-vector kernels
// beta_{i,k} = <z_i, z_k> for i in [i0, i0+n), n <= 8, one pass over z_k and the n vectors.
// N = number of vectors of this pass at compile time: the loads of all N + 1 operands of a site are issued before the
// first is used (with a run-time count the loop was load -> use -> load and ran at 3.3 TB/s)
template <class P, int N>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK, 2) gcr_dots_kernel(const MultiArgs m) {
  typedef typename P::real R;
  const BlasArgs& a = m.b;
  double red[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) red[k] = 0;
  for (int cb = blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x; cb < a.vh; cb += gridDim.x * LQ_BLAS_BLOCK) {
    R zk[24], zi[N][24];
    load_site<P, 24>(zk, m.z[m.k], a.ns, cb);
#pragma unroll
    for (int j = 0; j < N; ++j) load_site<P, 24>(zi[j], m.z[m.i0 + j], a.ns, cb);
#pragma unroll
    for (int j = 0; j < N; ++j) site_cdot(zi[j], zk, red[2 * j], red[2 * j + 1]);
  }
  reduce_and_finalize<16>(red, a, 0, [&](const double* s) {
#pragma unroll
    for (int j = 0; j < N; ++j) {
      double* b = a.S + S_GCR_BETA + 2 * ((m.i0 + j) * LQ_GCR_KMAX + m.k);
      b[0] = s[2 * j]; b[1] = s[2 * j + 1];
    }
  });
}

// z_k -= sum_{i<k} beta_{i,k} z_i ; then zz = ||z_k||^2, zr = <z_k, rhat> ;
// last CTA: gamma_k = sqrt(zz), alpha_k = zr / gamma_k  (Algorithm 1)
template <class P>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK, (sizeof(typename P::real) == 8 ? 1 : 2)) gcr_orth_kernel(const MultiArgs m) {
  typedef typename P::real R;
  const BlasArgs& a = m.b;
  double red[3] = {0, 0, 0};
  // -beta_{i,k} in the arithmetic type, once per CTA (read from the device scalars inside the site loop they cost two
  // dependent global loads and two conversions per vector and site)
  __shared__ R nb[2 * LQ_GCR_KMAX];
  if (threadIdx.x < m.k) {
    const double* b = a.S + S_GCR_BETA + 2 * (threadIdx.x * LQ_GCR_KMAX + m.k);
    nb[2 * threadIdx.x] = (R)(-b[0]); nb[2 * threadIdx.x + 1] = (R)(-b[1]);
  }
  __syncthreads();
  constexpr int U = sizeof(R) == 8 ? 1 : 3;      // earlier directions whose loads are in flight together
  for (int cb = blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x; cb < a.vh; cb += gridDim.x * LQ_BLAS_BLOCK) {
    R zk[24], r[24];
    load_site<P, 24>(zk, m.z[m.k], a.ns, cb);
    int i0 = 0;
    for (; i0 + U <= m.k; i0 += U) {             // whole rounds: no predicates, so the U loads are issued back to back
      R zi[U][24];
#pragma unroll
      for (int u = 0; u < U; ++u) load_site<P, 24>(zi[u], m.z[i0 + u], a.ns, cb);
#pragma unroll
      for (int u = 0; u < U; ++u) site_caxpy<R>(nb[2 * (i0 + u)], nb[2 * (i0 + u) + 1], zi[u], zk);
    }
    if (U > 2 && i0 + 2 <= m.k) {                // a tail of two: together as well
      R zi[2][24];
#pragma unroll
      for (int u = 0; u < 2; ++u) load_site<P, 24>(zi[u], m.z[i0 + u], a.ns, cb);
#pragma unroll
      for (int u = 0; u < 2; ++u) site_caxpy<R>(nb[2 * (i0 + u)], nb[2 * (i0 + u) + 1], zi[u], zk);
      i0 += 2;
    }
    for (; i0 < m.k; ++i0) {
      R zi[24];
      load_site<P, 24>(zi, m.z[i0], a.ns, cb);
      site_caxpy<R>(nb[2 * i0], nb[2 * i0 + 1], zi, zk);
    }
    if (m.k > 0) store_site<P, 24>(zk, (char*)m.z[m.k], a.ns, cb);
    load_site<P, 24>(r, a.v[0], a.ns, cb);
    site_norm2(zk, red[0]);
    site_cdot(zk, r, red[1], red[2]);
  }
  reduce_and_finalize<3>(red, a, 0, [&](const double* s) {
    double* S = a.S;
    const double gamma = sqrt(s[0]);
    // z_k = 0 exactly (rhat = 0, or p_k in the span of the earlier directions): alpha_k = 0 and the
    // direction drops out of the update; OpGcrScale and the host's back-substitution skip the division
    const double ig = gamma > 0.0 ? 1.0 / gamma : 0.0;
    S[S_GCR_ZZ] = s[0];
    S[S_GCR_GAMMA] = gamma;
    S[S_GCR_ALPHA] = s[1] * ig; S[S_GCR_ALPHA + 1] = s[2] * ig;
    S[S_GCR_GAMMAS + m.k] = gamma;
    S[S_GCR_ALPHAS + 2 * m.k] = s[1] * ig; S[S_GCR_ALPHAS + 2 * m.k + 1] = s[2] * ig;
  });
}

template <class P>
static cudaError_t gcr_dots_n(const MultiArgs& m, dim3 grid, dim3 block, cudaStream_t s) {
  switch (m.n) {
    case 1: gcr_dots_kernel<P, 1><<<grid, block, 0, s>>>(m); break;
    case 2: gcr_dots_kernel<P, 2><<<grid, block, 0, s>>>(m); break;
    case 3: gcr_dots_kernel<P, 3><<<grid, block, 0, s>>>(m); break;
    case 4: gcr_dots_kernel<P, 4><<<grid, block, 0, s>>>(m); break;
    case 5: gcr_dots_kernel<P, 5><<<grid, block, 0, s>>>(m); break;
    case 6: gcr_dots_kernel<P, 6><<<grid, block, 0, s>>>(m); break;
    case 7: gcr_dots_kernel<P, 7><<<grid, block, 0, s>>>(m); break;
    case 8: gcr_dots_kernel<P, 8><<<grid, block, 0, s>>>(m); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_gcr_dots(int prec, const MultiArgs& m, int max_ctas, cudaStream_t s) {
  int gx = (m.b.vh + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK;
  if (gx > max_ctas) gx = max_ctas;
  dim3 grid(gx), block(LQ_BLAS_BLOCK);
  switch (prec) {
    case 0: return gcr_dots_n<PrecD>(m, grid, block, s);
    case 1: return gcr_dots_n<PrecS>(m, grid, block, s);
    case 2: return gcr_dots_n<PrecH>(m, grid, block, s);
  }
  return cudaErrorInvalidValue;
}

cudaError_t run_gcr_orth(int prec, const MultiArgs& m, int max_ctas, cudaStream_t s) {
  int gx = (m.b.vh + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK;
  if (gx > max_ctas) gx = max_ctas;
  dim3 grid(gx), block(LQ_BLAS_BLOCK);
  switch (prec) {
    case 0: gcr_orth_kernel<PrecD><<<grid, block, 0, s>>>(m); break;
    case 1: gcr_orth_kernel<PrecS><<<grid, block, 0, s>>>(m); break;
    case 2: gcr_orth_kernel<PrecH><<<grid, block, 0, s>>>(m); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

// ---------------------------------------------------------------- mixed precision
// dst (PB) = src (PA), optionally permuting between the natural layout and the block-major
// layout of the Schwarz preconditioner (dir: 0 none, 1 natural -> blocks, 2 blocks -> natural).
template <class PA, class PB>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK) convert_kernel(char* dst, const char* src, const BlockMap bm, int dir, int parity,
                                                                int box0, int nbox) {
  // one thread per site of the block-major field (= per lattice site without overlap).  With overlapping domains
  // (host.h) a gather (dir 1) copies a lattice site into every box that holds it, with the box's sign; a scatter
  // (dir 2) writes the own sites of every box only, so each lattice site is written once.
  const long long i = (long long)blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x;
  if (i >= (dir == 0 ? bm.nat.ns : bm.blk.ns)) return;
  long long is = i, id = i, ns_s = bm.nat.ns, ns_d = bm.nat.ns;
  bool zero = false, own = true;
  int sign = 1;
  if (dir != 0) {
    const int box = (int)(i / bm.blk.vh), lcb = (int)(i % bm.blk.vh);
    const long long n = block_to_natural(bm, box, lcb, parity, &own, &sign);
    if (dir == 1) { is = n; id = i; ns_d = bm.blk.ns; } else { is = i; id = n; ns_s = bm.blk.ns; }
    zero = dir == 2 && nbox > 0 && (box < box0 || box >= box0 + nbox);     // outside the active box range (one colour)
    if (dir == 2 && !own) return;
  }
  typename PB::real vb[24];
  if (zero) {
#pragma unroll
    for (int k = 0; k < 24; ++k) vb[k] = 0;
  } else {
    typename PA::real va[24];
    load_site<PA, 24>(va, src, ns_s, is);
    const typename PB::real sg = (typename PB::real)((dir == 1) ? sign : 1);
#pragma unroll
    for (int k = 0; k < 24; ++k) vb[k] = sg * (typename PB::real)va[k];
  }
  store_site<PB, 24>(vb, dst, ns_d, id);
}

// y (PH) += sum_{i<n} chi_i * x_i (PL)   (implicit solution update; and
// x += x_lo at a reliable update with n = 1, chi = 1)
template <class PH_, class PL_>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK) accumulate_kernel(char* y, const MultiArgs m) {
  const long long i = (long long)blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x;
  if (i >= m.b.ns) return;
  typename PH_::real acc[24];
  load_site<PH_, 24>(acc, y, m.b.ns, i);
  auto add = [&](const typename PL_::real* x, int j) {
    const typename PH_::real cr = (typename PH_::real)m.chi[2 * j], ci = (typename PH_::real)m.chi[2 * j + 1];
#pragma unroll
    for (int k = 0; k < 12; ++k) {
      const typename PH_::real xr = (typename PH_::real)x[2 * k], xi = (typename PH_::real)x[2 * k + 1];
      acc[2 * k] += cr * xr - ci * xi;
      acc[2 * k + 1] += cr * xi + ci * xr;
    }
  };
  // whole rounds of U vectors without predicates, so that their loads are in flight together (same order of the sums)
  constexpr int U = sizeof(typename PL_::real) == 8 ? 1 : 3;
  int j = 0;
  for (; j + U <= m.n; j += U) {
    typename PL_::real x[U][24];
#pragma unroll
    for (int u = 0; u < U; ++u) load_site<PL_, 24>(x[u], m.z[j + u], m.b.ns, i);
#pragma unroll
    for (int u = 0; u < U; ++u) add(x[u], j + u);
  }
  if (U > 2 && j + 2 <= m.n) {                   // a tail of two: together as well
    typename PL_::real x[2][24];
#pragma unroll
    for (int u = 0; u < 2; ++u) load_site<PL_, 24>(x[u], m.z[j + u], m.b.ns, i);
#pragma unroll
    for (int u = 0; u < 2; ++u) add(x[u], j + u);
    j += 2;
  }
  for (; j < m.n; ++j) {
    typename PL_::real x[24];
    load_site<PL_, 24>(x, m.z[j], m.b.ns, i);
    add(x, j);
  }
  store_site<PH_, 24>(acc, y, m.b.ns, i);
}

template <class PA>
static cudaError_t convert_b(int pb, char* dst, const char* src, const BlockMap& bm, int dir, int parity, cudaStream_t s, int box0, int nbox) {
  const long long nsite = dir == 0 ? bm.nat.ns : bm.blk.ns;
  dim3 grid((unsigned)((nsite + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK)), block(LQ_BLAS_BLOCK);
  switch (pb) {
    case 0: convert_kernel<PA, PrecD><<<grid, block, 0, s>>>(dst, src, bm, dir, parity, box0, nbox); break;
    case 1: convert_kernel<PA, PrecS><<<grid, block, 0, s>>>(dst, src, bm, dir, parity, box0, nbox); break;
    case 2: convert_kernel<PA, PrecH><<<grid, block, 0, s>>>(dst, src, bm, dir, parity, box0, nbox); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_convert(int pa, int pb, char* dst, const char* src, const BlockMap& bm, int dir, int parity, cudaStream_t s, int box0, int nbox) {
  switch (pa) {
    case 0: return convert_b<PrecD>(pb, dst, src, bm, dir, parity, s, box0, nbox);
    case 1: return convert_b<PrecS>(pb, dst, src, bm, dir, parity, s, box0, nbox);
    case 2: return convert_b<PrecH>(pb, dst, src, bm, dir, parity, s, box0, nbox);
  }
  return cudaErrorInvalidValue;
}

template <class PH_>
static cudaError_t accumulate_b(int pl, char* y, const MultiArgs& m, cudaStream_t s) {
  dim3 grid((unsigned)((m.b.ns + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK)), block(LQ_BLAS_BLOCK);
  switch (pl) {
    case 0: accumulate_kernel<PH_, PrecD><<<grid, block, 0, s>>>(y, m); break;
    case 1: accumulate_kernel<PH_, PrecS><<<grid, block, 0, s>>>(y, m); break;
    case 2: accumulate_kernel<PH_, PrecH><<<grid, block, 0, s>>>(y, m); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_accumulate(int ph, int pl, char* y, const MultiArgs& m, cudaStream_t s) {
  switch (ph) {
    case 0: return accumulate_b<PrecD>(pl, y, m, s);
    case 1: return accumulate_b<PrecS>(pl, y, m, s);
    case 2: return accumulate_b<PrecH>(pl, y, m, s);
  }
  return cudaErrorInvalidValue;
}

// Final sum of the per-CTA partials of a reduction fused into the operator (dslash.cuh, DOTS >= 2) and the scalar
// update `fin`: one CTA, partials added in a fixed order (bit-reproducible).  W: workspace of get_dotws (api.cu).
__global__ void __launch_bounds__(1024) dots_finalize_kernel(double* W, int n, int fin) {
  __shared__ double sm[3 * 32];
  const double* part = W + 8;
  double s[3] = {0, 0, 0};
  for (int i0 = threadIdx.x; i0 < n; i0 += 8 * 1024) {
    double t[8][3];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int i = i0 + u * 1024;
      const bool ok = i < n;
#pragma unroll
      for (int k = 0; k < 3; ++k) t[u][k] = ok ? __ldcg(part + 3ll * i + k) : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) { s[0] += t[u][0]; s[1] += t[u][1]; s[2] += t[u][2]; }
  }
  cta_reduce<3, 1024>(s, sm);
  if (threadIdx.x == 0) dots_finalize(*reinterpret_cast<double**>(W), s, fin);
}

cudaError_t run_dots_finalize(double* W, int n, int fin, cudaStream_t s) {
  dots_finalize_kernel<<<1, 1024, 0, s>>>(W, n, fin);
  return cudaGetLastError();
}

}  // namespace lq
