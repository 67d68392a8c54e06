// blas.cuh -- fused BLAS-1 kernels with deterministic reductions on packed spinor fields.
//
// "BLAS1-type linear algebra ... extremely bandwidth intensive"; reductions run
// over the contiguous local field.  Every kernel is one pass: each operand is
// read once with 128-bit loads, each result written once, all reductions of the pass are
// accumulated in fp64 in the same pass (warp shuffle -> CTA -> per-CTA partial in HBM; the
// last CTA to finish sums the partials in a fixed order, so results are bit-reproducible) and
// the scalar recurrences of the solver (alpha, beta, omega of BiCGstab; gamma, alpha of GCR)
// are updated on the device by that last CTA -- no host round trip gates the next launch.
#pragma once
#include "dslash.cuh"

namespace lq {

#define LQ_BLAS_BLOCK 256
#ifndef LQ_BLAS_CTAS_PER_SM
#define LQ_BLAS_CTAS_PER_SM 8     /* grid of the grid-stride BLAS-1 kernels = this x number of SMs */
#endif
#define LQ_MAX_VEC 5
#define LQ_GCR_KMAX 32

// slots of the device scalar array S (doubles)
enum {
  S_RHO = 0, S_RHO_OLD = 2, S_ALPHA = 4, S_OMEGA = 6, S_BETA = 8, S_RR = 10, S_FLAG = 11,
  S_RTV = 12, S_TS = 14, S_TT = 16, S_OUT = 20 /* generic results: 20..27 */,
  S_DONE = 28,    // batched solves: nonzero = this right-hand side has converged, its passes are skipped
  S_GCR_GAMMA = 32, S_GCR_ALPHA = 34, S_GCR_ZZ = 36,
  S_GCR_BETA = 64,                         // beta[i][k] complex: S_GCR_BETA + 2*(i*LQ_GCR_KMAX + k)
  S_GCR_GAMMAS = S_GCR_BETA + 2 * LQ_GCR_KMAX * LQ_GCR_KMAX,   // gamma[k]
  S_GCR_ALPHAS = S_GCR_GAMMAS + LQ_GCR_KMAX,                   // alpha[k] complex
  S_TOTAL = S_GCR_ALPHAS + 2 * LQ_GCR_KMAX
};

static_assert(S_RHO == LQ_S_RHO && S_ALPHA == LQ_S_ALPHA && S_OMEGA == LQ_S_OMEGA && S_FLAG == LQ_S_FLAG && S_RTV == LQ_S_RTV &&
              S_TS == LQ_S_TS && S_TT == LQ_S_TT, "dslash.cuh dots_finalize uses these slot numbers");

struct BlasArgs {
  char* v[LQ_MAX_VEC];
  long long ns;
  int vh, nb;
  double* S;              // device scalars
  double* partials;       // [nb][gridDim.x][NV]
  unsigned* counters;     // [nb], zero on entry, reset by the last CTA
  const double* boxdots;  // MR: per-box partial dots written by the Dslash epilogue [nb][nchunk][4], nchunk = CTAs per box x warps per CTA
  int nchunk;
  const double* boxalpha; // MR: alpha_b (re, im) per box, formed from boxdots by mr_alpha_kernel (blas.cu)
  double c[4];            // host coefficients
  int i0, i1;
  // batched launch over right-hand sides (gridDim.z = nrhs, nb must be 1): right-hand side r uses
  // v[j] + r * rhs_bytes, S + r * S_TOTAL, partials + r * rhs_partials, counters + r
  long long rhs_bytes;
  long long rhs_partials;
  // pinned host words the last CTA may publish scalars to (zero-copy; no memcpy or event between two kernels)
  double* hmirror;
  int box0;               // first box of the launch (gridDim.y counts boxes from it): Schwarz block groups
};

struct cd { double re, im; };
LQ_DEV cd cd_mul(cd a, cd b) { return {a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
LQ_DEV cd cd_div(cd a, cd b) {
  const double d = b.re * b.re + b.im * b.im;
  return {(a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d};
}

// y += (ar + i ai) * x   on one site (12 complex)
template <typename R> LQ_DEV void site_caxpy(R ar, R ai, const R* x, R* y) {
#pragma unroll
  for (int k = 0; k < 12; ++k) {
    y[2 * k] += ar * x[2 * k] - ai * x[2 * k + 1];
    y[2 * k + 1] += ar * x[2 * k + 1] + ai * x[2 * k];
  }
}
// red[0..1] += conj(x) . y ; optional red2 += |y|^2
template <typename R> LQ_DEV void site_cdot(const R* x, const R* y, double& re, double& im) {
  R sr = 0, si = 0;
#pragma unroll
  for (int k = 0; k < 12; ++k) {
    sr += x[2 * k] * y[2 * k] + x[2 * k + 1] * y[2 * k + 1];
    si += x[2 * k] * y[2 * k + 1] - x[2 * k + 1] * y[2 * k];
  }
  re += (double)sr; im += (double)si;
}
template <typename R> LQ_DEV void site_norm2(const R* x, double& n) {
  R s = 0;
#pragma unroll
  for (int k = 0; k < 24; ++k) s += x[k] * x[k];
  n += (double)s;
}

// CTA reduce -> per-CTA partial -> last CTA of the box sums all partials in a fixed order and
// calls fin(sum).  Deterministic for a fixed launch configuration.
template <int NV, class F>
LQ_DEV void reduce_and_finalize(double* red, const BlasArgs& a, int box, F fin) {
  __shared__ double sm[NV * (LQ_BLAS_BLOCK / 32)];
  __shared__ bool last;
  cta_reduce<NV, LQ_BLAS_BLOCK>(red, sm);
  double* part = a.partials + (long long)box * gridDim.x * NV;
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) part[(long long)blockIdx.x * NV + k] = red[k];
    __threadfence();
    const unsigned t = atomicAdd(a.counters + box, 1u);
    last = (t == gridDim.x - 1);
  }
  __syncthreads();
  if (last) {
    __threadfence();
    double s[NV];
#pragma unroll
    for (int k = 0; k < NV; ++k) s[k] = 0;
    for (int i = threadIdx.x; i < (int)gridDim.x; i += LQ_BLAS_BLOCK) {
#pragma unroll
      for (int k = 0; k < NV; ++k) s[k] += __ldcg(part + (long long)i * NV + k);
    }
    __syncthreads();
    cta_reduce<NV, LQ_BLAS_BLOCK>(s, sm);
    if (threadIdx.x == 0) {
      fin(s);
      a.counters[box] = 0;
    }
  }
}

// Generic one-pass kernel.  Op provides:
//   NV (number of fp64 reductions), READ / WRITE bit masks over v[0..4],
//   struct Coef; prepare(Coef&, const BlasArgs&, int box);
//   site<R>(const Coef&, R* v0..v4, double* red);  finalize(const double* sum, const BlasArgs&, int box)
// half precision: a site needs all 24 decoded values of every operand before it can re-quantise, and the widest passes
// (OpBicgXR: 5 operands) would take 137 registers = one CTA of 8 warps per SM; capped at 128 for two (measured below)
#ifndef LQ_BLAS_MINB_HALF
#define LQ_BLAS_MINB_HALF 2
#endif
// the three-operand MR update runs three CTAs per SM (80 registers; 12 bytes spilled in one variant): K at config 5 14.05 -> 13.6 ms
template <bool FIRST, bool LASTSTEP> struct OpMrUpdate;
template <class Op> struct BlasMinbHalf { static constexpr int value = LQ_BLAS_MINB_HALF; };
template <bool F, bool L> struct BlasMinbHalf<OpMrUpdate<F, L>> { static constexpr int value = 3; };
template <class P, class Op>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK, (P::HALF ? BlasMinbHalf<Op>::value : 1)) blas_kernel(const BlasArgs a0) {
  typedef typename P::real R;
  const int box = blockIdx.y + a0.box0;
  BlasArgs a = a0;
  if (a0.rhs_bytes) {                       // one right-hand side per blockIdx.z, each with its own scalars
    const int r = blockIdx.z;
    a.S = a0.S + (long long)r * S_TOTAL;
    if (a.S[S_DONE] != 0.0) return;         // converged: leave its vectors alone
#pragma unroll
    for (int j = 0; j < LQ_MAX_VEC; ++j) a.v[j] = a0.v[j] ? a0.v[j] + (long long)r * a0.rhs_bytes : nullptr;
    a.partials = a0.partials + (long long)r * a0.rhs_partials;
    a.counters = a0.counters + r;
  }
  typename Op::Coef coef;
  Op::prepare(coef, a, box);
  constexpr int NV = Op::NV > 0 ? Op::NV : 1;
  double red[NV];
#pragma unroll
  for (int k = 0; k < NV; ++k) red[k] = 0;
  for (int cb = blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x; cb < a.vh; cb += gridDim.x * LQ_BLAS_BLOCK) {
    const long long idx = (long long)box * a.vh + cb;
    R v[LQ_MAX_VEC][24];
#pragma unroll
    for (int j = 0; j < LQ_MAX_VEC; ++j)
      if (Op::READ & (1 << j)) load_site<P, 24>(v[j], a.v[j], a.ns, idx);
    Op::template site<R>(coef, v[0], v[1], v[2], v[3], v[4], red);
#pragma unroll
    for (int j = 0; j < LQ_MAX_VEC; ++j)
      if (Op::WRITE & (1 << j)) store_site<P, 24>(v[j], a.v[j], a.ns, idx);
  }
  if constexpr (Op::NV > 0) {
    reduce_and_finalize<NV>(red, a, box, [&](const double* s) { Op::finalize(s, a, box); });
  }
}

template <class Op> cudaError_t run_blas(int prec, const BlasArgs& a, int max_ctas, cudaStream_t s, int nrhs = 1);

}  // namespace lq
