// dslash.cuh -- the Wilson-clover hopping term with fused clover / xpay epilogues.
//
// Computes, for every site x of parity p of every box in the batch (Eq. 2;
// readings R1,R2,R5 in DESIGN.md):
//
//   r(x) = sum_mu [ s+ (1 -/+ g_mu) U_mu(x) in(x+mu) + s- (1 +/- g_mu) U_mu(x-mu)^dag in(x-mu) ]
//
// (upper signs: D, lower signs: D^dagger), then the epilogue
//
//   XPAY    : r = y + a*r           (CLOVX: y := A_x y first)       -> Mhat second half, source prep
//   CLOVOUT : r = C_x r             (C = A^-1 of the output parity)  -> Mhat first half, reconstruction
//   DOTS 1  : per-box partial sums of <r,y> and <r,r>               -> fused MR reductions
//   DOTS 2/3: global <r,y> / <q,r> and <r,r>, scalar update by dots_finalize_kernel behind it -> BiCGstab omega / alpha, CGNR alpha
//             (BLAS-1 is "extremely bandwidth intensive", so the reduction-only passes are not paid twice)
//
// One thread per output site (PAPER.md:164, :200-202 K1): 8 neighbour spinors + 8 links are
// loaded with 128-bit coalesced loads; the 8-fold reuse of each input spinor is served by L2
// (126 MB on B200).  CUDA-core FMA only: 3x3 complex matvecs
// are not a dense contraction.  Spin projection uses the rank-2 structure of (1 +- g_mu) in
// the chiral basis: 12 reals per hop go through the SU(3) multiply instead of 24.  fp32 arithmetic is written in
// packed complex form (FFMA2 with broadcast / swap-negate operand modifiers, core.cuh f2): the kernels are bound by
// register-file bandwidth before the FMA lanes.  dslash_tile.cuh holds the CTA-tile form with bulk-async staging.
// Half / recon 12: the clover block and the xpay vector of the epilogue are cp.async'ed into the thread's own
// bytes of the ring slots that hops 4..6 have drained (EpiSlot), so the epilogue starts from shared memory.
#pragma once
#include "core.cuh"

namespace lq {

struct DslashArgs {
  Geom g;
  char* out;            // packed spinor, output parity
  const char* in;       // packed spinor, input parity
  const char* y;        // XPAY operand (output parity) or nullptr
  const char* gauge;    // packed links, [parity][mu] records of RECON reals
  const char* clov_y;   // A of the output parity (CLOVX)
  const char* clov_out; // A^-1 of the output parity (CLOVOUT)
  double a;             // xpay coefficient
  // The struct is kept at 128 bytes: one more word and ptxas (12.9, sm_100a) spills ~400 bytes
  // per thread in the 80-register clover-epilogue variants.  A DOTS launch always covers whole
  // boxes, so the site range shares storage with the partial-sum pointer.
  union {
    double* dots;       // DOTS: [box][chunk][warp][4] partials (re<r,y>, im<r,y>, <r,r>, unused)
    struct { int cb0, cb1; } range;  // !DOTS: sites [cb0, cb1) of every box are computed by this launch
  };
  int parity;           // output parity (bit 0); bits 8.. = first box of the launch (the grid's y extent counts boxes from it)
  int dagger;
};
static_assert(sizeof(DslashArgs) == 128, "DslashArgs must stay 128 bytes (see above)");

// multiply by a compile-time unit: C = 0: 1, 1: i, 2: -1, 3: -i
template <int C, typename R> LQ_DEV cx<R> unit_mul(cx<R> z) {
  if (C == 0) return z;
  if (C == 1) return {-z.im, z.re};
  if (C == 2) return {-z.re, -z.im};
  return {z.im, -z.re};
}

// (re, im) of unit<C>(z) as a packed pair: the swap and the signs become operand modifiers of the consuming FFMA2
template <int C> LQ_DEV f2 unit_pair(float re, float im) {
  if (C == 0) return f2_make(re, im);
  if (C == 1) return f2_make(-im, re);
  if (C == 2) return f2_make(-re, -im);
  return f2_make(im, -re);
}

// (gamma_mu psi)_0 = c0 psi_{j0}, (gamma_mu psi)_1 = c1 psi_{j1} in the DeGrand-Rossi basis (R2)
template <int MU> struct GammaRow;
template <> struct GammaRow<0> { static constexpr int j0 = 3, c0 = 1, j1 = 2, c1 = 1; };   // gamma_x
template <> struct GammaRow<1> { static constexpr int j0 = 3, c0 = 2, j1 = 2, c1 = 0; };   // gamma_y
template <> struct GammaRow<2> { static constexpr int j0 = 2, c0 = 1, j1 = 3, c1 = 3; };   // gamma_z
template <> struct GammaRow<3> { static constexpr int j0 = 2, c0 = 0, j1 = 3, c1 = 0; };   // gamma_t

// One hop: acc += coef * (1 + sigma*gamma_MU) W psi,  W = U (FWD) or U^dagger (!FWD).
// coef carries the boundary sign and, in half precision, the spinor norm and the link scale.
// All multiply-adds are written as explicit FMAs (nvcc does not re-associate a*b - c*d + e).
template <int MU, bool FWD, typename R>
LQ_DEV void hop_tail(R* __restrict__ acc, const cx<R> (&h)[2][3], const R* __restrict__ u, R sigma, R coef);

template <int MU, bool FWD, typename R>
LQ_DEV void hop(R* __restrict__ acc, const R* __restrict__ psi, const R* __restrict__ u, R sigma, R coef) {
  typedef GammaRow<MU> G;
  // project: h0 = psi_0 + sigma*c0*psi_j0, h1 = psi_1 + sigma*c1*psi_j1   (3 colours each)
  cx<R> h[2][3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if constexpr (sizeof(R) == 4) {
      const f2 sg = f2_bcast(sigma);
      f2_split(f2_fma(sg, unit_pair<G::c0>(psi[6 * G::j0 + 2 * c], psi[6 * G::j0 + 2 * c + 1]), f2_make(psi[2 * c], psi[2 * c + 1])), h[0][c].re, h[0][c].im);
      f2_split(f2_fma(sg, unit_pair<G::c1>(psi[6 * G::j1 + 2 * c], psi[6 * G::j1 + 2 * c + 1]), f2_make(psi[6 + 2 * c], psi[6 + 2 * c + 1])), h[1][c].re, h[1][c].im);
    } else {
      const cx<R> q0 = unit_mul<G::c0>(cx<R>{psi[6 * G::j0 + 2 * c], psi[6 * G::j0 + 2 * c + 1]});
      const cx<R> q1 = unit_mul<G::c1>(cx<R>{psi[6 * G::j1 + 2 * c], psi[6 * G::j1 + 2 * c + 1]});
      h[0][c] = {fma_(sigma, q0.re, psi[2 * c]), fma_(sigma, q0.im, psi[2 * c + 1])};
      h[1][c] = {fma_(sigma, q1.re, psi[6 + 2 * c]), fma_(sigma, q1.im, psi[6 + 2 * c + 1])};
    }
  }
  hop_tail<MU, FWD, R>(acc, h, u, sigma, coef);
}

// ---- 16-bit fixed point: projection fused with the decode (compile-time sigma) -----------------------
// A stored value q in [-32767, 32767] arrives as the float m = 2^23 + 32768 + q (one PRMT, core.cuh).  The
// projected component q_a + s q_b (s = +-1) is formed on these floats directly, exactly:
//   s = -1:  m_a - m_b                         (one FADD; both offsets cancel)
//   s = +1:  (m_a - 2(2^23 + 32768)) + m_b     (two FADDs; every intermediate is an integer below 2^24)
// instead of two decoding FADDs and one FFMA: 1.5 instead of 3 instructions per projected real.  Which
// of the two applies to a component depends on sigma, so the dagger flag is a template parameter of the
// half-precision kernels.  Results are bit-identical to decode-then-project.
// Packed (core.cuh, f2): both components of a projected complex number at once.  With signs (SRE, SIM):
//   (-,-): A + (-X)                      one FADD2
//   else : (A + K) + X',  K = -2(2^23+32768) in the '+' components and 0 in the '-' ones (adding 0 is exact),
//          X' = X with the '-' components negated        two FADD2
// (a + SG * unit<C>(b)) on magic floats: unit<0> = 1, <1> = i, <2> = -1, <3> = -i
template <int C, int SG> LQ_DEV cx<float> fixed_project(float ar, float ai, float br, float bi) {
  constexpr int SRE = SG * ((C == 0 || C == 3) ? 1 : -1);
  constexpr int SIM = SG * ((C == 0 || C == 1) ? 1 : -1);
  const float xr = (C == 0 || C == 2) ? br : bi;
  const float xi = (C == 0 || C == 2) ? bi : br;
  const f2 A = f2_make(ar, ai);
  const f2 X = f2_make(SRE < 0 ? -xr : xr, SIM < 0 ? -xi : xi);
  f2 r;
  if (SRE < 0 && SIM < 0) r = f2_add(A, X);
  else r = f2_add(f2_add(A, f2_make(SRE < 0 ? 0.0f : -2.0f * LQ_MAGIC_DEC, SIM < 0 ? 0.0f : -2.0f * LQ_MAGIC_DEC)), X);
  cx<float> o;
  f2_split(r, o.re, o.im);
  return o;
}
template <int MU, bool FWD, int SG>
LQ_DEV void hop_fixed(float* __restrict__ acc, const float* __restrict__ m, const float* __restrict__ u, float coef) {
  typedef GammaRow<MU> G;
  cx<float> h[2][3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    h[0][c] = fixed_project<G::c0, SG>(m[2 * c], m[2 * c + 1], m[6 * G::j0 + 2 * c], m[6 * G::j0 + 2 * c + 1]);
    h[1][c] = fixed_project<G::c1, SG>(m[6 + 2 * c], m[6 + 2 * c + 1], m[6 * G::j1 + 2 * c], m[6 * G::j1 + 2 * c + 1]);
  }
  hop_tail<MU, FWD, float>(acc, h, u, (float)SG, coef);
}

// fp32 arithmetic: packed complex form (core.cuh, f2): 2 FFMA2 per complex multiply-add, same per-component order
// of operations as the scalar form below (bit-identical results)
template <int MU, bool FWD>
LQ_DEV void hop_tail_packed(float* __restrict__ acc, const cx<float> (&h)[2][3], const float* __restrict__ u, float sigma, float coef) {
  typedef GammaRow<MU> G;
  f2 w[2][3];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      f2 t;
      if (FWD) {                         // sum_k U[r][k] * h[k]
        t = f2_mul(f2_make(h[s][0].re, h[s][0].im), f2_bcast(u[6 * r]));
        t = f2_fma(f2_make(-h[s][0].im, h[s][0].re), f2_bcast(u[6 * r + 1]), t);
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          t = f2_fma(f2_make(h[s][k].re, h[s][k].im), f2_bcast(u[6 * r + 2 * k]), t);
          t = f2_fma(f2_make(-h[s][k].im, h[s][k].re), f2_bcast(u[6 * r + 2 * k + 1]), t);
        }
      } else {                           // sum_k conj(U[k][r]) * h[k]
        t = f2_mul(f2_make(h[s][0].re, h[s][0].im), f2_bcast(u[2 * r]));
        t = f2_fma(f2_make(h[s][0].im, -h[s][0].re), f2_bcast(u[2 * r + 1]), t);
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          t = f2_fma(f2_make(h[s][k].re, h[s][k].im), f2_bcast(u[6 * k + 2 * r]), t);
          t = f2_fma(f2_make(h[s][k].im, -h[s][k].re), f2_bcast(u[6 * k + 2 * r + 1]), t);
        }
      }
      w[s][r] = t;
    }
  }
  const f2 cf = f2_bcast(coef), ss = f2_bcast(coef * sigma);
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    float w0r, w0i, w1r, w1i;
    f2_split(w[0][c], w0r, w0i);
    f2_split(w[1][c], w1r, w1i);
    f2_split(f2_fma(cf, w[0][c], f2_make(acc[2 * c], acc[2 * c + 1])), acc[2 * c], acc[2 * c + 1]);
    f2_split(f2_fma(cf, w[1][c], f2_make(acc[6 + 2 * c], acc[6 + 2 * c + 1])), acc[6 + 2 * c], acc[6 + 2 * c + 1]);
    f2_split(f2_fma(ss, unit_pair<(4 - G::c0) % 4>(w0r, w0i), f2_make(acc[6 * G::j0 + 2 * c], acc[6 * G::j0 + 2 * c + 1])),
             acc[6 * G::j0 + 2 * c], acc[6 * G::j0 + 2 * c + 1]);
    f2_split(f2_fma(ss, unit_pair<(4 - G::c1) % 4>(w1r, w1i), f2_make(acc[6 * G::j1 + 2 * c], acc[6 * G::j1 + 2 * c + 1])),
             acc[6 * G::j1 + 2 * c], acc[6 * G::j1 + 2 * c + 1]);
  }
}

template <int MU, bool FWD, typename R>
LQ_DEV void hop_tail_scalar(R* __restrict__ acc, const cx<R> (&h)[2][3], const R* __restrict__ u, R sigma, R coef) {
  typedef GammaRow<MU> G;
  // colour multiply: 6 FMA per real output
  cx<R> w[2][3];
#pragma unroll
  for (int s = 0; s < 2; ++s) {
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      R re, im;
      if (FWD) {                         // sum_k U[r][k] * h[k]
        re = u[6 * r] * h[s][0].re;             im = u[6 * r] * h[s][0].im;
        re = fma_(-u[6 * r + 1], h[s][0].im, re); im = fma_(u[6 * r + 1], h[s][0].re, im);
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          re = fma_(u[6 * r + 2 * k], h[s][k].re, re);      im = fma_(u[6 * r + 2 * k], h[s][k].im, im);
          re = fma_(-u[6 * r + 2 * k + 1], h[s][k].im, re); im = fma_(u[6 * r + 2 * k + 1], h[s][k].re, im);
        }
      } else {                           // sum_k conj(U[k][r]) * h[k]
        re = u[2 * r] * h[s][0].re;             im = u[2 * r] * h[s][0].im;
        re = fma_(u[2 * r + 1], h[s][0].im, re);  im = fma_(-u[2 * r + 1], h[s][0].re, im);
#pragma unroll
        for (int k = 1; k < 3; ++k) {
          re = fma_(u[6 * k + 2 * r], h[s][k].re, re);     im = fma_(u[6 * k + 2 * r], h[s][k].im, im);
          re = fma_(u[6 * k + 2 * r + 1], h[s][k].im, re); im = fma_(-u[6 * k + 2 * r + 1], h[s][k].re, im);
        }
      }
      w[s][r] = {re, im};
    }
  }
  // reconstruct: r_0 = w0, r_1 = w1, r_j0 = sigma*conj(c0)*w0, r_j1 = sigma*conj(c1)*w1
  const R ss = coef * sigma;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    acc[2 * c] = fma_(coef, w[0][c].re, acc[2 * c]);          acc[2 * c + 1] = fma_(coef, w[0][c].im, acc[2 * c + 1]);
    acc[6 + 2 * c] = fma_(coef, w[1][c].re, acc[6 + 2 * c]);  acc[6 + 2 * c + 1] = fma_(coef, w[1][c].im, acc[6 + 2 * c + 1]);
    const cx<R> t0 = unit_mul<(4 - G::c0) % 4>(w[0][c]);
    const cx<R> t1 = unit_mul<(4 - G::c1) % 4>(w[1][c]);
    acc[6 * G::j0 + 2 * c] = fma_(ss, t0.re, acc[6 * G::j0 + 2 * c]); acc[6 * G::j0 + 2 * c + 1] = fma_(ss, t0.im, acc[6 * G::j0 + 2 * c + 1]);
    acc[6 * G::j1 + 2 * c] = fma_(ss, t1.re, acc[6 * G::j1 + 2 * c]); acc[6 * G::j1 + 2 * c + 1] = fma_(ss, t1.im, acc[6 * G::j1 + 2 * c + 1]);
  }
}

template <int MU, bool FWD, typename R>
LQ_DEV void hop_tail(R* __restrict__ acc, const cx<R> (&h)[2][3], const R* __restrict__ u, R sigma, R coef) {
  if constexpr (sizeof(R) == 4) hop_tail_packed<MU, FWD>(acc, h, u, sigma, coef);
  else hop_tail_scalar<MU, FWD, R>(acc, h, u, sigma, coef);
}

// out = C in for one site: two Hermitian 6x6 blocks, 36 reals each: 6 diagonal then the 15
// lower-triangle entries (i>j) at 6 + 2*(i(i-1)/2 + j).  504 flop (PAPER.md:138 fn.1: 72 reals).
template <typename R>
LQ_DEV void clover_block(R* __restrict__ o, const R* __restrict__ x, const R* __restrict__ c) {
  if constexpr (sizeof(R) == 4) {        // packed complex form (core.cuh, f2); same per-component order as below
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      f2 t = f2_mul(f2_make(x[2 * i], x[2 * i + 1]), f2_bcast(c[i]));
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        if (j < i) {
          const float lr = c[6 + 2 * (i * (i - 1) / 2 + j)], li = c[6 + 2 * (i * (i - 1) / 2 + j) + 1];
          t = f2_fma(f2_make(x[2 * j], x[2 * j + 1]), f2_bcast(lr), t);
          t = f2_fma(f2_make(-x[2 * j + 1], x[2 * j]), f2_bcast(li), t);
        } else if (j > i) {
          const float lr = c[6 + 2 * (j * (j - 1) / 2 + i)], li = c[6 + 2 * (j * (j - 1) / 2 + i) + 1];
          t = f2_fma(f2_make(x[2 * j], x[2 * j + 1]), f2_bcast(lr), t);
          t = f2_fma(f2_make(x[2 * j + 1], -x[2 * j]), f2_bcast(li), t);
        }
      }
      f2_split(t, o[2 * i], o[2 * i + 1]);
    }
  } else {
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    R re = c[i] * x[2 * i], im = c[i] * x[2 * i + 1];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      if (j < i) {
        const R lr = c[6 + 2 * (i * (i - 1) / 2 + j)], li = c[6 + 2 * (i * (i - 1) / 2 + j) + 1];
        re = fma_(lr, x[2 * j], re);     re = fma_(-li, x[2 * j + 1], re);
        im = fma_(lr, x[2 * j + 1], im); im = fma_(li, x[2 * j], im);
      } else if (j > i) {
        const R lr = c[6 + 2 * (j * (j - 1) / 2 + i)], li = c[6 + 2 * (j * (j - 1) / 2 + i) + 1];
        re = fma_(lr, x[2 * j], re);     re = fma_(li, x[2 * j + 1], re);
        im = fma_(lr, x[2 * j + 1], im); im = fma_(-li, x[2 * j], im);
      }
    }
    o[2 * i] = re; o[2 * i + 1] = im;
  }
  }
}
template <typename R>
LQ_DEV void clover_mul(R* __restrict__ out, const R* __restrict__ in, const R* __restrict__ cl) {
#pragma unroll
  for (int ch = 0; ch < 2; ++ch) clover_block<R>(out + 12 * ch, in + 12 * ch, cl + 36 * ch);
}

// out = C in with C read from a packed clover field; in half precision the per-site norm is
// applied to the 24 outputs instead of the 72 stored entries.
template <class P>
LQ_DEV void clover_site(typename P::real* __restrict__ out, const typename P::real* __restrict__ in,
                        const char* __restrict__ clov, long long ns, long long idx) {
  typedef typename P::real R;
  R cl[72], sc;
  load_site_raw<P, 72>(cl, sc, clov, ns, idx);
  clover_mul<R>(out, in, cl);
  if constexpr (P::HALF) {
#pragma unroll
    for (int k = 0; k < 24; ++k) out[k] *= sc;
  }
}

// deterministic CTA reduction of NV doubles; result valid in thread 0
template <int NV, int BLOCK>
LQ_DEV void cta_reduce(double* v, double* smem /* [NV][BLOCK/32] */) {
#pragma unroll
  for (int k = 0; k < NV; ++k) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) smem[k * (BLOCK / 32) + wid] = v[k];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double s = 0;
#pragma unroll
      for (int w = 0; w < BLOCK / 32; ++w) s += smem[k * (BLOCK / 32) + w];
      v[k] = s;
    }
  }
}

// The scalar updates of OpBicgOmega / OpBicgAlpha / OpCgAlpha (blas_ops.cuh) for the reductions fused into the
// operator's epilogue; s = (re, im of the dot product, ||out||^2).  Slot numbers: blas.cuh (checked there).
#define LQ_S_RHO 0
#define LQ_S_ALPHA 4
#define LQ_S_OMEGA 6
#define LQ_S_FLAG 11
#define LQ_S_RTV 12
#define LQ_S_TS 14
#define LQ_S_TT 16
LQ_DEV void dots_finalize(double* S, const double* s, int fin) {
  if (fin == 1) {            // omega = <t,s> / <t,t>
    S[LQ_S_TS] = s[0]; S[LQ_S_TS + 1] = s[1]; S[LQ_S_TT] = s[2];
    if (!(s[2] > 0.0)) { S[LQ_S_OMEGA] = 0; S[LQ_S_OMEGA + 1] = 0; S[LQ_S_FLAG] = 2; return; }
    S[LQ_S_OMEGA] = s[0] / s[2]; S[LQ_S_OMEGA + 1] = s[1] / s[2];
  } else if (fin == 2) {     // alpha = rho / <rtilde, v>
    S[LQ_S_RTV] = s[0]; S[LQ_S_RTV + 1] = s[1];
    const double d = s[0] * s[0] + s[1] * s[1];
    if (!(d > 0.0)) { S[LQ_S_FLAG] = 1; S[LQ_S_ALPHA] = 0; S[LQ_S_ALPHA + 1] = 0; return; }
    const double rr = S[LQ_S_RHO], ri = S[LQ_S_RHO + 1];
    S[LQ_S_ALPHA] = (rr * s[0] + ri * s[1]) / d; S[LQ_S_ALPHA + 1] = (ri * s[0] - rr * s[1]) / d;
  } else if (fin == 3) {     // CG on the normal equations: alpha = zz / ||w||^2
    if (!(s[2] > 0.0)) { S[LQ_S_ALPHA] = 0; S[LQ_S_FLAG] = 1; return; }
    S[LQ_S_ALPHA] = S[LQ_S_RHO] / s[2];
  }
}

// ---- epilogue operands staged through freed ring slots (half precision, recon-12, 4-stage ring) ----------------
// The clover block (148 B) and the xpay vector (52 B) of a site are needed only after the 8 hops, and loading them
// then exposes their latency (ncu: long_scoreboard 2.1 per issue in the second launch of Mhat).  From hop 4 on the
// ring slot a thread has just read is not refilled (there is no hop 8), so its private pieces of that slot -- one
// 16-byte and one 8-byte link piece, three 16-byte spinor pieces and the 4-byte norm -- take the epilogue's operands
// instead, by cp.async like everything else: after hop 4 clover chunks 0-3, the first half of chunk 8 and the norm
// (slot 0), after hop 5 chunks 4-7 and the second half of chunk 8 (slot 1), after hop 6 the xpay vector (slot 2).
// Every piece is private to its thread, so no barrier is needed; results are bit-identical to the direct loads.
#ifndef LQ_DSLASH_BLOCK
#define LQ_DSLASH_BLOCK 128
#endif
#define LQ_DSLASH_BLOCK_V LQ_DSLASH_BLOCK
template <int B> struct EpiSlot {
  static constexpr int SLOT = B * 76;
  LQ_DEV static char* p16(char* ring, int s, int j, int tid) {     // j = 0: link piece; 1..3: spinor pieces
    return ring + s * SLOT + (j == 0 ? 0 : 24 * B + 16 * (j - 1) * B) + 16 * tid;
  }
  LQ_DEV static char* p8(char* ring, int s, int tid) { return ring + s * SLOT + 16 * B + 8 * tid; }
  LQ_DEV static char* p4(char* ring, int s, int tid) { return ring + s * SLOT + 72 * B + 4 * tid; }
};
template <int PART, int B>
LQ_DEV void epi_stage_clover(char* ring, int tid, const char* __restrict__ clov, long long ns, long long idx) {
#pragma unroll
  for (int j = 0; j < 4; ++j)
    cp_async<16>(EpiSlot<B>::p16(ring, PART, j, tid), clov + 16ll * (4 * PART + j) * ns + 16ll * idx);
  cp_async<8>(EpiSlot<B>::p8(ring, PART, tid), clov + 16ll * 8 * ns + 16ll * idx + 8 * PART);
  if (PART == 0) cp_async<4>(EpiSlot<B>::p4(ring, 0, tid), clov + 144ll * ns + 4ll * idx);
}
template <int B>
LQ_DEV void epi_stage_y(char* ring, int tid, const char* __restrict__ y, long long ns, long long idx) {
#pragma unroll
  for (int j = 0; j < 3; ++j) cp_async<16>(EpiSlot<B>::p16(ring, 2, j + 1, tid), y + 16ll * j * ns + 16ll * idx);
  cp_async<4>(EpiSlot<B>::p4(ring, 2, tid), y + 48ll * ns + 4ll * idx);
}
// the staged clover block as load_site_raw<PrecH, 72> returns it (integers as floats, scale apart)
template <int B> LQ_DEV void epi_load_clover(float* __restrict__ cl, float& sc, char* ring, int tid) {
  alignas(16) unsigned w[36];
#pragma unroll
  for (int k = 0; k < 8; ++k)
    *reinterpret_cast<int4*>(w + 4 * k) = ld_shared(reinterpret_cast<const int4*>(EpiSlot<B>::p16(ring, k >> 2, k & 3, tid)));
  *reinterpret_cast<int2*>(w + 32) = ld_shared(reinterpret_cast<const int2*>(EpiSlot<B>::p8(ring, 0, tid)));
  *reinterpret_cast<int2*>(w + 34) = ld_shared(reinterpret_cast<const int2*>(EpiSlot<B>::p8(ring, 1, tid)));
  sc = __int_as_float(ld_shared(reinterpret_cast<const int*>(EpiSlot<B>::p4(ring, 0, tid)))) * LQ_FIXED_INV;
#pragma unroll
  for (int k = 0; k < 36; ++k) fixed_pair(w[k], cl[2 * k], cl[2 * k + 1]);
}
// the staged xpay vector as load_site<PrecH, 24> returns it
template <int B> LQ_DEV void epi_load_y(float* __restrict__ yv, char* ring, int tid) {
  alignas(16) unsigned w[12];
#pragma unroll
  for (int k = 0; k < 3; ++k)
    *reinterpret_cast<int4*>(w + 4 * k) = ld_shared(reinterpret_cast<const int4*>(EpiSlot<B>::p16(ring, 2, k + 1, tid)));
  const float sc = __int_as_float(ld_shared(reinterpret_cast<const int*>(EpiSlot<B>::p4(ring, 2, tid)))) * LQ_FIXED_INV;
#pragma unroll
  for (int k = 0; k < 12; ++k) fixed_pair(w[k], yv[2 * k], yv[2 * k + 1]);
#pragma unroll
  for (int k = 0; k < 24; ++k) yv[k] *= sc;
}

// Fused epilogue of one site (shared by the single- and multi-right-hand-side kernels):
//   XPAY: acc = [A] y + coef * acc (CLOVX: A = clover block of the site);  CLOVOUT: acc = C acc;
//   XPAY && CLOVX && CLOVOUT: acc = y + coef * C acc (symmetric even-odd form);
//   DOTS 1, 2: d0 + i d1 += <acc, y>, d2 += <acc, acc> for this site; DOTS 3: d0 + i d1 += <q, acc> (only with CLOVX).
// STG_C / STG_Y: the clover block / the xpay vector were staged in the ring (EpiSlot above) instead of being loaded here.
template <class P, bool XPAY, bool CLOVX, bool CLOVOUT, int DOTS, bool STG_C = false, bool STG_Y = false>
LQ_DEV void dslash_epilogue(typename P::real* __restrict__ acc, const char* __restrict__ y, const char* __restrict__ clov_y,
                            const char* __restrict__ clov_out, double coef_d, int p, long long ns, long long idx,
                            typename P::real& d0, typename P::real& d1, typename P::real& d2,
                            char* ring = nullptr, int tid = 0) {
  typedef typename P::real R;
  if constexpr (XPAY && CLOVX && CLOVOUT) {
    // symmetric even-odd form, second half: acc = y + coef * C acc
    R t[24], yv[24];
    clover_site<P>(t, acc, clov_out + (long long)p * site_bytes<P>(72, true) * ns, ns, idx);
    load_site<P, 24>(yv, y, ns, idx);
    const R coef = (R)coef_d;
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = fma_(coef, t[k], yv[k]);
    return;
  }
  if constexpr (XPAY) {
    R yv[24];
    if constexpr (STG_Y) epi_load_y<LQ_DSLASH_BLOCK_V>(yv, ring, tid);
    else load_site<P, 24>(yv, y, ns, idx);
    const R coef = (R)coef_d;
    if constexpr (CLOVX) {
      // r = A y + coef * acc, one chiral block at a time so that y, A y and the clover block
      // die early (the DOTS variant needs y for the partial sums as well)
      R cl[72], sc;
      if constexpr (STG_C) epi_load_clover<LQ_DSLASH_BLOCK_V>(cl, sc, ring, tid);
      else load_site_raw<P, 72>(cl, sc, clov_y + (long long)p * site_bytes<P>(72, true) * ns, ns, idx);
#pragma unroll
      for (int ch = 0; ch < 2; ++ch) {
        R ay[12];
        clover_block<R>(ay, yv + 12 * ch, cl + 36 * ch);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
          if constexpr (P::HALF) ay[k] *= sc;
          acc[12 * ch + k] = fma_(coef, acc[12 * ch + k], ay[k]);
        }
        if constexpr (DOTS == 1 || DOTS == 2) {
#pragma unroll
          for (int k = 0; k < 6; ++k) {
            const R rr = acc[12 * ch + 2 * k], ri = acc[12 * ch + 2 * k + 1];
            const R yr = yv[12 * ch + 2 * k], yi = yv[12 * ch + 2 * k + 1];
            d0 = fma_(rr, yr, d0); d0 = fma_(ri, yi, d0);
            d1 = fma_(rr, yi, d1); d1 = fma_(-ri, yr, d1);
            d2 = fma_(rr, rr, d2); d2 = fma_(ri, ri, d2);
          }
        }
      }
      if constexpr (DOTS == 3) {
        // d0 + i d1 += <q, acc> with a third vector q (BiCGstab: <rtilde, v>); its pointer travels in clov_out,
        // which this epilogue does not use
        R q[24];
        load_site<P, 24>(q, clov_out, ns, idx);
#pragma unroll
        for (int k = 0; k < 12; ++k) {
          const R rr = acc[2 * k], ri = acc[2 * k + 1];
          d0 = fma_(q[2 * k], rr, d0); d0 = fma_(q[2 * k + 1], ri, d0);
          d1 = fma_(q[2 * k], ri, d1); d1 = fma_(-q[2 * k + 1], rr, d1);
          d2 = fma_(rr, rr, d2); d2 = fma_(ri, ri, d2);
        }
      }
    } else {
#pragma unroll
      for (int k = 0; k < 24; ++k) acc[k] = fma_(coef, acc[k], yv[k]);
    }
  }
  if constexpr (CLOVOUT) {
    R t[24];
    if constexpr (STG_C) {
      R cl[72], sc;
      epi_load_clover<LQ_DSLASH_BLOCK_V>(cl, sc, ring, tid);
      clover_mul<R>(t, acc, cl);
#pragma unroll
      for (int k = 0; k < 24; ++k) t[k] *= sc;
    } else {
      clover_site<P>(t, acc, clov_out + (long long)p * site_bytes<P>(72, true) * ns, ns, idx);
    }
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = t[k];
  }
}

#ifndef LQ_DSLASH_BLOCK
#define LQ_DSLASH_BLOCK 128
#endif
// minimum resident CTAs per SM for the fp32-arithmetic kernels: 5 (96 registers, 20 warps/SM).
// Measured at 32^3x64 in bursts at full clock, 6 / 5 / 4 CTAs: Mhat fp32 r12 302.7 / 296.2 / 300.1 us,
// Mhat half r12 234.4 / 228.3 / 233.0 us, Dslash fp32 r12 97.7 / 97.5 / 100.2 us.  At 6 (80 registers)
// the clover-epilogue variants spill 60-230 bytes per thread, and with the L1 carved out for the
// staging ring those spills miss L1 (ncu: 3 % hit rate) and travel to L2: the MR-step kernel lost
// 30 us of 150 to them.
// fp64: 3 CTAs/SM (168 registers), except the recon-12 clover-epilogue variants, which spill 40-90 bytes at 3 and
// keep 2.  Measured at 32^3x64 (2 -> 3 CTAs/SM): Dslash r18 247 -> 245, r12 211 -> 191.5, r8 283 -> 270 us;
// Mhat r18 696 -> 691, r8 796 -> 679, r12 601 -> 614 us (hence the exception).
#ifndef LQ_DSLASH_MINB64
#define LQ_DSLASH_MINB64 3
#endif
#ifndef LQ_DSLASH_MINB64_CLOV12
#define LQ_DSLASH_MINB64_CLOV12 2
#endif
#ifndef LQ_DSLASH_MINB
#define LQ_DSLASH_MINB 5
#endif

template <class P, int RECON, bool CLOVX, bool CLOVOUT> constexpr int dslash_minb() {
  if (sizeof(typename P::real) != 8) return LQ_DSLASH_MINB;
  return ((CLOVX || CLOVOUT) && RECON == 12) ? LQ_DSLASH_MINB64_CLOV12 : LQ_DSLASH_MINB64;
}

// bytes of one staging buffer (one hop of every thread of the CTA): link + neighbour spinor (+ norm)
template <class P, int RECON> struct HopStage {
  static constexpr int LINK_B = RECON * (int)sizeof(typename P::store_t);
  static constexpr int SPIN_B = site_bytes<P>(24, true);
  static constexpr int BYTES = LQ_DSLASH_BLOCK * (LINK_B + SPIN_B);
};

// NST = 0: neighbour data is loaded straight into registers (fp64).
// NST > 0: software pipeline over the 8 hops through NST per-thread staging buffers in shared
// memory filled by cp.async: while hop h is computed, the loads of hops h+1 .. h+NST-1 are in
// flight without holding registers.  The slots are private to a thread, so no CTA barrier is
// needed: cp.async.wait_group orders a thread's own copies.
// DAG: -1 = dagger read from the arguments at run time (fp64, fp32); 0 / 1 = compile-time dagger (half precision:
// the fixed-point projection fused with the decode needs the sign of every combination at compile time).
template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int DOTS, int NST, int DAG = -1>
__global__ void __launch_bounds__(LQ_DSLASH_BLOCK, (dslash_minb<P, RECON, CLOVX, CLOVOUT>()))
dslash_kernel(const DslashArgs a) {
  static_assert(P::HALF ? (DAG == 0 || DAG == 1) : DAG == -1, "compile-time dagger for half precision only");
  typedef typename P::real R;
  // epilogue operands through the ring (EpiSlot): half precision, recon-12 (16 + 8 byte link pieces), 4-stage ring
#ifdef LQ_NO_EPI_STAGE
  constexpr bool STG_OK = false;
#else
  constexpr bool STG_OK = P::HALF && RECON == 12 && NST == 4 && !(XPAY && CLOVX && CLOVOUT);
#endif
  constexpr bool STG_C = STG_OK && (CLOVX != CLOVOUT), STG_Y = STG_OK && XPAY;
  const Geom& g = a.g;
  const int cb = (DOTS ? 0 : a.range.cb0) + blockIdx.x * LQ_DSLASH_BLOCK + threadIdx.x;
  const int box = blockIdx.y + (a.parity >> 8);            // first box of the launch: Schwarz block groups (solver.cu)
  const bool active = cb < (DOTS ? g.vh : a.range.cb1);
  R d0 = 0, d1 = 0, d2 = 0;                 // DOTS: this site's <r,y> (re, im) and <r,r>
  if (active) {
    const long long base = (long long)box * g.vh;
    const long long idx = base + cb;
    const int p = a.parity & 1;
    int c[4];
    cb_to_coords(g, cb, p, c);
    const int xh = c[0] >> 1;
    const int rp = c[0] & 1;                 // row parity: x = 2*xh + rp
    const long long link_bytes = (long long)RECON * sizeof(typename P::store_t) * g.ns;
    const char* g_out = a.gauge + (long long)(p * 4) * link_bytes;        // links living on output-parity sites
    const char* g_in = a.gauge + (long long)((1 - p) * 4) * link_bytes;   // links living on input-parity sites
    const R sig_f = (a.dagger & 1) ? R(1) : R(-1);  // forward hop: (1 - g) for D, (1 + g) for D^dagger
    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;

    // neighbour checkerboard indices
    int nf[4], nbk[4];
    {
      const int xf = rp ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh;
      const int xb = rp ? xh : (xh == 0 ? g.Xh - 1 : xh - 1);
      nf[0] = cb - xh + xf;
      nbk[0] = cb - xh + xb;
      const int sy = g.Xh, sz = g.Xh * g.X[1], st = g.Xh * g.X[1] * g.X[2];
      nf[1] = (c[1] + 1 == g.X[1]) ? cb - (g.X[1] - 1) * sy : cb + sy;
      nbk[1] = (c[1] == 0) ? cb + (g.X[1] - 1) * sy : cb - sy;
      nf[2] = (c[2] + 1 == g.X[2]) ? cb - (g.X[2] - 1) * sz : cb + sz;
      nbk[2] = (c[2] == 0) ? cb + (g.X[2] - 1) * sz : cb - sz;
      nf[3] = (c[3] + 1 == g.X[3]) ? cb - (g.X[3] - 1) * st : cb + st;
      nbk[3] = (c[3] == 0) ? cb + (g.X[3] - 1) * st : cb - st;
    }

    if constexpr (NST == 0) {
    // a hop that crosses an open (Dirichlet) boundary gets coefficient 0; its loads stay inside
    // the box (wrapped index), so no branch is needed and the hops can be scheduled freely
#define LQ_HOP(MU)                                                                              \
    {                                                                                           \
      const R sf = (c[MU] + 1 == g.X[MU]) ? (R)g.bc[MU] : R(1);                                 \
      {                                                        \
        R u[18], psi[24], us, ps;                                                               \
        load_link<P, RECON>(u, us, g_out + MU * link_bytes, g.ns, idx);                         \
        load_site_raw<P, 24>(psi, ps, a.in, g.ns, base + nf[MU]);                               \
        hop<MU, true, R>(acc, psi, u, sig_f, P::HALF ? sf * us * ps : sf);                      \
      }                                                                                         \
      const R sb = (c[MU] == 0) ? (R)g.bc[MU] : R(1);                                           \
      {                                                        \
        R u[18], psi[24], us, ps;                                                               \
        load_link<P, RECON>(u, us, g_in + MU * link_bytes, g.ns, base + nbk[MU]);               \
        load_site_raw<P, 24>(psi, ps, a.in, g.ns, base + nbk[MU]);                              \
        hop<MU, false, R>(acc, psi, u, -sig_f, P::HALF ? sb * us * ps : sb);                    \
      }                                                                                         \
    }
    LQ_HOP(0) LQ_HOP(1) LQ_HOP(2) LQ_HOP(3)
#undef LQ_HOP
    } else {
      extern __shared__ __align__(16) char lq_stage[];
      typedef HopStage<P, RECON> HS;
      const int tid = threadIdx.x;
      const char* epi_clov = (CLOVX ? a.clov_y : a.clov_out) + (long long)p * site_bytes<P>(72, true) * g.ns;
      (void)epi_clov;
      // hop h: mu = h/2, forward for even h.  Issue = start the async copies of its link and spinor.
#define LQ_ISSUE(H)                                                                                        \
      {                                                                                                    \
        constexpr int MU_ = (H) / 2;                                                                       \
        constexpr bool FW_ = ((H) & 1) == 0;                                                               \
        char* sb_ = lq_stage + ((H) % NST) * HS::BYTES;                                                    \
        const long long li_ = FW_ ? idx : base + nbk[MU_];                                                 \
        const long long si_ = FW_ ? base + nf[MU_] : base + nbk[MU_];                                      \
        Rec<typename P::store_t, RECON>::stage(sb_, LQ_DSLASH_BLOCK, tid, (FW_ ? g_out : g_in) + MU_ * link_bytes, g.ns, li_); \
        char* ss_ = sb_ + LQ_DSLASH_BLOCK * HS::LINK_B;                                                    \
        Rec<typename P::store_t, 24>::stage(ss_, LQ_DSLASH_BLOCK, tid, a.in, g.ns, si_);                   \
        if (P::HALF) cp_async<4>(ss_ + 48 * LQ_DSLASH_BLOCK + 4 * tid, reinterpret_cast<const float*>(a.in + 48ll * g.ns) + si_); \
      }
#define LQ_PHOP(H)                                                                                         \
      {                                                                                                    \
        constexpr int MU_ = (H) / 2;                                                                       \
        constexpr bool FW_ = ((H) & 1) == 0;                                                               \
        cp_async_wait<NST - 1>();                                                                          \
        const char* sb_ = lq_stage + ((H) % NST) * HS::BYTES;                                              \
        R u[18], psi[24], us, ps;                                                                          \
        load_link<P, RECON, 2>(u, us, sb_, LQ_DSLASH_BLOCK, tid);                                          \
        if constexpr (P::HALF) load_site_magic<P, 24, 2>(psi, ps, sb_ + LQ_DSLASH_BLOCK * HS::LINK_B, LQ_DSLASH_BLOCK, tid); \
        else load_site_raw<P, 24, 2>(psi, ps, sb_ + LQ_DSLASH_BLOCK * HS::LINK_B, LQ_DSLASH_BLOCK, tid);   \
        if ((H) + NST < 8) LQ_ISSUE(((H) + NST) % 8)                                                       \
        /* slots that are not refilled take the epilogue's operands (EpiSlot) */                           \
        if constexpr (STG_C) {                                                                             \
          if ((H) == 4) epi_stage_clover<0, LQ_DSLASH_BLOCK>(lq_stage, tid, epi_clov, g.ns, idx);           \
          if ((H) == 5) epi_stage_clover<1, LQ_DSLASH_BLOCK>(lq_stage, tid, epi_clov, g.ns, idx);           \
        }                                                                                                  \
        if constexpr (STG_Y) { if ((H) == 6) epi_stage_y<LQ_DSLASH_BLOCK>(lq_stage, tid, a.y, g.ns, idx); } \
        cp_async_commit();                                                                                 \
        const R sg_ = FW_ ? ((c[MU_] + 1 == g.X[MU_]) ? (R)g.bc[MU_] : R(1)) : ((c[MU_] == 0) ? (R)g.bc[MU_] : R(1)); \
        if constexpr (P::HALF) hop_fixed<MU_, FW_, (FW_ == (DAG == 1)) ? 1 : -1>(acc, psi, u, sg_ * us * ps); \
        else hop<MU_, FW_, R>(acc, psi, u, FW_ ? sig_f : -sig_f, sg_);                                     \
      }
#pragma unroll
      for (int h = 0; h < NST; ++h) {
        switch (h) {                       // NST <= 4
          case 0: LQ_ISSUE(0) break;
          case 1: LQ_ISSUE(1) break;
          case 2: LQ_ISSUE(2) break;
          default: LQ_ISSUE(3) break;
        }
        cp_async_commit();
      }
      LQ_PHOP(0) LQ_PHOP(1) LQ_PHOP(2) LQ_PHOP(3) LQ_PHOP(4) LQ_PHOP(5) LQ_PHOP(6) LQ_PHOP(7)
#undef LQ_PHOP
#undef LQ_ISSUE
    }

    if constexpr (STG_C || STG_Y) {
      extern __shared__ __align__(16) char lq_stage[];
      cp_async_wait<0>();
      dslash_epilogue<P, XPAY, CLOVX, CLOVOUT, DOTS, STG_C, STG_Y>(acc, a.y, a.clov_y, a.clov_out, a.a, p, g.ns, idx, d0, d1, d2,
                                                                     lq_stage, threadIdx.x);
    } else {
      dslash_epilogue<P, XPAY, CLOVX, CLOVOUT, DOTS>(acc, a.y, a.clov_y, a.clov_out, a.a, p, g.ns, idx, d0, d1, d2);
    }
    store_site<P, 24>(acc, a.out, g.ns, idx);
  }
  if constexpr (DOTS >= 2) {
    // Solver reductions fused into the operator ("BLAS1 ... extremely bandwidth
    // intensive"): CTA sums -> per-CTA partials; dots_finalize_kernel (blas.cu), launched behind this kernel, adds them
    // in a fixed order (bit-reproducible) and updates the Krylov scalars on the device.  a.dots = workspace W:
    // W[0] = address of the scalar array S, W[8 + 3 i ..] = partials of CTA i.  The CTA writes and leaves: a fence +
    // arrival counter + last-CTA sum here (round 2's first form) kept every CTA resident ~1.5 us longer, which cost
    // the fp32 solver 5 % (measured).
    __shared__ double sm[3 * (LQ_DSLASH_BLOCK / 32)];
    double red[3] = {(double)d0, (double)d1, (double)d2};
    cta_reduce<3, LQ_DSLASH_BLOCK>(red, sm);
    if (threadIdx.x == 0) {
      double* part = a.dots + 8 + 3ll * blockIdx.x;
      part[0] = red[0]; part[1] = red[1]; part[2] = red[2];
    }
  }
  if constexpr (DOTS == 1) {
    // per-warp partial sums (sites in fp64, fixed shuffle order: deterministic); no CTA barrier.
    // The MR update kernel adds the gridDim.x * (LQ_DSLASH_BLOCK/32) partials of its box.
    double red[3] = {(double)d0, (double)d1, (double)d2};
#pragma unroll
    for (int k = 0; k < 3; ++k) {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) red[k] += __shfl_down_sync(0xffffffffu, red[k], o);
    }
    if ((threadIdx.x & 31) == 0) {
      double* d = a.dots + (((long long)box * gridDim.x + blockIdx.x) * (LQ_DSLASH_BLOCK / 32) + (threadIdx.x >> 5)) * 4;
      d[0] = red[0]; d[1] = red[1]; d[2] = red[2]; d[3] = 0;
    }
  }
}

// Epilogue selector used by the host dispatch
enum DslashEpi {
  EPI_NONE = 0,       // out = D in
  EPI_CLOVOUT = 1,    // out = C (D in)
  EPI_CLOVX_XPAY = 2, // out = A y + a D in
  EPI_XPAY = 3,       // out = y + a D in
  EPI_XPAY_CLOVOUT = 4, // out = C (y + a D in)
  EPI_CLOVX_XPAY_DOTS = 5, // EPI_CLOVX_XPAY + per-box <out,y>, <out,out>
  EPI_XPAY_CLOVD = 6,      // out = y + a C (D in)   (symmetric even-odd form)
  EPI_CLOVX_XPAY_YDOT = 7, // EPI_CLOVX_XPAY + global <out,y>, <out,out> and a scalar update (dots_finalize_kernel)
  EPI_CLOVX_XPAY_QDOT = 8  // EPI_CLOVX_XPAY + global <q,out>, <out,out> (q in DslashArgs::clov_out) and a scalar update
};

// scalar updates the fused reductions can perform (argument of dots_finalize_kernel, blas.cu)
enum DotsFin { FIN_NONE = 0, FIN_BICG_OMEGA = 1, FIN_BICG_ALPHA = 2, FIN_CG_ALPHA = 3 };

template <class P> cudaError_t launch_dslash(const DslashArgs& a, int recon, int epi, cudaStream_t s);

}  // namespace lq
