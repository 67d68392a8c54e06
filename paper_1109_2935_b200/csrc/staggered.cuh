// staggered.cuh -- improved staggered (asqtad) hopping term.
//
//   (D chi)(x) = sum_mu eta_mu(x) [ fat_mu(x) chi(x+mu) - fat_mu(x-mu)^dag chi(x-mu)
//                                 + lng_mu(x) chi(x+3mu) - lng_mu(x-3mu)^dag chi(x-3mu) ]
//
// PAPER.md:114-122 (Sec. 2.3, Eq. 3) in the reading R13-R15 of DESIGN.md: staggered phases eta_mu
// and the minus sign of the backward hops explicit (Eq. 3 as printed is not anti-Hermitian, which
// PAPER.md:130 requires), fat and long links given ("precalculated"), boundary sign on
// every hop that wraps.  chi is a 3-component colour vector per site (6 reals, Fig. 2).
//
// Layout.  Links: [parity][mu] records of 18 reals in the chunked SoA of core.cuh (no compression:
// fat links are sums of paths, not unitary).  Colour vectors: four consecutive sites of a parity form
// one 24-real record of the same chunked SoA as a Wilson spinor (site cb -> record cb/4, complex
// component i -> pair 3*(cb%4)+i), so every fused BLAS-1 kernel of blas_ops.cuh works on staggered
// fields unchanged with ns = Vh/4 records.  A thread reads a neighbour's vector with three 16-byte
// (fp64) or 8-byte (fp32) loads; a warp's loads cover whole 128-byte lines.
//
// One thread per output site, 16 hops, each link read exactly once per application: compulsory
// bytes per site = 16 links + 2 vectors = 16*72 + 48 = 1200 B in fp32 (2400 B in fp64; 1008 / 2016 B when the long
// links are stored as 12 reals), 1146 flop
// (16 x 66 for the 3x3 complex matvecs + 15 x 6 adds): HBM-bound at ~1 flop/byte.
#pragma once
#include "core.cuh"

namespace lq {

struct StagArgs {
  Geom g;               // whole lattice, ns = Vh
  char* out;            // packed colour field, output parity
  const char* in;       // packed colour field, input parity
  const char* y;        // XPAY operand (output parity) or nullptr
  const char* fat;      // [parity][mu] x 18 reals
  const char* lng;
  double a, b;          // XPAY: out = a*y + b*(D in); else out = D in
  double linv;          // LRECON == 12: 1 / long_scale (third row of a long link = conj(row0 x row1) * linv)
  int parity;           // output parity
};

template <class P> struct Colour {
  typedef typename P::real R;
  static_assert(!P::HALF, "staggered fields are stored in fp64 or fp32 (PAPER.md:298 fn. 3)");
  LQ_DEV static const char* slot(const char* f, long long ns4, long long cb, int i) {
    const long long j = cb >> 2;
    const int s = 3 * (int)(cb & 3) + i;
    if (sizeof(R) == 8) return f + 16ll * s * ns4 + 16ll * j;
    return f + 16ll * (s >> 1) * ns4 + 16ll * j + 8 * (s & 1);
  }
  LQ_DEV static void load(R* __restrict__ v, const char* __restrict__ f, long long ns4, long long cb) {
    LQ_CHECK_INDEX(cb, 4 * ns4);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      if constexpr (sizeof(R) == 8) {
        const double2 t = __ldg(reinterpret_cast<const double2*>(slot(f, ns4, cb, i)));
        v[2 * i] = t.x; v[2 * i + 1] = t.y;
      } else {
        const float2 t = __ldg(reinterpret_cast<const float2*>(slot(f, ns4, cb, i)));
        v[2 * i] = t.x; v[2 * i + 1] = t.y;
      }
    }
  }
  LQ_DEV static void store(const R* __restrict__ v, char* __restrict__ f, long long ns4, long long cb) {
    LQ_CHECK_INDEX(cb, 4 * ns4);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      char* p = const_cast<char*>(slot(f, ns4, cb, i));
      if constexpr (sizeof(R) == 8) *reinterpret_cast<double2*>(p) = make_double2(v[2 * i], v[2 * i + 1]);
      else *reinterpret_cast<float2*>(p) = make_float2(v[2 * i], v[2 * i + 1]);
    }
  }
};

// acc += coef * W chi,  W = U (FWD) or U^dagger
template <bool FWD, typename R>
LQ_DEV void su3_mac(R* __restrict__ acc, const R* __restrict__ u, const R* __restrict__ chi, R coef) {
#pragma unroll
  for (int r = 0; r < 3; ++r) {
    R re = 0, im = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const R ur = FWD ? u[6 * r + 2 * k] : u[6 * k + 2 * r];
      const R ui = FWD ? u[6 * r + 2 * k + 1] : -u[6 * k + 2 * r + 1];
      re = fma_(ur, chi[2 * k], re);     re = fma_(-ui, chi[2 * k + 1], re);
      im = fma_(ur, chi[2 * k + 1], im); im = fma_(ui, chi[2 * k], im);
    }
    acc[2 * r] = fma_(coef, re, acc[2 * r]);
    acc[2 * r + 1] = fma_(coef, im, acc[2 * r + 1]);
  }
}

#define LQ_STAG_BLOCK 128

// 18 reals of a link: as stored (N == 18), or rows 0,1 stored and row 2 = conj(row0 x row1) * linv (N == 12;
// long links that are long_scale x SU(3), as the three-link Naik term of asqtad is: PAPER.md:164 (a), :122)
template <typename R, int N>
LQ_DEV void load_stag_link(R* __restrict__ u, const char* __restrict__ f, long long ns, long long i, R linv) {
  Rec<R, N>::template load<LQ_GAUGE_STREAM>(u, f, ns, i);
  if constexpr (N == 12) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int j = (c + 1) % 3, k = (c + 2) % 3;
      R re = u[2 * j] * u[6 + 2 * k];
      re = fma_(-u[2 * j + 1], u[6 + 2 * k + 1], re);
      re = fma_(-u[2 * k], u[6 + 2 * j], re);
      re = fma_(u[2 * k + 1], u[6 + 2 * j + 1], re);
      R im = u[2 * k] * u[6 + 2 * j + 1];
      im = fma_(u[2 * k + 1], u[6 + 2 * j], im);
      im = fma_(-u[2 * j], u[6 + 2 * k + 1], im);
      im = fma_(-u[2 * j + 1], u[6 + 2 * k], im);
      u[12 + 2 * c] = re * linv;
      u[12 + 2 * c + 1] = im * linv;
    }
  }
}

template <class P, bool XPAY, int LRECON>
__global__ void __launch_bounds__(LQ_STAG_BLOCK) stag_dslash_kernel(const StagArgs a) {
  typedef typename P::real R;
  const Geom& g = a.g;
  const int cb = blockIdx.x * LQ_STAG_BLOCK + threadIdx.x;
  if (cb >= g.vh) return;
  const int p = a.parity;
  const long long ns4 = g.ns >> 2;
  int c[4];
  cb_to_coords(g, cb, p, c);
  const long long fat_bytes = 18ll * sizeof(R) * g.ns, lng_bytes = (long long)LRECON * sizeof(R) * g.ns;
  const R linv = (R)a.linv;
  R acc[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    int e = 0;
#pragma unroll
    for (int nu = 0; nu < mu; ++nu) e += c[nu];
    const R eta = (e & 1) ? R(-1) : R(1);
#pragma unroll
    for (int kind = 0; kind < 2; ++kind) {               // 0: fat link, one hop; 1: long link, three hops
      const int step = kind ? 3 : 1;
      const char* links = kind ? a.lng : a.fat;
      const long long link_bytes = kind ? lng_bytes : fat_bytes;
      int d[4] = {c[0], c[1], c[2], c[3]};
      {                                                   // forward: link of this site, chi(x + step mu)
        int v = c[mu] + step;
        R sg = eta;
        if (v >= g.X[mu]) { v -= g.X[mu]; sg *= (R)g.bc[mu]; }
        d[mu] = v;
        const int nb = coords_to_cb(g, d);
        R u[18], chi[6];
        if (kind) load_stag_link<R, LRECON>(u, links + (long long)(p * 4 + mu) * link_bytes, g.ns, cb, linv);
        else load_stag_link<R, 18>(u, links + (long long)(p * 4 + mu) * link_bytes, g.ns, cb, linv);
        Colour<P>::load(chi, a.in, ns4, nb);
        su3_mac<true, R>(acc, u, chi, sg);
      }
      {                                                   // backward: link of the neighbour, chi(x - step mu)
        int v = c[mu] - step;
        R sg = -eta;
        if (v < 0) { v += g.X[mu]; sg *= (R)g.bc[mu]; }
        d[mu] = v;
        const int nb = coords_to_cb(g, d);
        R u[18], chi[6];
        if (kind) load_stag_link<R, LRECON>(u, links + (long long)((1 - p) * 4 + mu) * link_bytes, g.ns, nb, linv);
        else load_stag_link<R, 18>(u, links + (long long)((1 - p) * 4 + mu) * link_bytes, g.ns, nb, linv);
        Colour<P>::load(chi, a.in, ns4, nb);
        su3_mac<false, R>(acc, u, chi, sg);
      }
    }
  }
  if constexpr (XPAY) {
    R yv[6];
    Colour<P>::load(yv, a.y, ns4, cb);
    const R ca = (R)a.a, cbb = (R)a.b;
#pragma unroll
    for (int k = 0; k < 6; ++k) acc[k] = fma_(cbb, acc[k], ca * yv[k]);
  }
  Colour<P>::store(acc, a.out, ns4, cb);
}

}  // namespace lq
