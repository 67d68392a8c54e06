// dslash_mrhs.cuh -- the hopping term applied to several right-hand sides per launch.
//
// Same operator and same fused epilogues as dslash.cuh (Eq. 2), for NRHS
// spinor fields that share one gauge field.  Motivation: a
// link is read exactly once per application and cannot be reused by other sites, so on B200 the
// 8 links are 2/3 of the compulsory bytes of a single-source Dslash (384 of 576 B/site in
// fp32/recon-12) and their reconstruction + fixed-point decode a quarter of the instructions of
// the issue-bound half-precision kernel.  Sharing the links between right-hand sides is the one
// lever that raises the arithmetic intensity.
//
// A CTA owns 32 consecutive sites of one parity and 4 right-hand sides: warp w computes
// right-hand side blockIdx.z*4 + w on lane = site.  Phase 1: warp w loads, decodes and
// reconstructs the two links of direction mu = w (forward: link of the site; backward: link of
// the neighbour) for the CTA's 32 sites and writes all 18 reals to shared memory, while every
// thread already has the neighbour spinors of its first hops in flight (cp.async ring as in
// dslash.cuh).  Phase 2 (after one CTA barrier): every warp runs the 8 hops with links read from
// shared memory.  Per right-hand side a thread loads and reconstructs 2 links instead of 8.
#pragma once
#include "dslash.cuh"

namespace lq {

// NR = right-hand sides per CTA = warps per CTA = 4: warp w reconstructs both links of direction w.
// (8 per CTA, one link per warp, and a register prefetch of the next hop's spinor instead of the
// cp.async ring were measured and are slower: 83 and 99 us against 79 us per right-hand side for
// the fp32/recon-12 Dslash at 32^3x64.)

// reconstructed links of one CTA in shared memory: [hop][chunk][lane], 18 reals per link as
// 16-byte chunks plus one 8-byte chunk in fp32 (72 bytes; fp64: 144 bytes = 9 chunks)
template <typename R> struct LinkTile {
  static constexpr int N16 = 18 * (int)sizeof(R) / 16, N8 = (18 * (int)sizeof(R) % 16) / 8;
  static constexpr int E16 = 16 / (int)sizeof(R);
  static constexpr int HOP_B = 32 * 18 * (int)sizeof(R);
  static constexpr int BYTES = 8 * HOP_B;
  LQ_DEV static void put(char* tile, int hop, int lane, const R* __restrict__ u) {
    char* t = tile + hop * HOP_B;
#pragma unroll
    for (int k = 0; k < N16; ++k) {
      alignas(16) R v[E16];
#pragma unroll
      for (int e = 0; e < E16; ++e) v[e] = u[k * E16 + e];
      *reinterpret_cast<int4*>(t + (k * 32 + lane) * 16) = *reinterpret_cast<const int4*>(v);
    }
    if (N8) {
      alignas(8) R v[2] = {u[N16 * E16], u[N16 * E16 + 1]};
      *reinterpret_cast<int2*>(t + N16 * 32 * 16 + lane * 8) = *reinterpret_cast<const int2*>(v);
    }
  }
  LQ_DEV static void get(const char* tile, int hop, int lane, R* __restrict__ u) {
    const char* t = tile + hop * HOP_B;
#pragma unroll
    for (int k = 0; k < N16; ++k) {
      alignas(16) R v[E16];
      *reinterpret_cast<int4*>(v) = ld_shared(reinterpret_cast<const int4*>(t + (k * 32 + lane) * 16));
#pragma unroll
      for (int e = 0; e < E16; ++e) u[k * E16 + e] = v[e];
    }
    if (N8) {
      alignas(8) R v[2];
      *reinterpret_cast<int2*>(v) = ld_shared(reinterpret_cast<const int2*>(t + N16 * 32 * 16 + lane * 8));
      u[N16 * E16] = v[0]; u[N16 * E16 + 1] = v[1];
    }
  }
};

template <class P, int NR> struct SpinStage {
  static constexpr int SPIN_B = site_bytes<P>(24, true);
  static constexpr int BYTES = 32 * NR * SPIN_B;
};

// minimum resident CTAs per SM: fp64 2, fp32 4 (128 registers), half 5 (96 registers) -- measured best
template <class P> struct MrhsMinB { static constexpr int V = sizeof(typename P::real) == 8 ? 2 : (P::HALF ? 5 : 4); };

// a.in / a.out / a.y hold nrhs packed fields back to back (field r at r * bytes of one field);
// a.dagger carries nrhs in bits 8.. (the argument struct must stay 128 bytes, dslash.cuh).
// DAG: as in dslash_kernel (-1 run-time dagger for fp64 / fp32, 0 / 1 compile-time for half precision)
template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int NST, int NR, int DAG = -1>
__global__ void __launch_bounds__(32 * NR, MrhsMinB<P>::V)
dslash_mrhs_kernel(const DslashArgs a) {
  typedef typename P::real R;
  static_assert(P::HALF ? (DAG == 0 || DAG == 1) : DAG == -1, "compile-time dagger for half precision only");
  static_assert(NST >= 1 && NST <= 4, "spinor ring depth");
  static_assert(NR == 4, "right-hand sides per CTA = directions");
  constexpr int LQ_MRHS_BLOCK = 32 * NR;
  const Geom& g = a.g;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, tid = threadIdx.x;
  const int cb = a.range.cb0 + blockIdx.x * 32 + lane;
  const int box = blockIdx.y;
  const int nrhs = a.dagger >> 8, dagger = a.dagger & 1;
  const int rhs = blockIdx.z * NR + w;
  const bool site_ok = cb < a.range.cb1;
  const bool active = site_ok && rhs < nrhs;
  extern __shared__ __align__(16) char lq_smem[];
  char* tile = lq_smem;
  char* ring = lq_smem + LinkTile<R>::BYTES;

  const long long base = (long long)box * g.vh;
  const long long idx = base + cb;
  const int p = a.parity;
  const long long fbytes = (long long)site_bytes<P>(24, true) * g.ns;      // one packed field
  const char* in = a.in + (long long)rhs * fbytes;
  int c[4] = {0, 0, 0, 0}, nf[4] = {0, 0, 0, 0}, nbk[4] = {0, 0, 0, 0};
  if (site_ok) {
    cb_to_coords(g, cb, p, c);
    const int xh = c[0] >> 1, rp = c[0] & 1;
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

  // hop h: mu = h/2, forward for even h.  Issue = start the async copy of its neighbour spinor.
#define LQ_ISSUE(H)                                                                                        \
  {                                                                                                        \
    constexpr int MU_ = (H) / 2;                                                                           \
    constexpr bool FW_ = ((H) & 1) == 0;                                                                   \
    char* ss_ = ring + ((H) % NST) * SpinStage<P, NR>::BYTES;                                              \
    const long long si_ = FW_ ? base + nf[MU_] : base + nbk[MU_];                                          \
    Rec<typename P::store_t, 24>::stage(ss_, LQ_MRHS_BLOCK, tid, in, g.ns, si_);                           \
    if (P::HALF) cp_async<4>(ss_ + 48 * LQ_MRHS_BLOCK + 4 * tid, reinterpret_cast<const float*>(in + 48ll * g.ns) + si_); \
  }
  if (active) {
#pragma unroll
    for (int h = 0; h < NST; ++h) {
      switch (h) {
        case 0: LQ_ISSUE(0) break;
        case 1: LQ_ISSUE(1) break;
        case 2: LQ_ISSUE(2) break;
        default: LQ_ISSUE(3) break;
      }
      cp_async_commit();
    }
  }

  // phase 1: warp w reconstructs 8/NR links (hops w*8/NR ...) for the CTA's 32 sites
  if (site_ok) {
    const long long link_bytes = (long long)RECON * sizeof(typename P::store_t) * g.ns;
#pragma unroll
    for (int j = 0; j < 8 / NR; ++j) {
      const int h = w * (8 / NR) + j, mu = h >> 1;
      int nb = nbk[0];
      if (mu == 1) nb = nbk[1];
      if (mu == 2) nb = nbk[2];
      if (mu == 3) nb = nbk[3];
      // forward hop: link of the site (output parity); backward hop: link of the neighbour (input parity)
      const bool fw = (h & 1) == 0;
      const char* gp = a.gauge + (long long)((fw ? p : 1 - p) * 4 + mu) * link_bytes;
      R u[18], us;
      load_link<P, RECON>(u, us, gp, g.ns, fw ? idx : base + nb);
      LinkTile<R>::put(tile, h, lane, u);
    }
  }
  __syncthreads();

  if (active) {
    const R sig_f = dagger ? R(1) : R(-1);
    constexpr R USCALE = (P::HALF && RECON != 8) ? R(LQ_FIXED_INV) : R(1);    // load_link's uscale
    R acc[24];
#pragma unroll
    for (int k = 0; k < 24; ++k) acc[k] = 0;
#define LQ_PHOP(H)                                                                                         \
    {                                                                                                      \
      constexpr int MU_ = (H) / 2;                                                                         \
      constexpr bool FW_ = ((H) & 1) == 0;                                                                 \
      cp_async_wait<NST - 1>();                                                                            \
      const char* ss_ = ring + ((H) % NST) * SpinStage<P, NR>::BYTES;                                      \
      R u[18], psi[24], ps;                                                                                \
      LinkTile<R>::get(tile, (H), lane, u);                                                                \
      if constexpr (P::HALF) load_site_magic<P, 24, 2>(psi, ps, ss_, LQ_MRHS_BLOCK, tid);                  \
      else load_site_raw<P, 24, 2>(psi, ps, ss_, LQ_MRHS_BLOCK, tid);                                      \
      if ((H) + NST < 8) LQ_ISSUE(((H) + NST) % 8)                                                         \
      cp_async_commit();                                                                                   \
      const R sg_ = FW_ ? ((c[MU_] + 1 == g.X[MU_]) ? (R)g.bc[MU_] : R(1)) : ((c[MU_] == 0) ? (R)g.bc[MU_] : R(1)); \
      if constexpr (P::HALF) hop_fixed<MU_, FW_, (FW_ == (DAG == 1)) ? 1 : -1>(acc, psi, u, sg_ * USCALE * ps); \
      else hop<MU_, FW_, R>(acc, psi, u, FW_ ? sig_f : -sig_f, sg_);                                       \
    }
    LQ_PHOP(0) LQ_PHOP(1) LQ_PHOP(2) LQ_PHOP(3) LQ_PHOP(4) LQ_PHOP(5) LQ_PHOP(6) LQ_PHOP(7)
#undef LQ_PHOP
    R d0 = 0, d1 = 0, d2 = 0;
    dslash_epilogue<P, XPAY, CLOVX, CLOVOUT, false>(acc, a.y + (long long)rhs * fbytes, a.clov_y, a.clov_out, a.a, p, g.ns, idx, d0, d1, d2);
    store_site<P, 24>(acc, a.out + (long long)rhs * fbytes, g.ns, idx);
  }
#undef LQ_ISSUE
}

template <class P> cudaError_t launch_dslash_mrhs(const DslashArgs& a, int nrhs, int recon, int epi, cudaStream_t s);

}  // namespace lq
