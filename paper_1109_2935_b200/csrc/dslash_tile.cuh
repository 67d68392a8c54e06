// dslash_tile.cuh -- half-precision Wilson-clover hopping term, CTA-tile form with bulk-async staging.
//
// Same arithmetic, same epilogues and bit-identical results as dslash_kernel (dslash.cuh); what differs is how
// the 8 links and 8 neighbour spinors of a site reach the thread (north_star: "TMA or shared-memory staging").
// dslash_kernel: every thread cp.async's its own 6 pieces per hop (48 LDGSTS + their 64-bit address arithmetic per
// site, ~330 of its ~1,650 instructions; a probe with the copies removed runs 13 us faster at 32^3x64).
// Here a CTA owns a tile of T consecutive checkerboard sites = T / Xh whole rows of one (z, t) plane, and the data of
// one hop for the whole tile is 1-2 contiguous runs per chunk plane (the neighbours of a run of
// sites in a direction other than x are again a run; core.cuh layout):
//   x hops      : the tile's own index range (the +-x neighbour of a site lies in its own row)
//   y hops      : the range shifted by one row, plus the wrapped row when the tile touches y = 0 / Y-1
//   z, t hops   : the range shifted by one plane / one time slice (wrapped or not as a whole)
// One thread issues these runs as bulk asynchronous copies (cp.async.bulk global -> shared, completion counted in
// bytes on an mbarrier; SASS UBLKCP): 6-12 copy instructions per hop per CTA instead of 6 per thread.  Stages form a ring of NST hops; a stage is refilled once all T threads have read it (second mbarrier).
// Threads index the staged planes with threadIdx.x (x hops: the neighbour's position in the tile), so the
// per-thread neighbour index arithmetic of dslash_kernel is gone as well.
//
// Geometry the tile form needs (everything else runs dslash_kernel): Xh % 4 == 0 (16-byte runs of the 4-byte norm
// plane), T % Xh == 0, (Xh * Y) % T == 0, one box (natural layout), site range = whole time slices.
#pragma once
#include "dslash.cuh"

namespace lq {

struct TileInfo {
  int rows;       // T / Xh
  int magic;      // floor(i / Xh) == (i * magic) >> 16 for 0 <= i < T (checked on the host)
  int t0;         // first time slice of the launch (grid = tiles per (z,t) plane x Z x time slices: no index divisions)
  int pad;
  // start of every chunk plane the copies read (host-computed, so that a copy costs one 64-bit multiply-add on the
  // uniform datapath): input spinor (3 chunks + norm); links of the forward / backward hops [0 / 1][mu][plane]
  const char* sp[4];
  const char* lk[2][4][3];
};

LQ_DEV void mbar_init(void* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
LQ_DEV void mbar_expect_tx(void* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
LQ_DEV void mbar_arrive(void* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
LQ_DEV void mbar_wait(void* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "LQ_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra LQ_DONE_%=;\n"
      "bra LQ_WAIT_%=;\n"
      "LQ_DONE_%=:\n"
      "}\n" ::"r"(smem_addr(bar)), "r"(parity) : "memory");
}
// global -> shared bulk copy; bytes % 16 == 0, both addresses 16-byte aligned
LQ_DEV void bulk_g2s(void* dst, const void* src, unsigned bytes, void* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}

// chunk plane k of a record of N 16-bit reals (core.cuh Rec): bytes per site and byte offset of the plane per site count
template <int N> LQ_DEV void plane_of(int k, int& bpp, int& off) {
  typedef Rec<short, N> RC;
  if (k < RC::N16) { bpp = 16; off = 16 * k; }
  else if (RC::N8 && k == RC::N16) { bpp = 8; off = 16 * RC::N16; }
  else { bpp = 4; off = 16 * RC::N16 + 8 * RC::N8; }
}

template <int RECON, int T> struct TileStage {
  static constexpr int LINK_B = RECON * 2;
  static constexpr int SPIN_B = 52;
  static constexpr int BYTES = T * (LINK_B + SPIN_B);
  static constexpr int NLP = Rec<short, RECON>::N16 + Rec<short, RECON>::N8 + Rec<short, RECON>::N4;   // link planes
  static constexpr int NPL = NLP + 4;                                                                  // + 3 spinor chunks + norm
};

// Lane 0 of the calling warp starts the copies of hop H of the tile at cb0 into `stage`.
template <int RECON, int T, int H>
LQ_DEV void tile_issue(const DslashArgs& a, const TileInfo& ti, int cb0, int y0, int z, int t,
                       char* stage, void* bar, int lane) {
  typedef TileStage<RECON, T> TS;
  constexpr int MU = H / 2;
  constexpr bool FW = (H & 1) == 0;
  const Geom& g = a.g;
  const int Xh = g.Xh;
  // runs of the neighbour-indexed fields (spinor; link of a backward hop): source start, position in the tile, sites
  int s0, d0 = 0, n0 = T, s1 = 0, d1 = 0, n1 = 0;
  if (MU == 0) {
    s0 = cb0;
  } else if (MU == 1) {
    const int Y = g.X[1];
    if (FW) {
      s0 = cb0 + Xh;
      if (y0 + ti.rows == Y) { n0 = T - Xh; s1 = cb0 + T - Y * Xh; d1 = T - Xh; n1 = Xh; }   // last row: y = Y-1 -> y = 0
    } else {
      s0 = cb0 - Xh;
      if (y0 == 0) { s0 = cb0; d0 = Xh; n0 = T - Xh; s1 = cb0 + (Y - 1) * Xh; d1 = 0; n1 = Xh; }   // first row: y = 0 -> Y-1
    }
  } else {
    const int s = (MU == 2) ? Xh * g.X[1] : Xh * g.X[1] * g.X[2];
    const int c = (MU == 2) ? z : t, L = g.X[MU];
    if (FW) s0 = (c + 1 == L) ? cb0 - (L - 1) * s : cb0 + s;
    else s0 = (c == 0) ? cb0 + (L - 1) * s : cb0 - s;
  }
  // one thread issues the copies: every address is warp-uniform, so the sequence runs on the uniform datapath
  // (UBLKCP takes uniform registers; a copy per lane would be serialised by a lane-election loop anyway)
  if (lane == 0) {
    mbar_expect_tx(bar, TS::BYTES);
#pragma unroll
    for (int pl = 0; pl < TS::NLP; ++pl) {               // link: forward hop = at the output site, backward = at the neighbour
      int bpp, off;
      plane_of<RECON>(pl, bpp, off);
      const char* src = ti.lk[FW ? 0 : 1][MU][pl];
      char* dst = stage + off * T;
      if (FW) {
        bulk_g2s(dst, src + (long long)bpp * cb0, (unsigned)(bpp * T), bar);
      } else {
        if (n0 > 0) bulk_g2s(dst + bpp * d0, src + (long long)bpp * s0, (unsigned)(bpp * n0), bar);
        if (MU == 1 && n1 > 0) bulk_g2s(dst + bpp * d1, src + (long long)bpp * s1, (unsigned)(bpp * n1), bar);
      }
    }
#pragma unroll
    for (int pl = 0; pl < 4; ++pl) {                     // neighbour spinor: three 16-byte chunks, then the 4-byte norm plane
      int bpp, off;
      plane_of<24>(pl, bpp, off);
      const char* src = ti.sp[pl];
      char* dst = stage + T * TS::LINK_B + off * T;
      if (n0 > 0) bulk_g2s(dst + bpp * d0, src + (long long)bpp * s0, (unsigned)(bpp * n0), bar);
      if (MU == 1 && n1 > 0) bulk_g2s(dst + bpp * d1, src + (long long)bpp * s1, (unsigned)(bpp * n1), bar);
    }
  }
}

#ifndef LQ_TILE_MINB
#define LQ_TILE_MINB 5
#endif

template <int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int T, int NST, int DAG>
__global__ void __launch_bounds__(T, (LQ_TILE_MINB * 128) / T)
dslash_tile_kernel(const DslashArgs a, const TileInfo ti) {
  typedef PrecH P;
  typedef TileStage<RECON, T> TS;
  typedef float R;
  static_assert(NST >= 2 && NST <= 4, "ring depth");
  constexpr int NW = T / 32;
  extern __shared__ __align__(128) char lq_tile[];
  unsigned long long* full = reinterpret_cast<unsigned long long*>(lq_tile + NST * TS::BYTES);
  unsigned long long* empty = full + NST;
  const Geom& g = a.g;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const long long base = 0;                       // one box (tile_ok)
  const int p = a.parity & 1;
  // the tile: rows y0 .. y0 + rows - 1 of the plane (z, t)
  const int y0 = blockIdx.x * ti.rows, z = blockIdx.y, t = ti.t0 + blockIdx.z;
  const int cb0 = ((t * g.X[2] + z) * g.X[1] + y0) * g.Xh;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, T); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  // prologue: hop h < NST is started by warp h (spread, so that no warp carries the whole issue sequence)
  if (wid == 0 % NW) tile_issue<RECON, T, 0>(a, ti, cb0, y0, z, t, lq_tile + 0 * TS::BYTES, full + 0, lane);
  if (wid == 1 % NW) tile_issue<RECON, T, 1>(a, ti, cb0, y0, z, t, lq_tile + 1 * TS::BYTES, full + 1, lane);
  if (NST > 2 && wid == 2 % NW) tile_issue<RECON, T, 2>(a, ti, cb0, y0, z, t, lq_tile + 2 * TS::BYTES, full + 2, lane);
  if (NST > 3 && wid == 3 % NW) tile_issue<RECON, T, 3>(a, ti, cb0, y0, z, t, lq_tile + 3 * TS::BYTES, full + 3, lane);
  // this thread's site
  const int row = (tid * ti.magic) >> 16;
  const int xh = tid - row * g.Xh;
  const int y = y0 + row;
  const int rp = (y + z + t + p) & 1;
  const int xf = rp ? (xh + 1 == g.Xh ? 0 : xh + 1) : xh;
  const int xb = rp ? xh : (xh == 0 ? g.Xh - 1 : xh - 1);
  const int nxf = tid - xh + xf, nxb = tid - xh + xb;           // +-x neighbours: positions in the tile
  const long long idx = base + cb0 + tid;
  R acc[24];
#pragma unroll
  for (int k = 0; k < 24; ++k) acc[k] = 0;

#define LQ_THOP(H)                                                                                         \
  {                                                                                                        \
    constexpr int MU_ = (H) / 2;                                                                           \
    constexpr bool FW_ = ((H) & 1) == 0;                                                                   \
    constexpr int ST_ = (H) % NST;                                                                         \
    const char* sb_ = lq_tile + ST_ * TS::BYTES;                                                           \
    mbar_wait(full + ST_, ((H) / NST) & 1);                                                                \
    R u[18], psi[24], us, ps;                                                                              \
    load_link<P, RECON, 2>(u, us, sb_, T, (MU_ == 0 && !FW_) ? nxb : tid);                                 \
    load_site_magic<P, 24, 2>(psi, ps, sb_ + T * TS::LINK_B, T, MU_ == 0 ? (FW_ ? nxf : nxb) : tid);       \
    /* generic-proxy reads of the stage are ordered before the async-proxy (bulk copy) writes that will refill */ \
    /* it by a proxy fence in the reading thread; without it the refill was seen to corrupt ~1 % of the sites   */ \
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");                                           \
    mbar_arrive(empty + ST_);                                                                              \
    if ((H) >= 1 && (H) - 1 + NST < 8 && wid == (H) % NW) {                                                \
      /* refill the stage of the previous hop once every thread has read it */                             \
      mbar_wait(empty + ((H) - 1) % NST, (((H) - 1) / NST) & 1);                                           \
      tile_issue<RECON, T, ((H) - 1 + NST) % 8>(a, ti, cb0, y0, z, t, lq_tile + (((H) - 1) % NST) * TS::BYTES, \
                                                full + ((H) - 1) % NST, lane);                             \
    }                                                                                                      \
    int cm_, lm_;                                                                                          \
    if (MU_ == 0) { cm_ = 2 * xh + rp; lm_ = g.X[0]; }                                                     \
    else if (MU_ == 1) { cm_ = y; lm_ = g.X[1]; }                                                          \
    else if (MU_ == 2) { cm_ = z; lm_ = g.X[2]; }                                                          \
    else { cm_ = t; lm_ = g.X[3]; }                                                                        \
    const R sg_ = FW_ ? ((cm_ + 1 == lm_) ? (R)g.bc[MU_] : R(1)) : ((cm_ == 0) ? (R)g.bc[MU_] : R(1));     \
    hop_fixed<MU_, FW_, (FW_ == (DAG == 1)) ? 1 : -1>(acc, psi, u, sg_ * us * ps);                         \
  }
  LQ_THOP(0) LQ_THOP(1) LQ_THOP(2) LQ_THOP(3) LQ_THOP(4) LQ_THOP(5) LQ_THOP(6) LQ_THOP(7)
#undef LQ_THOP

  R d0 = 0, d1 = 0, d2 = 0;
  dslash_epilogue<P, XPAY, CLOVX, CLOVOUT, false>(acc, a.y, a.clov_y, a.clov_out, a.a, p, g.ns, idx, d0, d1, d2);
  store_site<P, 24>(acc, a.out, g.ns, idx);
}

// true if the tile form with T threads per CTA applies to this launch
template <int T> inline bool tile_ok(const DslashArgs& a, TileInfo& ti) {
  const Geom& g = a.g;
  if (g.nb != 1 || g.Xh % 4 || T % g.Xh || (g.Xh * g.X[1]) % T) return false;
  const int slice = g.Xh * g.X[1] * g.X[2];       // whole time slices only
  if (a.range.cb0 % slice || (a.range.cb1 - a.range.cb0) % slice || a.range.cb1 <= a.range.cb0) return false;
  if (g.X[2] > 65535 || (a.range.cb1 - a.range.cb0) / slice > 65535) return false;
  ti.t0 = a.range.cb0 / slice;
  ti.pad = 0;
  ti.rows = T / g.Xh;
  ti.magic = 65536 / g.Xh + 1;
  for (int i = 0; i < T; ++i) if (((i * ti.magic) >> 16) != i / g.Xh) return false;
  return true;
}

// plane starts of the fields of one launch (TileInfo::sp, ::lk)
template <int RECON> inline void tile_planes(const DslashArgs& a, TileInfo& ti) {
  const long long ns = a.g.ns, link_bytes = 2ll * RECON * ns;
  typedef Rec<short, RECON> RC;
  for (int pl = 0; pl < 4; ++pl) ti.sp[pl] = a.in + (pl < 3 ? 16ll * pl : 48ll) * ns;
  for (int fb = 0; fb < 2; ++fb)
    for (int mu = 0; mu < 4; ++mu) {
      const char* f = a.gauge + (long long)(((fb == 0 ? (a.parity & 1) : 1 - (a.parity & 1)) * 4) + mu) * link_bytes;
      for (int pl = 0; pl < 3; ++pl) {
        const long long off = pl < RC::N16 ? 16ll * pl : (RC::N8 && pl == RC::N16) ? 16ll * RC::N16 : 16ll * RC::N16 + 8ll * RC::N8;
        ti.lk[fb][mu][pl] = f + off * ns;
      }
    }
}

}  // namespace lq
