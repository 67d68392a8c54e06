// host.h -- internal declarations shared by the translation units of liblqcd_b200.so:
// the context, the block-major (Schwarz) index map, and the launch wrappers.
#pragma once
#include <string>
#include <vector>
#include "core.cuh"
#include "blas.cuh"
#include "../../include/lqcd.h"

#ifndef LQ_HOST_SLABS
#define LQ_HOST_SLABS 16    /* max t-slabs of the host-buffer pipeline (host_api.cu) */
#endif

namespace lq {

// Natural layout <-> block-major layout.  The Schwarz preconditioner sees
// the lattice as nbd[0]*nbd[1]*nbd[2]*nbd[3] independent boxes of extents blk.X with open
// (Dirichlet) boundaries; box b = bx + nbd0*(by + nbd1*(bz + nbd2*bt)) occupies the contiguous
// index range [b*blk.vh, (b+1)*blk.vh) of every block-major field.  Block extents are even,
// so the parity of a site inside its box equals its global parity.
// cmaj != 0 (multiplicative Schwarz): the boxes are stored colour-major, colour = (bx+by+bz+bt) & 1 --
// the nb/2 boxes of colour 0 first, then those of colour 1 -- so that one colour is a contiguous box range
// (needs an even number of boxes in x: position q of colour c has bx = 2 (q % (nbd0/2)) + ((by+bz+bt+c) & 1),
// the checkerboard trick of the site index one level up).
// Overlapping domains (reading R18): ovl[m] > 0 grows every box by ovl[m] sites on both sides of the
// partitioned direction m, through the lattice's periodic wrap.  blk then holds the GROWN extents (blk.X = core + 2 ovl,
// blk.ns = nb * blk.vh > nat.ns: a block-major field has its own size), a site of the lattice appears in several boxes,
// and a box site knows whether it belongs to the box's own core.  The sum of the ovl[m] is even (set_blocks), so the
// parity of a site inside its grown box is still its global parity.  A grown box may contain an antiperiodic boundary
// of the lattice in its interior; the box operator carries no sign there (Dirichlet coefficients only at box edges):
// inside a box the sign plane is removed by psi -> -psi on the far side, applied when a field is gathered into the
// boxes (`sign` below) -- the own sites, the only ones scattered back, all have sign +1.
struct BlockMap {
  Geom nat;     // whole lattice, nb = 1
  Geom blk;     // one box (grown extents), nb = number of boxes, ns = nb * vh (= nat.ns without overlap)
  int nbd[4];
  int cmaj;
  int core[4];  // extents of the box itself
  int ovl[4];   // overlap per direction (0: none / direction not partitioned)
};

// natural checkerboard index of site lcb of box `box`; own: the site is in the box's core; sign: -1 if the site lies beyond
// an antiperiodic lattice boundary as seen from the box's core
LQ_DEV long long block_to_natural(const BlockMap& bm, int box, int lcb, int parity, bool* own = nullptr, int* sign = nullptr) {
  int lc[4];
  cb_to_coords(bm.blk, lcb, parity, lc);
  int bc[4];
  if (bm.cmaj) {
    const int half = bm.blk.nb >> 1, col = box >= half ? 1 : 0;
    int q = box - col * half;
    const int h0 = bm.nbd[0] >> 1;
    const int bxh = q % h0; q /= h0;
    bc[1] = q % bm.nbd[1]; q /= bm.nbd[1];
    bc[2] = q % bm.nbd[2];
    bc[3] = q / bm.nbd[2];
    bc[0] = 2 * bxh + ((bc[1] + bc[2] + bc[3] + col) & 1);
  } else {
    int b = box;
#pragma unroll
    for (int m = 0; m < 4; ++m) { bc[m] = b % bm.nbd[m]; b /= bm.nbd[m]; }
  }
  int gc[4], sg = 1;
  bool mine = true;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    int g = bc[m] * bm.core[m] - bm.ovl[m] + lc[m];
    if (g < 0) { g += bm.nat.X[m]; sg *= bm.nat.bc[m]; }
    else if (g >= bm.nat.X[m]) { g -= bm.nat.X[m]; sg *= bm.nat.bc[m]; }
    mine = mine && lc[m] >= bm.ovl[m] && lc[m] < bm.ovl[m] + bm.core[m];
    gc[m] = g;
  }
  if (own) *own = mine;
  if (sign) *sign = sg;
  return coords_to_cb(bm.nat, gc);
}

struct MultiArgs {
  BlasArgs b;
  const char* z[LQ_GCR_KMAX];
  double chi[2 * LQ_GCR_KMAX];
  int k, i0, n;
};

cudaError_t run_mr_alpha(const BlasArgs& a, cudaStream_t s);   // boxes [a.box0, a.box0 + a.nb): alpha_b = a.c[0] <w,rho>_b / <w,w>_b
cudaError_t run_gcr_dots(int prec, const MultiArgs& m, int max_ctas, cudaStream_t s);
cudaError_t run_gcr_orth(int prec, const MultiArgs& m, int max_ctas, cudaStream_t s);
cudaError_t run_convert(int pa, int pb, char* dst, const char* src, const BlockMap& bm, int dir, int parity, cudaStream_t s,
                        int box0 = 0, int nbox = 0);   // dir 2, nbox > 0: sites of boxes outside [box0, box0 + nbox) are written as zero
cudaError_t run_accumulate(int ph, int pl, char* y, const MultiArgs& m, cudaStream_t s);
cudaError_t run_dots_finalize(double* W, int n, int fin, cudaStream_t s);

// setup kernels (pack.cu, clover.cu)
cudaError_t run_pack_gauge(double* g64, const double* U_canonical, const Geom& nat, cudaStream_t s);
cudaError_t run_convert_gauge(int prec, int recon, char* dst, const double* g64, const BlockMap& bm, int blocked, cudaStream_t s,
                              unsigned* bad = nullptr);   // bad: device word, bit 0 = not SU(3), bit 1 = recon-8 singular (pack.cu)
cudaError_t run_pack_spinor(int prec, char* packed, const double* canonical, const Geom& nat, int parity, int unpack, cudaStream_t s,
                            long long i0 = 0, long long i1 = -1,    // sites [i0, i1) of the parity field (default: all)
                            int canonical_single = 0);              // canonical array is complex64 (lqcd_apply_host_c64)
cudaError_t run_clover_term(double* T72, const double* g64, const Geom& nat, double c_sw, cudaStream_t s);
cudaError_t run_clover_make(int prec, char* A, char* Ainv, const double* T72, const BlockMap& bm, int blocked, double kappa, cudaStream_t s);
cudaError_t run_clover_apply(int prec, char* out, const char* in, const char* clov, const Geom& g, int parity, cudaStream_t s);

inline size_t spinor_bytes(int prec, long long ns) { return (size_t)ns * (prec == 0 ? 192 : prec == 1 ? 96 : 52); }
inline size_t clover_bytes(int prec, long long ns) { return (size_t)ns * 2 * (prec == 0 ? 576 : prec == 1 ? 288 : 148); }
inline size_t gauge_bytes(int prec, int recon, long long ns) { return (size_t)ns * 8 * recon * (prec == 0 ? 8 : prec == 1 ? 4 : 2); }
inline int recon_index(int recon) { return recon == 18 ? 0 : recon == 12 ? 1 : recon == 8 ? 2 : -1; }

}  // namespace lq

// ------------------------------------------------------------------------------------------------
struct lqcd_ctx {
  int dims[4], bc[4], device;
  long long V, Vh;
  std::string err;
  std::vector<double> hist;   // iterated residual norms of the running solve (lqcd_invert_params::residual_history)
  lq::Geom nat;
  int n_sm;
  long long launches;

  // gauge: fp64 recon-18 natural master copy + derived copies [prec][recon index]
  bool have_gauge;
  double* g64;
  char* gauge[3][3];
  // Schwarz blocking currently materialised
  bool have_blocks;
  lq::BlockMap bm;
  char* bgauge[3][3];
  int schwarz_group;      // blocks per launch group of the preconditioner (0 = all; lqcd_invert_params::schwarz_group)
  int schwarz_overlap;    // overlap of the Schwarz domains (0 = none; lqcd_invert_params::schwarz_overlap)
  // clover
  bool have_clover;
  double c_sw;
  double* T72;            // kappa-independent term, fp64, natural, [parity][72 reals planes]
  double kappa;           // kappa of the materialised A / A^-1 copies (NaN = none)
  char* clov[3];          // A      [prec]  natural  (both parities)
  char* clovinv[3];       // A^-1
  char* bclov[3];         // block-major copies
  char* bclovinv[3];
  // workspace
  char* tmp[3];           // matpc temporary, natural layout, per precision
  char* tmp2[3];          // second temporary (symmetric form, dagger)
  char* btmp[3];          // block-major temporary
  double* S;              // device scalars (lq::S_TOTAL doubles)
  double* partials;       // reduction partials
  size_t partials_doubles;
  unsigned* counters;
  unsigned* gflag;        // device word written by the gauge conversion check (pack.cu)
  double* dotws;          // workspace of the reductions fused into the operator (dslash.cuh DOTS >= 2)
  size_t dotws_doubles;
  double* boxdots;        // MR per-box partial dots
  size_t boxdots_doubles;
  double* hS;             // pinned host mirror of S
  // workspace cache: buffers handed back by finished calls, reused by the next call that asks for the same size
  // (cudaMalloc / cudaFree of ~1 GB per solve cost milliseconds and, after a free, occasionally 100 ms);
  // released by lqcd_release_workspace and lqcd_destroy
  struct WsBuf { void* p; size_t bytes; cudaStream_t last; };
  std::vector<WsBuf> pool;
  // lqcd_apply_host: cached staging buffers, copy streams and events of the slab pipeline
  void* hws[8];
  size_t hws_bytes[8];
  cudaStream_t hs_in, hs_out;
  cudaEvent_t hev_in[LQ_HOST_SLABS], hev_out[LQ_HOST_SLABS], hev_sync;
  bool have_hpipe;
  // improved staggered path (staggered.cu): fp64 master links, fp32 copies, M^dag M temporaries
  bool have_stag;
  double *sfat64, *slng64;
  char *sfatp[2], *slngp[2];   // per precision: fat (fp32 copy; fp64 uses the master), long (18 or 12 reals)
  double slong_scale;          // != 0: every long link is slong_scale x SU(3) and is stored as 12 reals
  char* stmp[2];
  char* mtmp;             // multi-right-hand-side Mhat temporary (grow-only)
  size_t mtmp_bytes;
};
