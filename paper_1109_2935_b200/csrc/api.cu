// api.cu -- C ABI entry points of include/lqcd.h: context, field management, operators.
#include <cmath>
#include <cstdio>
#include <cstring>
#include "ops.h"

using namespace lq;

namespace lq {

int fail(lqcd_ctx* c, int code, const char* what, cudaError_t e) {
  if (c) {
    c->err = what;
    if (e != cudaSuccess) { c->err += ": "; c->err += cudaGetErrorString(e); }
  }
  return code;
}

static Geom make_geom(const int* X, const int* bc, int nb) {
  Geom g;
  for (int m = 0; m < 4; ++m) { g.X[m] = X[m]; g.bc[m] = bc[m]; }
  g.Xh = X[0] / 2;
  g.vh = X[0] * X[1] * X[2] * X[3] / 2;
  g.nb = nb;
  g.ns = (long long)nb * g.vh;
  auto magic = [](int d) { return d <= 1 ? 0u : (unsigned)(((1ull << 32) + (unsigned)d - 1) / (unsigned)d); };
  g.mXh = magic(g.Xh); g.mY = magic(X[1]); g.mZ = magic(X[2]);
  return g;
}

int dev_alloc(lqcd_ctx* c, void** p, size_t bytes) {
  cudaError_t e = cudaMalloc(p, bytes);
  if (e != cudaSuccess) { *p = nullptr; return fail(c, LQCD_ENOMEM, "cudaMalloc", e); }
  return LQCD_OK;
}

int ws_get(lqcd_ctx* c, void** p, size_t bytes, cudaStream_t s) {
  for (size_t i = 0; i < c->pool.size(); ++i) {
    if (c->pool[i].bytes != bytes) continue;
    lqcd_ctx::WsBuf b = c->pool[i];
    c->pool.erase(c->pool.begin() + i);
    if (b.last != s) cudaStreamSynchronize(b.last);     // handed back on another stream: let its work finish first
    *p = b.p;
    return LQCD_OK;
  }
  int rc = dev_alloc(c, p, bytes);
  if (rc && !c->pool.empty()) {                          // out of memory: drop the cache and try once more
    cudaDeviceSynchronize();
    for (auto& b : c->pool) cudaFree(b.p);
    c->pool.clear();
    rc = dev_alloc(c, p, bytes);
  }
  return rc;
}

void ws_put(lqcd_ctx* c, void* p, size_t bytes, cudaStream_t s) {
  if (p) c->pool.push_back(lqcd_ctx::WsBuf{p, bytes, s});
}

static void free_p(char*& p) { if (p) cudaFree(p); p = nullptr; }

static void drop_clover_copies(lqcd_ctx* c) {
  for (int i = 0; i < 3; ++i) { free_p(c->clov[i]); free_p(c->clovinv[i]); free_p(c->bclov[i]); free_p(c->bclovinv[i]); }
  c->kappa = NAN;
}
static void drop_block_copies(lqcd_ctx* c) {
  for (int i = 0; i < 3; ++i) {
    for (int r = 0; r < 3; ++r) free_p(c->bgauge[i][r]);
    free_p(c->bclov[i]); free_p(c->bclovinv[i]); free_p(c->btmp[i]);
  }
  c->have_blocks = false;
}
static void drop_gauge_copies(lqcd_ctx* c) {
  for (int i = 0; i < 3; ++i) for (int r = 0; r < 3; ++r) { free_p(c->gauge[i][r]); free_p(c->bgauge[i][r]); }
}

int get_gauge(lqcd_ctx* c, int prec, int recon, bool blocked, const char** out, cudaStream_t s) {
  const int ri = recon_index(recon);
  if (prec < 0 || prec > 2 || ri < 0) return fail(c, LQCD_EINVAL, "bad precision / recon");
  if (!c->have_gauge) return fail(c, LQCD_ESTATE, "gauge field not loaded");
  if (blocked && !c->have_blocks) return fail(c, LQCD_ESTATE, "no Schwarz blocking set");
  char*& slot = blocked ? c->bgauge[prec][ri] : c->gauge[prec][ri];
  if (!slot) {
    // built into a local and published only when it holds valid links; the stream is synchronised once, so the copy
    // is complete for every stream that uses it later
    char* g = nullptr;
    int rc = dev_alloc(c, (void**)&g, gauge_bytes(prec, recon, blocked ? c->bm.blk.ns : c->nat.ns));
    if (rc) return rc;
    unsigned bad = 0;
    cudaError_t e = cudaMemsetAsync(c->gflag, 0, sizeof(unsigned), s);
    if (e == cudaSuccess) e = run_convert_gauge(prec, recon, g, c->g64, c->bm, blocked ? 1 : 0, s, c->gflag);
    c->launches++;
    if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, c->gflag, sizeof(unsigned), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cudaFree(g); return fail(c, LQCD_ECUDA, "convert_gauge", e); }
    if (bad) {
      cudaFree(g);
      return fail(c, LQCD_EINVAL, (bad & 1u) ? "gauge links are not SU(3) to 1e-9: use recon 18 (recon 12 / 8 reconstruct unitary links only)"
                                            : "recon 8 cannot represent this gauge field: a link has |a2|^2 + |a3|^2 = 0 in the stored precision (e.g. U = 1); use recon 12 or 18");
    }
    slot = g;
  }
  *out = slot;
  return LQCD_OK;
}

int get_clover(lqcd_ctx* c, int prec, double kappa, bool blocked, const char** A, const char** Ainv, cudaStream_t s) {
  if (prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "bad precision");
  if (!c->have_clover) return fail(c, LQCD_ESTATE, "clover term not built");
  if (blocked && !c->have_blocks) return fail(c, LQCD_ESTATE, "no Schwarz blocking set");
  if (!(c->kappa == kappa)) { drop_clover_copies(c); c->kappa = kappa; }
  char*& a = blocked ? c->bclov[prec] : c->clov[prec];
  char*& ai = blocked ? c->bclovinv[prec] : c->clovinv[prec];
  if (!a || !ai) {
    char *na = nullptr, *nai = nullptr;       // published only when both hold valid data (see get_gauge)
    const long long ns = blocked ? c->bm.blk.ns : c->nat.ns;
    int rc = dev_alloc(c, (void**)&na, clover_bytes(prec, ns));
    if (rc) return rc;
    rc = dev_alloc(c, (void**)&nai, clover_bytes(prec, ns));
    if (rc) { cudaFree(na); return rc; }
    cudaError_t e = run_clover_make(prec, na, nai, c->T72, c->bm, blocked ? 1 : 0, kappa, s);
    c->launches++;
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cudaFree(na); cudaFree(nai); return fail(c, LQCD_ECUDA, "clover_make", e); }
    free_p(a); free_p(ai);
    a = na; ai = nai;
  }
  *A = a; *Ainv = ai;
  return LQCD_OK;
}

int get_tmp(lqcd_ctx* c, int prec, bool blocked, char** out) {
  char*& t = blocked ? c->btmp[prec] : c->tmp[prec];
  if (!t) { int rc = dev_alloc(c, (void**)&t, spinor_bytes(prec, blocked ? c->bm.blk.ns : c->nat.ns)); if (rc) return rc; }
  *out = t;
  return LQCD_OK;
}

int set_blocks(lqcd_ctx* c, const int* blk, int cmaj, int overlap) {
  if (!blk) return fail(c, LQCD_EINVAL, "null block");
  for (int m = 0; m < 4; ++m)
    if (blk[m] < 2 || (blk[m] & 1) || c->dims[m] % blk[m]) return fail(c, LQCD_EINVAL, "Schwarz block extents must be even and divide the lattice");
  if (cmaj && ((c->dims[0] / blk[0]) & 1)) return fail(c, LQCD_EINVAL, "multiplicative Schwarz needs an even number of blocks in x");
  // overlapping domains (reading R18): every partitioned direction grows by `overlap` sites on both sides
  int ovl[4], osum = 0;
  for (int m = 0; m < 4; ++m) {
    ovl[m] = (overlap > 0 && c->dims[m] / blk[m] > 1) ? overlap : 0;
    osum += ovl[m];
    if (ovl[m] && blk[m] + 2 * ovl[m] >= c->dims[m]) return fail(c, LQCD_EINVAL, "Schwarz overlap: a domain would reach around the lattice");
  }
  if (overlap < 0 || (osum & 1)) return fail(c, LQCD_EINVAL, "Schwarz overlap: overlap x number of partitioned directions must be even");
  if (osum && cmaj) return fail(c, LQCD_EINVAL, "multiplicative Schwarz is built for non-overlapping blocks");
  // cmaj = 0: either box order will do (the additive preconditioner does not care), so matching copies are kept
  if (c->have_blocks && !memcmp(blk, c->bm.core, 4 * sizeof(int)) && !memcmp(ovl, c->bm.ovl, 4 * sizeof(int)) && (!cmaj || c->bm.cmaj)) return LQCD_OK;
  drop_block_copies(c);
  c->bm.cmaj = cmaj ? 1 : 0;
  int nb = 1, bcb[4], ext[4];
  for (int m = 0; m < 4; ++m) {
    c->bm.nbd[m] = c->dims[m] / blk[m];
    nb *= c->bm.nbd[m];
    bcb[m] = (c->bm.nbd[m] == 1) ? c->bc[m] : 0;    // unpartitioned direction keeps its wrap (R7)
    c->bm.core[m] = blk[m]; c->bm.ovl[m] = ovl[m];
    ext[m] = blk[m] + 2 * ovl[m];
  }
  c->bm.nat = c->nat;
  c->bm.blk = make_geom(ext, bcb, nb);
  c->have_blocks = true;
  // per-warp partial dots of every box, then alpha_b (re, im) of every box
  const size_t need = (size_t)nb * ((c->bm.blk.vh + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK) * (LQ_DSLASH_BLOCK / 32) * 4 + 2 * (size_t)nb;
  if (need > c->boxdots_doubles) {
    if (c->boxdots) cudaFree(c->boxdots);
    c->boxdots = nullptr; c->boxdots_doubles = 0;
    int rc = dev_alloc(c, (void**)&c->boxdots, need * sizeof(double));
    if (rc) return rc;
    c->boxdots_doubles = need;
  }
  return LQCD_OK;
}

// out = [C] ([A] y + a * D in) : one fused launch (dslash.cuh)
// workspace of the reductions fused into the operator (dslash.cuh, DOTS >= 2): header + 3 doubles per CTA
static int get_dotws(lqcd_ctx* c, int nsite, double** out, cudaStream_t s) {
  const size_t need = 8 + 3 * (size_t)((nsite + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK);
  if (c->dotws_doubles < need) {
    if (c->dotws) cudaFree(c->dotws);             // synchronises
    c->dotws = nullptr; c->dotws_doubles = 0;
    int rc = dev_alloc(c, (void**)&c->dotws, need * sizeof(double));
    if (rc) return rc;
    c->dotws_doubles = need;
    double hdr[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    memcpy(&hdr[0], &c->S, sizeof(double*));      // W[0] = address of the scalar array
    cudaError_t e = cudaMemcpyAsync(c->dotws, hdr, sizeof(hdr), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "dot workspace", e);
  }
  *out = c->dotws;
  return LQCD_OK;
}

int op_dslash(lqcd_ctx* c, char* out, const char* in, const char* y, int parity_out, int dagger, int prec, int recon,
              int epi, double a, double kappa, bool blocked, cudaStream_t s, int cb0, int cb1, int fin, const char* q,
              int box0, int nbox) {
  DslashArgs d;
  memset(&d, 0, sizeof(d));
  d.g = blocked ? c->bm.blk : c->nat;
  d.out = out; d.in = in; d.y = y; d.a = a; d.parity = parity_out; d.dagger = dagger;
  if (nbox > 0) {                                   // a group of Schwarz blocks: boxes [box0, box0 + nbox)
    if (!blocked || box0 < 0 || box0 + nbox > d.g.nb) return fail(c, LQCD_EINVAL, "box range");
    d.g.nb = nbox;                                  // boxes of this launch; g.ns stays the stride of the whole field
    d.parity = parity_out | (box0 << 8);
  }
  int rc = get_gauge(c, prec, recon, blocked, &d.gauge, s);
  if (rc) return rc;
  if (epi != EPI_NONE && epi != EPI_XPAY) {
    const char *A, *Ai;
    rc = get_clover(c, prec, kappa, blocked, &A, &Ai, s);
    if (rc) return rc;
    d.clov_y = A; d.clov_out = Ai;
  }
  if (epi == EPI_CLOVX_XPAY_DOTS) d.dots = c->boxdots;          // whole boxes (the two share storage, dslash.cuh)
  else if (epi == EPI_CLOVX_XPAY_YDOT || epi == EPI_CLOVX_XPAY_QDOT) {
    if (blocked || fin <= 0 || (epi == EPI_CLOVX_XPAY_QDOT && !q)) return fail(c, LQCD_EINVAL, "fused reduction arguments");
    if ((rc = get_dotws(c, d.g.vh, &d.dots, s))) return rc;
    if (epi == EPI_CLOVX_XPAY_QDOT) d.clov_out = q;            // the third vector travels in the unused A^-1 slot
  }
  else { d.range.cb0 = cb0; d.range.cb1 = cb1 < 0 ? d.g.vh : cb1; }
  cudaError_t e;
  switch (prec) {
    case 0: e = launch_dslash<PrecD>(d, recon, epi, s); break;
    case 1: e = launch_dslash<PrecS>(d, recon, epi, s); break;
    case 2: e = launch_dslash<PrecH>(d, recon, epi, s); break;
    default: return fail(c, LQCD_EINVAL, "bad precision");
  }
  c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "dslash launch", e);
  if (epi == EPI_CLOVX_XPAY_YDOT || epi == EPI_CLOVX_XPAY_QDOT) {
    e = run_dots_finalize(d.dots, (d.g.vh + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK, fin, s);
    c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "dots finalize launch", e);
  }
  return LQCD_OK;
}

// out = Mhat in  (R6):  tmp = A^-1 D in ;  out = A in - kappa^2 D tmp.
// sym != 0: the symmetric form Mhat_s = 1 - kappa^2 A^-1 D A^-1 D:  tmp = A^-1 D in ; out = in - kappa^2 A^-1 D tmp,
// and Mhat_s^dag = 1 - kappa^2 D^dag A^-1 D^dag A^-1:  t0 = A^-1 in ; tmp = A^-1 D^dag t0 ; out = in - kappa^2 D^dag tmp.
// fin != 0 (asymmetric form, natural layout only): the second launch also reduces <out,in>, ||out||^2 (q == nullptr) or
// <q,out>, ||out||^2 over the field and dots_finalize_kernel (blas.cu), launched behind it, performs the scalar update `fin` (DotsFin, dslash.cuh)
int op_matpc(lqcd_ctx* c, char* out, const char* in, int parity, int dagger, double kappa, int prec, int recon,
             bool blocked, bool dots, cudaStream_t s, int sym, int fin, const char* q, int box0, int nbox) {
  char* tmp;
  int rc = get_tmp(c, prec, blocked, &tmp);
  if (rc) return rc;
  if (sym) {
    if (blocked || dots || fin) return fail(c, LQCD_EINVAL, "symmetric form is not available for the Schwarz operator / fused reductions");
    if (!dagger) {
      rc = op_dslash(c, tmp, in, nullptr, 1 - parity, 0, prec, recon, EPI_CLOVOUT, 0.0, kappa, false, s);
      if (rc) return rc;
      return op_dslash(c, out, tmp, in, parity, 0, prec, recon, EPI_XPAY_CLOVD, -kappa * kappa, kappa, false, s);
    }
    char*& t2 = c->tmp2[prec];
    if (!t2) { rc = dev_alloc(c, (void**)&t2, spinor_bytes(prec, c->nat.ns)); if (rc) return rc; }
    const char *A, *Ai;
    rc = get_clover(c, prec, kappa, false, &A, &Ai, s);
    if (rc) return rc;
    cudaError_t e = run_clover_apply(prec, t2, in, Ai, c->nat, parity, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "clover_apply", e);
    rc = op_dslash(c, tmp, t2, nullptr, 1 - parity, 1, prec, recon, EPI_CLOVOUT, 0.0, kappa, false, s);
    if (rc) return rc;
    return op_dslash(c, out, tmp, in, parity, 1, prec, recon, EPI_XPAY, -kappa * kappa, kappa, false, s);
  }
  rc = op_dslash(c, tmp, in, nullptr, 1 - parity, dagger, prec, recon, EPI_CLOVOUT, 0.0, kappa, blocked, s, 0, -1, 0, nullptr, box0, nbox);
  if (rc) return rc;
  if (fin) return op_dslash(c, out, tmp, in, parity, dagger, prec, recon, q ? EPI_CLOVX_XPAY_QDOT : EPI_CLOVX_XPAY_YDOT,
                            -kappa * kappa, kappa, blocked, s, 0, -1, fin, q);
  return op_dslash(c, out, tmp, in, parity, dagger, prec, recon, dots ? EPI_CLOVX_XPAY_DOTS : EPI_CLOVX_XPAY,
                   -kappa * kappa, kappa, blocked, s, 0, -1, 0, nullptr, box0, nbox);
}

// multi-right-hand-side Dslash: the same fused launch for nrhs fields sharing the links
int op_dslash_mrhs(lqcd_ctx* c, char* out, const char* in, const char* y, int nrhs, int parity_out, int dagger, int prec,
                   int recon, int epi, double a, double kappa, cudaStream_t s) {
  if (nrhs < 1 || nrhs > LQCD_MAX_RHS) return fail(c, LQCD_EINVAL, "nrhs");
  DslashArgs d;
  memset(&d, 0, sizeof(d));
  d.g = c->nat;
  d.out = out; d.in = in; d.y = y; d.a = a; d.parity = parity_out;
  d.dagger = (dagger ? 1 : 0) | (nrhs << 8);
  d.range.cb0 = 0; d.range.cb1 = d.g.vh;
  int rc = get_gauge(c, prec, recon, false, &d.gauge, s);
  if (rc) return rc;
  if (epi != EPI_NONE && epi != EPI_XPAY) {
    const char *A, *Ai;
    rc = get_clover(c, prec, kappa, false, &A, &Ai, s);
    if (rc) return rc;
    d.clov_y = A; d.clov_out = Ai;
  }
  cudaError_t e;
  switch (prec) {
    case 0: e = launch_dslash_mrhs<PrecD>(d, nrhs, recon, epi, s); break;
    case 1: e = launch_dslash_mrhs<PrecS>(d, nrhs, recon, epi, s); break;
    case 2: e = launch_dslash_mrhs<PrecH>(d, nrhs, recon, epi, s); break;
    default: return fail(c, LQCD_EINVAL, "bad precision");
  }
  c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "dslash_mrhs launch", e);
  return LQCD_OK;
}

int op_matpc_mrhs(lqcd_ctx* c, char* out, const char* in, int nrhs, int parity, int dagger, double kappa, int prec, int recon,
                  cudaStream_t s) {
  const size_t need = spinor_bytes(prec, c->nat.ns) * (size_t)nrhs;
  if (c->mtmp_bytes < need) {
    if (c->mtmp) cudaFree(c->mtmp);                   // synchronises: no launch still uses the old buffer
    c->mtmp = nullptr; c->mtmp_bytes = 0;
    int rc = dev_alloc(c, (void**)&c->mtmp, need);
    if (rc) return rc;
    c->mtmp_bytes = need;
  }
  int rc = op_dslash_mrhs(c, c->mtmp, in, nullptr, nrhs, 1 - parity, dagger, prec, recon, EPI_CLOVOUT, 0.0, kappa, s);
  if (rc) return rc;
  return op_dslash_mrhs(c, out, c->mtmp, in, nrhs, parity, dagger, prec, recon, EPI_CLOVX_XPAY, -kappa * kappa, kappa, s);
}

}  // namespace lq

// ================================================================================================
extern "C" {

int lqcd_create(lqcd_ctx** out, const int dims[4], const int boundary[4], int device) {
  if (!out || !dims || !boundary) return LQCD_EINVAL;
  *out = nullptr;
  for (int m = 0; m < 4; ++m) {
    if (dims[m] < 2 || (dims[m] & 1)) return LQCD_EINVAL;
    if (boundary[m] != 1 && boundary[m] != -1) return LQCD_EINVAL;
  }
  if ((long long)dims[0] * dims[1] * dims[2] * dims[3] / 2 > 0x7fffffffLL) return LQCD_EINVAL;
  {   // the site index is decomposed with multiply-high divisions (core.cuh Geom): n / d is exact while n d < 2^32
    const long long vh = (long long)dims[0] * dims[1] * dims[2] * dims[3] / 2, xh = dims[0] / 2;
    if (vh * xh >= (1ll << 32) || (vh / xh) * dims[1] >= (1ll << 32) || (vh / xh / dims[1]) * dims[2] >= (1ll << 32)) return LQCD_EINVAL;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return LQCD_ECUDA;
  if (cudaSetDevice(device) != cudaSuccess) return LQCD_ECUDA;
  lqcd_ctx* c = new (std::nothrow) lqcd_ctx();
  if (!c) return LQCD_ENOMEM;
  for (int m = 0; m < 4; ++m) { c->dims[m] = dims[m]; c->bc[m] = boundary[m]; }
  c->device = device;
  c->V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
  c->Vh = c->V / 2;
  c->nat = make_geom(dims, boundary, 1);
  c->bm.nat = c->nat; c->bm.blk = c->nat; c->bm.nbd[0] = c->bm.nbd[1] = c->bm.nbd[2] = c->bm.nbd[3] = 1; c->bm.cmaj = 0;
  for (int m = 0; m < 4; ++m) { c->bm.core[m] = c->dims[m]; c->bm.ovl[m] = 0; }
  c->launches = 0;
  c->have_gauge = c->have_blocks = c->have_clover = false;
  c->schwarz_group = 0;
  c->schwarz_overlap = 0;
  c->g64 = nullptr; c->T72 = nullptr; c->kappa = NAN; c->c_sw = NAN;
  memset(c->gauge, 0, sizeof(c->gauge)); memset(c->bgauge, 0, sizeof(c->bgauge));
  memset(c->clov, 0, sizeof(c->clov)); memset(c->clovinv, 0, sizeof(c->clovinv));
  memset(c->bclov, 0, sizeof(c->bclov)); memset(c->bclovinv, 0, sizeof(c->bclovinv));
  memset(c->tmp, 0, sizeof(c->tmp)); memset(c->btmp, 0, sizeof(c->btmp)); memset(c->tmp2, 0, sizeof(c->tmp2));
  c->S = nullptr; c->partials = nullptr; c->counters = nullptr; c->boxdots = nullptr; c->hS = nullptr;
  c->boxdots_doubles = 0;
  c->gflag = nullptr;
  c->dotws = nullptr; c->dotws_doubles = 0;
  memset(c->hws, 0, sizeof(c->hws)); memset(c->hws_bytes, 0, sizeof(c->hws_bytes));
  c->have_hpipe = false;
  c->mtmp = nullptr; c->mtmp_bytes = 0;
  c->have_stag = false; c->sfat64 = c->slng64 = nullptr; c->sfatp[0] = c->sfatp[1] = c->slngp[0] = c->slngp[1] = nullptr; c->slong_scale = 0; c->stmp[0] = c->stmp[1] = nullptr;
  cudaDeviceProp prop;
  cudaGetDeviceProperties(&prop, device);
  c->n_sm = prop.multiProcessorCount;
  c->partials_doubles = (size_t)c->n_sm * LQ_BLAS_CTAS_PER_SM * 16 + 4096;
  // scalars / partials for LQCD_MAX_RHS right-hand sides (batched solves; a single solve uses set 0)
  bool ok = cudaMalloc((void**)&c->S, (size_t)LQCD_MAX_RHS * S_TOTAL * sizeof(double)) == cudaSuccess &&
            cudaMalloc((void**)&c->partials, (size_t)LQCD_MAX_RHS * c->partials_doubles * sizeof(double)) == cudaSuccess &&
            cudaMalloc((void**)&c->counters, 4096 * sizeof(unsigned)) == cudaSuccess &&
            cudaMalloc((void**)&c->gflag, sizeof(unsigned)) == cudaSuccess &&
            cudaMallocHost((void**)&c->hS, (size_t)(S_TOTAL + 4 * LQCD_MAX_RHS) * sizeof(double)) == cudaSuccess;
  if (ok) ok = cudaMemset(c->S, 0, (size_t)LQCD_MAX_RHS * S_TOTAL * sizeof(double)) == cudaSuccess &&
               cudaMemset(c->counters, 0, 4096 * sizeof(unsigned)) == cudaSuccess;
  if (!ok) { lqcd_destroy(c); return LQCD_ENOMEM; }
  *out = c;
  return LQCD_OK;
}

int lqcd_destroy(lqcd_ctx* c) {
  if (!c) return LQCD_EINVAL;
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  drop_gauge_copies(c); drop_clover_copies(c); drop_block_copies(c);
  for (int i = 0; i < 3; ++i) { free_p(c->tmp[i]); free_p(c->tmp2[i]); }
  if (c->g64) cudaFree(c->g64);
  if (c->T72) cudaFree(c->T72);
  if (c->S) cudaFree(c->S);
  if (c->partials) cudaFree(c->partials);
  if (c->counters) cudaFree(c->counters);
  if (c->gflag) cudaFree(c->gflag);
  if (c->dotws) cudaFree(c->dotws);
  if (c->boxdots) cudaFree(c->boxdots);
  if (c->hS) cudaFreeHost(c->hS);
  for (auto& b : c->pool) cudaFree(b.p);
  for (void* p : c->hws) if (p) cudaFree(p);
  if (c->mtmp) cudaFree(c->mtmp);
  for (void* p : {(void*)c->sfat64, (void*)c->slng64, (void*)c->sfatp[0], (void*)c->sfatp[1], (void*)c->slngp[0], (void*)c->slngp[1], (void*)c->stmp[0], (void*)c->stmp[1]}) if (p) cudaFree(p);
  if (c->have_hpipe) {
    cudaStreamDestroy(c->hs_in); cudaStreamDestroy(c->hs_out); cudaEventDestroy(c->hev_sync);
    for (int i = 0; i < LQ_HOST_SLABS; ++i) { cudaEventDestroy(c->hev_in[i]); cudaEventDestroy(c->hev_out[i]); }
  }
  delete c;
  return LQCD_OK;
}

int lqcd_release_workspace(lqcd_ctx* c) {
  if (!c) return LQCD_EINVAL;
  cudaSetDevice(c->device);
  cudaDeviceSynchronize();
  for (auto& b : c->pool) cudaFree(b.p);
  c->pool.clear();
  return LQCD_OK;
}

const char* lqcd_last_error(const lqcd_ctx* c) { return c ? c->err.c_str() : "null context"; }

long long lqcd_launch_count(const lqcd_ctx* c) { return c ? c->launches : 0; }

int lqcd_load_gauge(lqcd_ctx* c, const void* U, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!U) return fail(c, LQCD_EINVAL, "null gauge pointer");
  cudaStream_t s = (cudaStream_t)stream;
  cudaSetDevice(c->device);
  drop_gauge_copies(c); drop_clover_copies(c);
  c->have_clover = false;
  if (!c->g64) { int rc = dev_alloc(c, (void**)&c->g64, gauge_bytes(0, 18, c->nat.ns)); if (rc) return rc; }
  cudaError_t e = run_pack_gauge(c->g64, (const double*)U, c->nat, s);
  c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack_gauge", e);
  c->have_gauge = true;
  return LQCD_OK;
}

int lqcd_build_clover(lqcd_ctx* c, double c_sw, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!c->have_gauge) return fail(c, LQCD_ESTATE, "build_clover before load_gauge");
  cudaStream_t s = (cudaStream_t)stream;
  cudaSetDevice(c->device);
  drop_clover_copies(c);
  if (!c->T72) { int rc = dev_alloc(c, (void**)&c->T72, (size_t)c->nat.ns * 2 * 576); if (rc) return rc; }
  cudaError_t e = run_clover_term(c->T72, c->g64, c->nat, c_sw, s);
  c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "clover_term", e);
  c->c_sw = c_sw;
  c->have_clover = true;
  return LQCD_OK;
}

size_t lqcd_field_bytes(const lqcd_ctx* c, int kind, int prec) {
  if (!c || prec < 0 || prec > 2) return 0;
  if (kind == LQCD_FIELD_STAGGERED_PARITY) return prec == 2 ? 0 : (size_t)c->Vh * 6 * (prec == 0 ? 8 : 4);
  if (kind != LQCD_FIELD_SPINOR_PARITY) return 0;
  return spinor_bytes(prec, c->nat.ns);
}

int lqcd_pack_spinor(lqcd_ctx* c, void* packed, const void* canonical, int parity, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!packed || !canonical || (parity | 1) != 1 || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "pack_spinor arguments");
  cudaSetDevice(c->device);
  cudaError_t e = run_pack_spinor(prec, (char*)packed, (const double*)canonical, c->nat, parity, 0, (cudaStream_t)stream);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "pack_spinor", e);
}

int lqcd_unpack_spinor(lqcd_ctx* c, void* canonical, const void* packed, int parity, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!packed || !canonical || (parity | 1) != 1 || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "unpack_spinor arguments");
  cudaSetDevice(c->device);
  cudaError_t e = run_pack_spinor(prec, (char*)packed, (const double*)canonical, c->nat, parity, 1, (cudaStream_t)stream);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "unpack_spinor", e);
}

int lqcd_dslash(lqcd_ctx* c, void* out, const void* in, int parity_out, int dagger, int prec, int recon, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity_out | 1) != 1) return fail(c, LQCD_EINVAL, "dslash arguments");
  cudaSetDevice(c->device);
  return op_dslash(c, (char*)out, (const char*)in, nullptr, parity_out, dagger ? 1 : 0, prec, recon, EPI_NONE, 0.0, 0.0,
                   false, (cudaStream_t)stream);
}

int lqcd_clover(lqcd_ctx* c, void* out, const void* in, int parity, int inverse, double kappa, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || (parity | 1) != 1) return fail(c, LQCD_EINVAL, "clover arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  const char *A, *Ai;
  int rc = get_clover(c, prec, kappa, false, &A, &Ai, s);
  if (rc) return rc;
  cudaError_t e = run_clover_apply(prec, (char*)out, (const char*)in, inverse ? Ai : A, c->nat, parity, s);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "clover_apply", e);
}

int lqcd_matpc_sym(lqcd_ctx* c, void* out, const void* in, int parity, int dagger, double kappa, int prec, int recon, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity | 1) != 1 || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "matpc_sym arguments");
  cudaSetDevice(c->device);
  return op_matpc(c, (char*)out, (const char*)in, parity, dagger ? 1 : 0, kappa, prec, recon, false, false, (cudaStream_t)stream, 1);
}

int lqcd_dslash_mrhs(lqcd_ctx* c, void* out, const void* in, int nrhs, int parity_out, int dagger, int prec, int recon, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity_out | 1) != 1) return fail(c, LQCD_EINVAL, "dslash_mrhs arguments");
  cudaSetDevice(c->device);
  return op_dslash_mrhs(c, (char*)out, (const char*)in, nullptr, nrhs, parity_out, dagger, prec, recon, EPI_NONE, 0.0, 0.0,
                        (cudaStream_t)stream);
}

int lqcd_matpc_mrhs(lqcd_ctx* c, void* out, const void* in, int nrhs, int parity, int dagger, double kappa, int prec, int recon,
                    void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity | 1) != 1 || nrhs < 1 || nrhs > LQCD_MAX_RHS || prec < 0 || prec > 2)
    return fail(c, LQCD_EINVAL, "matpc_mrhs arguments");
  cudaSetDevice(c->device);
  return op_matpc_mrhs(c, (char*)out, (const char*)in, nrhs, parity, dagger, kappa, prec, recon, (cudaStream_t)stream);
}

int lqcd_matpc(lqcd_ctx* c, void* out, const void* in, int parity, int dagger, double kappa, int prec, int recon, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity | 1) != 1) return fail(c, LQCD_EINVAL, "matpc arguments");
  cudaSetDevice(c->device);
  return op_matpc(c, (char*)out, (const char*)in, parity, dagger ? 1 : 0, kappa, prec, recon, false, false, (cudaStream_t)stream);
}

}  // extern "C"
