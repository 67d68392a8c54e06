// solver.cu -- the solvers the operator runs inside:
//   * mixed-precision BiCGstab with reliable updates  (reading R11)
//   * additive-Schwarz preconditioner K = n_MR minimum-residual steps on the Dirichlet-cut
//     Mhat_D, one alpha per block                      (reading R7)
//   * CGNR / CGNE with reliable updates                 ("CG on the normal equations")
//   * GCR-DD, Algorithm 1                               (reading R8)
//   * multiplicative Schwarz (SAP) as the alternative preconditioner (reading R16)
// The host loop only launches kernels; all Krylov scalars live on the device (blas_ops.cuh), two of BiCGstab's
// reductions ride in the operator's epilogue (dslash.cuh DOTS 2 / 3), and ||r||^2 reaches the host through zero-copy
// pinned words one iteration behind the device (solve_bicgstab); CGNR / CGNE / GCR read it back per iteration.
#include <cmath>
#include <complex>
#include <cstring>
#include <nvtx3/nvToolsExt.h>
#include "blas_ops.cuh"
#include "ops.h"

using namespace lq;

namespace {

typedef OpMrUpdate<true, false> OpMrFirst;
typedef OpMrUpdate<false, false> OpMrMid;
typedef OpMrUpdate<false, true> OpMrLast;
typedef OpMrUpdate<true, true> OpMrOnly;

// NVTX range around a solver phase (tracing); shows up in Nsight timelines, costs nothing without a tool attached
struct Range { explicit Range(const char* name) { nvtxRangePushA(name); } ~Range() { nvtxRangePop(); } };

struct EventPair { cudaEvent_t a = nullptr, b = nullptr; ~EventPair() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); } };

struct Work {                      // workspace of one call; goes back to the context's cache when it leaves scope
  lqcd_ctx* c;
  cudaStream_t s;
  std::vector<std::pair<void*, size_t>> bufs;
  Work(lqcd_ctx* c_, cudaStream_t s_) : c(c_), s(s_) {}
  ~Work() { for (auto& b : bufs) ws_put(c, b.first, b.second, s); }
  int get(char** out, size_t bytes) {
    void* p = nullptr;
    int rc = ws_get(c, &p, bytes, s);
    if (rc) return rc;
    bufs.push_back({p, bytes});
    *out = (char*)p;
    return LQCD_OK;
  }
};

BlasArgs mk(lqcd_ctx* c, bool blocked, char* v0 = nullptr, char* v1 = nullptr, char* v2 = nullptr, char* v3 = nullptr, char* v4 = nullptr) {
  BlasArgs a;
  memset(&a, 0, sizeof(a));
  a.v[0] = v0; a.v[1] = v1; a.v[2] = v2; a.v[3] = v3; a.v[4] = v4;
  const Geom& g = blocked ? c->bm.blk : c->nat;
  a.ns = g.ns; a.vh = g.vh; a.nb = g.nb;
  a.S = c->S; a.partials = c->partials; a.counters = c->counters;
  a.boxdots = c->boxdots;
  a.nchunk = (g.vh + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK * (LQ_DSLASH_BLOCK / 32);   // per-warp partials per box
  a.boxalpha = c->boxdots ? c->boxdots + (size_t)g.nb * a.nchunk * 4 : nullptr;         // behind the partials (set_blocks)
  return a;
}

template <class Op>
int blas(lqcd_ctx* c, int prec, const BlasArgs& a, cudaStream_t s) {
  cudaError_t e = run_blas<Op>(prec, a, c->n_sm * LQ_BLAS_CTAS_PER_SM, s);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "blas launch", e);
}

int mr_alpha(lqcd_ctx* c, const BlasArgs& a, cudaStream_t s) {
  cudaError_t e = run_mr_alpha(a, s);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "mr alpha launch", e);
}

int read_S(lqcd_ctx* c, int off, int n, cudaStream_t s) {
  cudaError_t e = cudaMemcpyAsync(c->hS + off, c->S + off, n * sizeof(double), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "scalar read-back", e);
}

int convert(lqcd_ctx* c, int pa, int pb, char* dst, const char* src, int dir, int parity, cudaStream_t s, int box0 = 0, int nbox = 0) {
  cudaError_t e = run_convert(pa, pb, dst, src, c->bm, dir, parity, s, box0, nbox);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "convert", e);
}

int norm2(lqcd_ctx* c, int prec, char* v, double* out, cudaStream_t s) {
  BlasArgs a = mk(c, false, v);
  int rc = blas<OpNorm2>(c, prec, a, s);
  if (rc) return rc;
  rc = read_S(c, S_OUT, 1, s);
  *out = c->hS[S_OUT];
  return rc;
}

// r = b - Mhat x in precision prec; returns ||r||
int residual(lqcd_ctx* c, char* r, const char* b, const char* x, int parity, double kappa, int prec, int recon,
             double* rn, cudaStream_t s) {
  int rc = op_matpc(c, r, x, parity, 0, kappa, prec, recon, false, false, s);
  if (rc) return rc;
  BlasArgs a = mk(c, false, const_cast<char*>(b), r);
  rc = blas<OpXmyNorm>(c, prec, a, s);
  if (rc) return rc;
  rc = read_S(c, S_OUT, 1, s);
  *rn = sqrt(c->hS[S_OUT]);
  return rc;
}

struct Counts { long long mat_sloppy = 0, mat_outer = 0, mat_precond = 0; double blas_flop_sites = 0; };

// Symmetric even-odd form (lqcd.h LQCD_MATPC_SYMMETRIC): the Krylov iteration runs on
// Mhat_s x = A^-1 bhat, whose residual is r_s = A^-1 (bhat - Mhat x).  Called right after residual():
// r <- A_pp^-1 r in place (outer precision) and *rsn = ||r_s||.  The convergence test stays on ||bhat - Mhat x||.
int to_symmetric_residual(lqcd_ctx* c, char* r, int parity, double kappa, int prec, double* rsn, cudaStream_t s) {
  const char *A, *Ai;
  int rc = get_clover(c, prec, kappa, false, &A, &Ai, s);
  if (rc) return rc;
  cudaError_t e = run_clover_apply(prec, r, r, Ai, c->nat, parity, s); c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "clover_apply", e);
  double n2;
  if ((rc = norm2(c, prec, r, &n2, s))) return rc;
  *rsn = sqrt(n2);
  return LQCD_OK;
}

}  // namespace

namespace lq {

// out = K in  (reading R7).  in/out: natural layout, precision prec_io.  rho, w, xk: block-major
// workspace in precision prec (allocated by the caller).
int schwarz_apply(lqcd_ctx* c, char* out, const char* in, int parity, double kappa, int n_mr, double omega,
                  int prec, int recon, int prec_io, char* rho, char* w, char* xk, cudaStream_t s) {
  Range nv("lqcd: Schwarz preconditioner K");
  int rc = convert(c, prec_io, prec, rho, in, 1, parity, s);
  if (rc) return rc;
  // Block-group schedule ("multiple levels of Schwarz-type blocking to take advantage of the multiple
  // levels of memory locality"): the blocks are independent, so all n_mr steps can run on a group of
  // `group` blocks -- sized so that the group's spinors, links and clover blocks stay in L2 -- before the next group
  // is touched.  The block-major layout makes a group a contiguous box range.  group = 0: all blocks per launch.
  const int nb = c->bm.blk.nb;
  const int group = (c->schwarz_group > 0 && c->schwarz_group < nb) ? c->schwarz_group : nb;
  for (int b0 = 0; b0 < nb; b0 += group) {
    const int gn = (b0 + group <= nb) ? group : nb - b0;
    const int box0 = group == nb ? 0 : b0, nbox = group == nb ? 0 : gn;
    for (int step = 0; step < n_mr; ++step) {
      rc = op_matpc(c, w, rho, parity, 0, kappa, prec, recon, true, true, s, 0, 0, nullptr, box0, nbox);
      if (rc) return rc;
      BlasArgs a = mk(c, true, xk, rho, w);
      a.c[0] = omega;
      if (nbox) { a.box0 = box0; a.nb = nbox; }
      if ((rc = mr_alpha(c, a, s))) return rc;
      const bool first = step == 0, last = step == n_mr - 1;
      if (first && last) rc = blas<OpMrOnly>(c, prec, a, s);
      else if (first) rc = blas<OpMrFirst>(c, prec, a, s);
      else if (last) rc = blas<OpMrLast>(c, prec, a, s);
      else rc = blas<OpMrMid>(c, prec, a, s);
      if (rc) return rc;
    }
  }
  return convert(c, prec, prec_io, out, xk, 2, parity, s);
}

// out = K_sap in: multiplicative Schwarz (SAP; PAPER.md:158 section 4, :146; reading R16).  n_cycle cycles over the two
// block colours; the blocks of one colour are a contiguous box range of the colour-major block layout (host.h), so a
// half-step is the additive machinery launched on that range; after it the residual is updated with the FULL operator:
//   rho = r restricted to colour c;  y = MR^{n_mr}(Mhat_D) rho;  out += y;  r -= Mhat y.
// in / out / r / y / t: natural layout, precision prec_io; rho, w, xk: block-major, precision prec.
int schwarz_sap_apply(lqcd_ctx* c, char* out, const char* in, int parity, double kappa, int n_mr, double omega, int n_cycle,
                      int prec, int recon, int prec_io, int recon_io, char* rho, char* w, char* xk, char* r, char* y, char* t,
                      cudaStream_t s) {
  Range nv("lqcd: multiplicative Schwarz K_sap");
  if (!c->bm.cmaj) return fail(c, LQCD_ESTATE, "multiplicative Schwarz needs the colour-major block layout");
  const int nb = c->bm.blk.nb, half = nb / 2;
  int rc = convert(c, prec_io, prec_io, r, in, 0, parity, s);
  if (rc) return rc;
  { BlasArgs a = mk(c, false, out); if ((rc = blas<OpZero>(c, prec_io, a, s))) return rc; }
  for (int cyc = 0; cyc < n_cycle; ++cyc)
    for (int col = 0; col < 2; ++col) {
      const int box0 = col * half, nbox = half;
      // only this colour's boxes are computed below, so the other colour's part of rho need not be cleared
      if ((rc = convert(c, prec_io, prec, rho, r, 1, parity, s))) return rc;
      for (int step = 0; step < n_mr; ++step) {
        if ((rc = op_matpc(c, w, rho, parity, 0, kappa, prec, recon, true, true, s, 0, 0, nullptr, box0, nbox))) return rc;
        BlasArgs a = mk(c, true, xk, rho, w);
        a.c[0] = omega; a.box0 = box0; a.nb = nbox;
        if ((rc = mr_alpha(c, a, s))) return rc;
        const bool first = step == 0, last = step == n_mr - 1;
        if (first && last) rc = blas<OpMrOnly>(c, prec, a, s);
        else if (first) rc = blas<OpMrFirst>(c, prec, a, s);
        else if (last) rc = blas<OpMrLast>(c, prec, a, s);
        else rc = blas<OpMrMid>(c, prec, a, s);
        if (rc) return rc;
      }
      if ((rc = convert(c, prec, prec_io, y, xk, 2, parity, s, box0, nbox))) return rc;       // zero on the other colour
      { BlasArgs a = mk(c, false, y, out); a.c[0] = 1.0; if ((rc = blas<OpAxpyNorm>(c, prec_io, a, s))) return rc; }
      if (cyc == n_cycle - 1 && col == 1) break;                                             // the last residual is not needed
      if ((rc = op_matpc(c, t, y, parity, 0, kappa, prec_io, recon_io, false, false, s))) return rc;
      { BlasArgs a = mk(c, false, t, r); a.c[0] = -1.0; if ((rc = blas<OpAxpyNorm>(c, prec_io, a, s))) return rc; }
    }
  return LQCD_OK;
}

}  // namespace lq

namespace {

// ---------------------------------------------------------------- BiCGstab with reliable updates
int solve_bicgstab(lqcd_ctx* c, char* x, const char* b, const lqcd_invert_params& p, double stop,
                   lqcd_invert_result* res, Counts& cnt, cudaStream_t s) {
  const int po = p.prec_outer, ps = p.prec_sloppy, par = p.parity;
  const long long ns = c->nat.ns;
  Work wk(c, s);
  char *r_hi, *xl, *rl, *rt, *pv, *v, *t;
  int rc;
  if ((rc = wk.get(&r_hi, spinor_bytes(po, ns)))) return rc;
  char** lo[] = {&xl, &rl, &rt, &pv, &v, &t};
  for (char** q : lo) if ((rc = wk.get(q, spinor_bytes(ps, ns)))) return rc;
  const int sym = p.matpc_type == LQCD_MATPC_SYMMETRIC;
  double rn, rin, istop = stop;       // rin, istop: norm and stopping threshold of the residual the inner iteration sees
  // true residual in the outer precision; symmetric form: hand A^-1 r to the inner iteration and scale its threshold
  auto true_residual = [&]() -> int {
    Range nv("lqcd: true residual (outer precision)");
    int rc2 = residual(c, r_hi, b, x, par, p.kappa, po, p.recon_outer, &rn, s);
    if (rc2) return rc2;
    cnt.mat_outer++;
    rin = rn;
    if (sym && rn > stop) {
      if ((rc2 = to_symmetric_residual(c, r_hi, par, p.kappa, po, &rin, s))) return rc2;
      istop = stop * (rin / rn);
    }
    return LQCD_OK;
  };
  if ((rc = true_residual())) return rc;
  res->iterations = 0; res->restarts = 0;
  const double delta = p.delta > 0 ? p.delta : 0.1;
  int status = LQCD_OK;
  if (rn > stop) {
    if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
    if ((rc = convert(c, ps, ps, rt, rl, 0, par, s))) return rc;
    for (char* z : {xl, pv, v}) { BlasArgs a = mk(c, false, z); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
    { BlasArgs a = mk(c, false, rt, rl); a.i0 = 0; if ((rc = blas<OpBicgInit>(c, ps, a, s))) return rc; }
    double maxr = rin;
    const double r_start = rn;                // divergence guard: BiCGstab can blow up on an indefinite operator (kappa > kappa_c)
    // The host decides on reliable updates and convergence from ||r_l||^2 and the breakdown flag of every iteration,
    // but it reads them ONE ITERATION LATE: iteration k+1 is enqueued before the host waits for the scalars of
    // iteration k, so the device never idles on the read-back (it cost 38 us of a 730 us iteration).  An update then
    // happens one iteration after its trigger; that iteration is an ordinary BiCGstab step and is folded into x with
    // the rest, so only the very last one of a solve is spent for nothing.
    // The scalars travel through pinned host memory the last CTA of the iteration's final kernel writes directly
    // (blas_ops.cuh OpBicgXR::publish): no memcpy and no event sits between two kernels of the stream.
    volatile double* hs = c->hS + S_TOTAL;    // pinned: words 4 (k & 1) .. +2 hold (rr, flag, k) of iteration k
    hs[2] = hs[6] = -1.0;
    auto fold = [&]() -> int {                // x += x_l (outer precision)
      MultiArgs m; memset(&m, 0, sizeof(m));
      m.b = mk(c, false); m.z[0] = xl; m.chi[0] = 1.0; m.n = 1;
      cudaError_t e = run_accumulate(po, ps, x, m, s); c->launches++;
      return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "accumulate", e);
    };
    auto enqueue = [&](int k) -> int {        // iteration k (1-based): kernels, then the asynchronous read-back of its scalars
      int rc2;
      { BlasArgs a = mk(c, false, pv, rl, v); if ((rc2 = blas<OpBicgP>(c, ps, a, s))) return rc2; }
      if (!sym) {
        // <rtilde, v> -> alpha and (<t,s>, <t,t>) -> omega are reduced in the second launch of Mhat (dslash.cuh DOTS 3 / 2)
        if ((rc2 = op_matpc(c, v, pv, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, 0, FIN_BICG_ALPHA, rt))) return rc2;
      } else {
        if ((rc2 = op_matpc(c, v, pv, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc2;
        BlasArgs a = mk(c, false, rt, v); if ((rc2 = blas<OpBicgAlpha>(c, ps, a, s))) return rc2;
      }
      { BlasArgs a = mk(c, false, rl, v); if ((rc2 = blas<OpBicgS>(c, ps, a, s))) return rc2; }
      if (!sym) {
        if ((rc2 = op_matpc(c, t, rl, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, 0, FIN_BICG_OMEGA, nullptr))) return rc2;
      } else {
        if ((rc2 = op_matpc(c, t, rl, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc2;
        BlasArgs a = mk(c, false, t, rl); if ((rc2 = blas<OpBicgOmega>(c, ps, a, s))) return rc2;
      }
      { BlasArgs a = mk(c, false, xl, pv, rl, t, rt); a.i0 = k; a.hmirror = c->hS + S_TOTAL;
        if ((rc2 = blas<OpBicgXR>(c, ps, a, s))) return rc2; }
      cnt.mat_sloppy += 2; cnt.blas_flop_sites += 1056;
      return LQCD_OK;
    };
    auto wait_for = [&](int k) -> int {       // spin until iteration k has published; a failed stream ends the wait
      long long spins = 0;
      while (hs[4 * (k & 1) + 2] != (double)k) {
        if ((++spins & 0xfffff) == 0 && cudaStreamQuery(s) != cudaErrorNotReady) {
          if (hs[4 * (k & 1) + 2] == (double)k) break;
          return fail(c, LQCD_ECUDA, "scalar read-back", cudaGetLastError());
        }
      }
      return LQCD_OK;
    };
    int it = 0, seen = 0;                     // iterations enqueued / examined by the host
    while (true) {
      const bool can = it < p.max_iter;
      if (can) { if ((rc = enqueue(it + 1))) return rc; ++it; }
      const int upto = can ? it - 1 : it;     // keep one iteration in flight unless the cap is reached
      bool trigger = false;
      while (seen < upto && !trigger) {
        ++seen;
        if ((rc = wait_for(seen))) return rc;
        const double rr = hs[4 * (seen & 1)], flag = hs[4 * (seen & 1) + 1];
        if (!(rr == rr) || flag != 0.0) status = LQCD_EBREAKDOWN;
        const double rln = sqrt(rr);
        c->hist.push_back(rln);
        if (rln > maxr) maxr = rln;
        trigger = status == LQCD_EBREAKDOWN || rln <= istop || rln < delta * maxr;
      }
      if (!trigger) {
        if (can || seen < it) continue;
        // iteration cap: fold what the low-precision iteration has accumulated since the last reliable update
        // into x, so that the caller gets the best iterate and its true residual
        if ((rc = fold())) return rc;
        status = LQCD_ENOCONV;
        break;
      }
      // reliable update: fold x_l into x (everything enqueued so far), recompute the true residual in the outer precision
      while (seen < it) {                      // the iteration in flight belongs to the history as well
        ++seen;
        if ((rc = wait_for(seen))) return rc;
        c->hist.push_back(sqrt(hs[4 * (seen & 1)]));
      }
      if ((rc = fold())) return rc;
      { BlasArgs a = mk(c, false, xl); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
      if ((rc = true_residual())) return rc;
      res->restarts++;
      if (rn <= stop) { status = LQCD_OK; break; }
      if (rn > 1e5 * r_start) { status = LQCD_EBREAKDOWN; break; }      // the true residual has grown 1e5-fold: give up
      if (!(rn == rn)) { status = LQCD_EBREAKDOWN; break; }
      if (status == LQCD_EBREAKDOWN) {
        // restart the recurrence from the true residual
        status = LQCD_OK;
        if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
        if ((rc = convert(c, ps, ps, rt, rl, 0, par, s))) return rc;
        for (char* z : {pv, v}) { BlasArgs a = mk(c, false, z); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
        BlasArgs a = mk(c, false, rt, rl); a.i0 = 0; if ((rc = blas<OpBicgInit>(c, ps, a, s))) return rc;
      } else {
        if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
        BlasArgs a = mk(c, false, rt, rl); a.i0 = 1; if ((rc = blas<OpBicgInit>(c, ps, a, s))) return rc;
      }
      maxr = rin;
      if (!can) {                              // the cap was reached and this update did not converge
        status = LQCD_ENOCONV;
        break;
      }
    }
    res->iterations = it;
  }
  res->iterated_residual = rn;
  return status;
}

// ---------------------------------------------------------------- CGNR with reliable updates
// CG on Mhat^dag Mhat x = Mhat^dag bhat.  The residual of the ORIGINAL system
// r = bhat - Mhat x is carried in low precision and replaced by the true fp64 residual at reliable
// updates (same trigger as BiCGstab, R11); the search direction is kept across updates with
// beta = ||z_new||^2 / ||z_old||^2.  Per iteration: Mhat p, Mhat^dag r and four fused BLAS-1 passes.
int solve_cgnr(lqcd_ctx* c, char* x, const char* b, const lqcd_invert_params& p, double stop,
               lqcd_invert_result* res, Counts& cnt, cudaStream_t s) {
  const int po = p.prec_outer, ps = p.prec_sloppy, par = p.parity;
  const long long ns = c->nat.ns;
  Work wk(c, s);
  char *r_hi, *xl, *rl, *z, *pv, *w;
  int rc;
  if ((rc = wk.get(&r_hi, spinor_bytes(po, ns)))) return rc;
  char** lo[] = {&xl, &rl, &z, &pv, &w};
  for (char** q : lo) if ((rc = wk.get(q, spinor_bytes(ps, ns)))) return rc;
  const int sym = p.matpc_type == LQCD_MATPC_SYMMETRIC;
  double rn, rin, istop = stop;
  auto true_residual = [&]() -> int {      // as in solve_bicgstab
    Range nv("lqcd: true residual (outer precision)");
    int rc2 = residual(c, r_hi, b, x, par, p.kappa, po, p.recon_outer, &rn, s);
    if (rc2) return rc2;
    cnt.mat_outer++;
    rin = rn;
    if (sym && rn > stop) {
      if ((rc2 = to_symmetric_residual(c, r_hi, par, p.kappa, po, &rin, s))) return rc2;
      istop = stop * (rin / rn);
    }
    return LQCD_OK;
  };
  if ((rc = true_residual())) return rc;
  res->iterations = 0; res->restarts = 0;
  const double delta = p.delta > 0 ? p.delta : 0.1;
  int status = LQCD_OK;
  auto fold = [&]() -> int {            // x += x_l (outer precision), x_l = 0
    MultiArgs m; memset(&m, 0, sizeof(m));
    m.b = mk(c, false); m.z[0] = xl; m.chi[0] = 1.0; m.n = 1;
    cudaError_t e = run_accumulate(po, ps, x, m, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "accumulate", e);
    BlasArgs a = mk(c, false, xl);
    return blas<OpZero>(c, ps, a, s);
  };
  if (rn > stop) {
    if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
    for (char* q : {xl, pv}) { BlasArgs a = mk(c, false, q); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
    if ((rc = op_matpc(c, z, rl, par, 1, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc;
    cnt.mat_sloppy++;
    { BlasArgs a = mk(c, false, z); a.i0 = 0; if ((rc = blas<OpCgInit>(c, ps, a, s))) return rc; }
    { BlasArgs a = mk(c, false, pv, z); if ((rc = blas<OpCgP>(c, ps, a, s))) return rc; }      // beta = 0: p = z
    double maxr = rin;
    int it = 0;
    while (true) {
      if (it >= p.max_iter) { if ((rc = fold())) return rc; status = LQCD_ENOCONV; break; }
      if (!sym) {                               // ||w||^2 -> alpha reduced in the second launch of Mhat (dslash.cuh DOTS 2)
        if ((rc = op_matpc(c, w, pv, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, 0, FIN_CG_ALPHA, nullptr))) return rc;
      } else {
        if ((rc = op_matpc(c, w, pv, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc;
        BlasArgs a = mk(c, false, w); if ((rc = blas<OpCgAlpha>(c, ps, a, s))) return rc;
      }
      { BlasArgs a = mk(c, false, xl, pv, rl, w); if ((rc = blas<OpCgXR>(c, ps, a, s))) return rc; }
      cnt.mat_sloppy++; cnt.blas_flop_sites += 24.0 * (2 + 4 + 2); ++it;
      if ((rc = read_S(c, S_RR, 2, s))) return rc;
      const double rr = c->hS[S_RR], flag = c->hS[S_FLAG];
      if (!(rr == rr) || flag != 0.0) status = LQCD_EBREAKDOWN;
      const double rln = sqrt(rr);
      c->hist.push_back(rln);
      if (rln > maxr) maxr = rln;
      if (status == LQCD_EBREAKDOWN || rln <= istop || rln < delta * maxr) {
        if ((rc = fold())) return rc;
        if ((rc = true_residual())) return rc;
        res->restarts++;
        if (rn <= stop) { status = LQCD_OK; break; }
        if (!(rn == rn)) { status = LQCD_EBREAKDOWN; break; }
        if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
        maxr = rin;
      }
      // z = Mhat^dag r ; beta = <z,z>/<z,z>_old ; p = z + beta p   (after a breakdown: restart, beta = 0)
      if ((rc = op_matpc(c, z, rl, par, 1, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc;
      cnt.mat_sloppy++;
      { BlasArgs a = mk(c, false, z); a.i0 = (status == LQCD_EBREAKDOWN) ? 0 : 1; if ((rc = blas<OpCgInit>(c, ps, a, s))) return rc; }
      status = LQCD_OK;
      { BlasArgs a = mk(c, false, pv, z); if ((rc = blas<OpCgP>(c, ps, a, s))) return rc; }
      cnt.blas_flop_sites += 24.0 * (2 + 2);
    }
    res->iterations = it;
  }
  res->iterated_residual = rn;
  return status;
}

// ---------------------------------------------------------------- CGNE (Craig's method) with reliable updates
// CG on Mhat Mhat^dag y = bhat with x = Mhat^dag y carried directly ("CGNE or CGNR"):
// alpha = <r,r>/<p,p>; x += alpha p; r -= alpha Mhat p; beta = <r',r'>/<r,r>; p = Mhat^dag r' + beta p.
// Minimises the error instead of the residual.  Same precision scheme and BLAS-1 passes as CGNR.
int solve_cgne(lqcd_ctx* c, char* x, const char* b, const lqcd_invert_params& p, double stop,
               lqcd_invert_result* res, Counts& cnt, cudaStream_t s) {
  const int po = p.prec_outer, ps = p.prec_sloppy, par = p.parity;
  const long long ns = c->nat.ns;
  Work wk(c, s);
  char *r_hi, *xl, *rl, *z, *pv, *w;
  int rc;
  if ((rc = wk.get(&r_hi, spinor_bytes(po, ns)))) return rc;
  char** lo[] = {&xl, &rl, &z, &pv, &w};
  for (char** q : lo) if ((rc = wk.get(q, spinor_bytes(ps, ns)))) return rc;
  const int sym = p.matpc_type == LQCD_MATPC_SYMMETRIC;
  double rn, rin, istop = stop;
  auto true_residual = [&]() -> int {      // as in solve_bicgstab
    Range nv("lqcd: true residual (outer precision)");
    int rc2 = residual(c, r_hi, b, x, par, p.kappa, po, p.recon_outer, &rn, s);
    if (rc2) return rc2;
    cnt.mat_outer++;
    rin = rn;
    if (sym && rn > stop) {
      if ((rc2 = to_symmetric_residual(c, r_hi, par, p.kappa, po, &rin, s))) return rc2;
      istop = stop * (rin / rn);
    }
    return LQCD_OK;
  };
  if ((rc = true_residual())) return rc;
  res->iterations = 0; res->restarts = 0;
  const double delta = p.delta > 0 ? p.delta : 0.1;
  int status = LQCD_OK;
  auto fold = [&]() -> int {
    MultiArgs m; memset(&m, 0, sizeof(m));
    m.b = mk(c, false); m.z[0] = xl; m.chi[0] = 1.0; m.n = 1;
    cudaError_t e = run_accumulate(po, ps, x, m, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "accumulate", e);
    BlasArgs a = mk(c, false, xl);
    return blas<OpZero>(c, ps, a, s);
  };
  // (re)start or continue the direction from the low-precision residual r_l: rr (and beta) on the device,
  // z = Mhat^dag r_l, p = z + beta p.   keep = 0: beta = 0
  auto direction = [&](int keep) -> int {
    BlasArgs a = mk(c, false, rl); a.i0 = keep;
    int rc2 = blas<OpCgInit>(c, ps, a, s);
    if (rc2) return rc2;
    if ((rc2 = op_matpc(c, z, rl, par, 1, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc2;
    cnt.mat_sloppy++;
    BlasArgs a2 = mk(c, false, pv, z);
    return blas<OpCgP>(c, ps, a2, s);
  };
  if (rn > stop) {
    if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
    for (char* q : {xl, pv}) { BlasArgs a = mk(c, false, q); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
    if ((rc = direction(0))) return rc;
    double maxr = rin;
    int it = 0;
    while (true) {
      if (it >= p.max_iter) { if ((rc = fold())) return rc; status = LQCD_ENOCONV; break; }
      { BlasArgs a = mk(c, false, pv); if ((rc = blas<OpCgAlpha>(c, ps, a, s))) return rc; }          // alpha = rr / ||p||^2
      if ((rc = op_matpc(c, w, pv, par, 0, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc;
      { BlasArgs a = mk(c, false, xl, pv, rl, w); if ((rc = blas<OpCgXRB>(c, ps, a, s))) return rc; }   // x, r, rr', beta
      cnt.mat_sloppy++; cnt.blas_flop_sites += 24.0 * (2 + 4 + 2); ++it;
      if ((rc = read_S(c, S_RR, 2, s))) return rc;
      const double rr = c->hS[S_RR], flag = c->hS[S_FLAG];
      const bool bad = !(rr == rr) || flag != 0.0;
      const double rln = sqrt(rr);
      c->hist.push_back(rln);
      if (rln > maxr) maxr = rln;
      bool replaced = false;
      if (bad || rln <= istop || rln < delta * maxr) {
        if ((rc = fold())) return rc;
        if ((rc = true_residual())) return rc;
        res->restarts++;
        if (rn <= stop) { status = LQCD_OK; break; }
        if (!(rn == rn)) { status = LQCD_EBREAKDOWN; break; }
        if ((rc = convert(c, po, ps, rl, r_hi, 0, par, s))) return rc;
        maxr = rin;
        replaced = true;
      }
      if (replaced) {
        if ((rc = direction(bad ? 0 : 2))) return rc;       // beta rescaled to the new residual (0 after a breakdown)
      } else {
        if ((rc = op_matpc(c, z, rl, par, 1, p.kappa, ps, p.recon_sloppy, false, false, s, sym))) return rc;
        cnt.mat_sloppy++;
        BlasArgs a = mk(c, false, pv, z);
        if ((rc = blas<OpCgP>(c, ps, a, s))) return rc;
      }
      cnt.blas_flop_sites += 24.0 * 2;
    }
    res->iterations = it;
  }
  res->iterated_residual = rn;
  return status;
}

// ---------------------------------------------------------------- GCR-DD (Algorithm 1)
int solve_gcr(lqcd_ctx* c, char* x, const char* b, const lqcd_invert_params& p, double stop,
              lqcd_invert_result* res, Counts& cnt, cudaStream_t s) {
  const int po = p.prec_outer, ps = p.prec_sloppy, pp = p.prec_precond, par = p.parity;
  const long long ns = c->nat.ns;
  const int kmax = p.gcr_kmax > 0 ? p.gcr_kmax : 16;
  if (kmax > LQ_GCR_KMAX) return fail(c, LQCD_EINVAL, "gcr_kmax too large");
  const double delta = p.delta > 0 ? p.delta : 0.1;
  Work wk(c, s);
  int rc;
  char *r0, *rh, *rho = nullptr, *w = nullptr, *xk = nullptr;
  std::vector<char*> ph(kmax), zh(kmax);
  if ((rc = wk.get(&r0, spinor_bytes(po, ns)))) return rc;
  if ((rc = wk.get(&rh, spinor_bytes(ps, ns)))) return rc;
  for (int i = 0; i < kmax; ++i) {
    if ((rc = wk.get(&ph[i], spinor_bytes(ps, ns)))) return rc;
    if ((rc = wk.get(&zh[i], spinor_bytes(ps, ns)))) return rc;
  }
  const bool sap = p.precondition && p.schwarz_type == LQCD_SCHWARZ_MULTIPLICATIVE;
  // the solve's group size must not outlive it (lqcd_set_schwarz_group is the context-level setting)
  struct GroupGuard { lqcd_ctx* c; int saved, saved_ovl; bool armed; ~GroupGuard() { if (armed) { c->schwarz_group = saved; c->schwarz_overlap = saved_ovl; } } }
      group_guard{c, c->schwarz_group, c->schwarz_overlap, false};
  char *sr = nullptr, *sy = nullptr, *st = nullptr;
  if (p.precondition) {
    if (p.schwarz_group < 0) return fail(c, LQCD_EINVAL, "schwarz_group");
    group_guard.armed = true;
    c->schwarz_group = p.schwarz_group;
    if (p.schwarz_overlap < 0 || (sap && p.schwarz_overlap)) return fail(c, LQCD_EINVAL, "schwarz_overlap");
    c->schwarz_overlap = p.schwarz_overlap;
    if ((rc = set_blocks(c, p.schwarz_block, sap ? 1 : 0, c->schwarz_overlap))) return rc;
    for (char** q : {&rho, &w, &xk}) if ((rc = wk.get(q, spinor_bytes(pp, c->bm.blk.ns)))) return rc;   // block-major: grown domains
    if (sap) for (char** q : {&sr, &sy, &st}) if ((rc = wk.get(q, spinor_bytes(ps, ns)))) return rc;
  }
  double r0n;
  if ((rc = residual(c, r0, b, x, par, p.kappa, po, p.recon_outer, &r0n, s))) return rc;
  cnt.mat_outer++;
  int total = 0, status = LQCD_OK;
  res->restarts = 0;
  while (r0n > stop) {
    if (total >= p.max_iter) { status = LQCD_ENOCONV; break; }
    if (!(r0n == r0n)) { status = LQCD_EBREAKDOWN; break; }
    if ((rc = convert(c, po, ps, rh, r0, 0, par, s))) return rc;
    int k = 0;
    while (true) {
      // p_k = K rhat
      if (sap) {
        const int ncyc = p.sap_cycles > 0 ? p.sap_cycles : 1;
        if ((rc = schwarz_sap_apply(c, ph[k], rh, par, p.kappa, p.mr_steps, p.mr_omega, ncyc, pp, p.recon_precond, ps, p.recon_sloppy,
                                    rho, w, xk, sr, sy, st, s))) return rc;
        // each half-step runs the MR steps on half of the blocks: one cycle = mr_steps Mhat_D on the whole lattice
        cnt.mat_precond += p.mr_steps * ncyc; cnt.mat_sloppy += 2 * ncyc - 1;
        cnt.blas_flop_sites += ncyc * (p.mr_steps * (12.0 * 16 + 12.0 * 12) + 4 * 48.0);
      } else if (p.precondition) {
        if ((rc = schwarz_apply(c, ph[k], rh, par, p.kappa, p.mr_steps, p.mr_omega, pp, p.recon_precond, ps, rho, w, xk, s))) return rc;
        cnt.mat_precond += p.mr_steps; cnt.blas_flop_sites += p.mr_steps * (12.0 * 16 + 12.0 * 12);
      } else if ((rc = convert(c, ps, ps, ph[k], rh, 0, par, s))) return rc;
      // z_k = Mhat p_k
      if ((rc = op_matpc(c, zh[k], ph[k], par, 0, p.kappa, ps, p.recon_sloppy, false, false, s))) return rc;
      cnt.mat_sloppy++;
      // orthogonalise (one batched pass: classical Gram-Schmidt), normalise, update rhat
      MultiArgs m; memset(&m, 0, sizeof(m));
      m.b = mk(c, false, rh);
      for (int i = 0; i <= k; ++i) m.z[i] = zh[i];
      m.k = k;
      for (int i0 = 0; i0 < k; i0 += 8) {
        m.i0 = i0; m.n = (k - i0 < 8) ? k - i0 : 8;
        cudaError_t e = run_gcr_dots(ps, m, c->n_sm * LQ_BLAS_CTAS_PER_SM, s); c->launches++;
        if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "gcr dots", e);
      }
      { cudaError_t e = run_gcr_orth(ps, m, c->n_sm * LQ_BLAS_CTAS_PER_SM, s); c->launches++;
        if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "gcr orth", e); }
      { BlasArgs a = mk(c, false, zh[k], rh); if ((rc = blas<OpGcrScale>(c, ps, a, s))) return rc; }
      cnt.blas_flop_sites += 12.0 * (16.0 * k + 12 + 14);
      ++k; ++total;
      if ((rc = read_S(c, S_RR, 1, s))) return rc;
      const double rhn = sqrt(c->hS[S_RR]);
      c->hist.push_back(rhn);
      if (k == kmax || rhn / r0n < delta || rhn < stop || total >= p.max_iter || !(rhn == rhn)) break;
    }
    // implicit solution update: back-substitution for chi, then x += sum chi_i p_i
    if ((rc = read_S(c, S_GCR_BETA, S_TOTAL - S_GCR_BETA, s))) return rc;
    std::complex<double> chi[LQ_GCR_KMAX];
    for (int l = k - 1; l >= 0; --l) {
      std::complex<double> tacc(c->hS[S_GCR_ALPHAS + 2 * l], c->hS[S_GCR_ALPHAS + 2 * l + 1]);
      for (int i = l + 1; i < k; ++i)
        tacc -= std::complex<double>(c->hS[S_GCR_BETA + 2 * (l * LQ_GCR_KMAX + i)], c->hS[S_GCR_BETA + 2 * (l * LQ_GCR_KMAX + i) + 1]) * chi[i];
      const double gl = c->hS[S_GCR_GAMMAS + l];
      chi[l] = gl > 0.0 ? tacc / gl : std::complex<double>(0.0, 0.0);     // gamma_l = 0: z_l was exactly zero (blas.cu)
    }
    MultiArgs m; memset(&m, 0, sizeof(m));
    m.b = mk(c, false);
    for (int i = 0; i < k; ++i) { m.z[i] = ph[i]; m.chi[2 * i] = chi[i].real(); m.chi[2 * i + 1] = chi[i].imag(); }
    m.n = k;
    cudaError_t e = run_accumulate(po, ps, x, m, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "accumulate", e);
    if ((rc = residual(c, r0, b, x, par, p.kappa, po, p.recon_outer, &r0n, s))) return rc;
    cnt.mat_outer++; res->restarts++;
  }
  res->iterations = total;
  res->iterated_residual = r0n;
  return status;
}

// ---------------------------------------------------------------- batched BiCGstab (several right-hand sides)
// nrhs independent BiCGstab recurrences advanced in lockstep: the operator is applied to all of them
// with the multi-right-hand-side kernels (one link load per 4 sources, dslash_mrhs.cuh), the five
// fused BLAS-1 passes of an iteration run as one launch each over gridDim.z = nrhs with one set of
// device scalars per source.  A reliable update (R11) is taken for all sources as soon as one asks for
// it; a converged source is frozen (S_DONE) and its passes return at once.  x, b: nrhs packed fields.
BlasArgs mkb(lqcd_ctx* c, int prec, char* v0 = nullptr, char* v1 = nullptr, char* v2 = nullptr, char* v3 = nullptr, char* v4 = nullptr) {
  BlasArgs a = mk(c, false, v0, v1, v2, v3, v4);
  a.rhs_bytes = (long long)spinor_bytes(prec, c->nat.ns);
  a.rhs_partials = (long long)c->partials_doubles;
  return a;
}
BlasArgs mkr(lqcd_ctx* c, int r, char* v0 = nullptr, char* v1 = nullptr, char* v2 = nullptr, char* v3 = nullptr, char* v4 = nullptr) {
  BlasArgs a = mk(c, false, v0, v1, v2, v3, v4);           // single launch on the scalar set of source r
  a.S = c->S + (long long)r * S_TOTAL;
  a.partials = c->partials + (long long)r * c->partials_doubles;
  a.counters = c->counters + r;
  return a;
}
template <class Op>
int blasb(lqcd_ctx* c, int prec, const BlasArgs& a, int nrhs, cudaStream_t s) {
  cudaError_t e = run_blas<Op>(prec, a, c->n_sm * LQ_BLAS_CTAS_PER_SM, s, nrhs);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "batched blas launch", e);
}
// hS[S_TOTAL + 2r .. +1] = S_r[off], S_r[off+1] for all sources (one strided copy), synchronises
int read_S_all(lqcd_ctx* c, int off, int nrhs, cudaStream_t s) {
  cudaError_t e = cudaMemcpy2DAsync(c->hS + S_TOTAL, 2 * sizeof(double), c->S + off, S_TOTAL * sizeof(double),
                                    2 * sizeof(double), nrhs, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "scalar read-back", e);
}
int set_done(lqcd_ctx* c, int r, double v, cudaStream_t s) {
  double* h = c->hS + S_TOTAL + 2 * LQCD_MAX_RHS + r;       // pinned staging word of source r
  *h = v;
  cudaError_t e = cudaMemcpyAsync(c->S + (long long)r * S_TOTAL + S_DONE, h, sizeof(double), cudaMemcpyHostToDevice, s);
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "flag write", e);
}

// r_hi = b - Mhat x for all sources (outer precision); rn[r] = ||r_hi[r]||
int residual_mrhs(lqcd_ctx* c, char* r_hi, const char* b, const char* x, int nrhs, int par, double kappa, int prec, int recon,
                  double* rn, cudaStream_t s) {
  int rc = op_matpc_mrhs(c, r_hi, x, nrhs, par, 0, kappa, prec, recon, s);
  if (rc) return rc;
  const size_t fb = spinor_bytes(prec, c->nat.ns);
  for (int r = 0; r < nrhs; ++r) {
    BlasArgs a = mkr(c, r, const_cast<char*>(b) + r * fb, r_hi + r * fb);
    if ((rc = blas<OpXmyNorm>(c, prec, a, s))) return rc;
  }
  if ((rc = read_S_all(c, S_OUT, nrhs, s))) return rc;
  for (int r = 0; r < nrhs; ++r) rn[r] = sqrt(c->hS[S_TOTAL + 2 * r]);
  return LQCD_OK;
}

int solve_bicgstab_mrhs(lqcd_ctx* c, char* x, const char* b, int nrhs, const lqcd_invert_params& p, const double* stop,
                        lqcd_invert_result* res, Counts& cnt, cudaStream_t s) {
  const int po = p.prec_outer, ps = p.prec_sloppy, par = p.parity;
  const long long ns = c->nat.ns;
  const size_t fo = spinor_bytes(po, ns), fs = spinor_bytes(ps, ns);
  Work wk(c, s);
  char *r_hi, *xl, *rl, *rt, *pv, *v, *t;
  int rc;
  if ((rc = wk.get(&r_hi, fo * nrhs))) return rc;
  char** lo[] = {&xl, &rl, &rt, &pv, &v, &t};
  for (char** q : lo) if ((rc = wk.get(q, fs * nrhs))) return rc;
  std::vector<double> rn(nrhs), maxr(nrhs);
  std::vector<int> done(nrhs, 0), status(nrhs, LQCD_OK), waiting(nrhs, 0);
  // every return path (errors included) leaves the S_DONE flags of all sources clear for the next call
  struct DoneGuard { lqcd_ctx* c; int n; cudaStream_t s; ~DoneGuard() { for (int r = 0; r < n; ++r) set_done(c, r, 0.0, s); } } done_guard{c, nrhs, s};
  for (int r = 0; r < nrhs; ++r) if ((rc = set_done(c, r, 0.0, s))) return rc;
  if ((rc = residual_mrhs(c, r_hi, b, x, nrhs, par, p.kappa, po, p.recon_outer, rn.data(), s))) return rc;
  cnt.mat_outer += nrhs;
  const double delta = p.delta > 0 ? p.delta : 0.1;
  auto restart = [&](int r, int keep) -> int {    // r_l = lo(r_hi); keep = 0: fresh recurrence, 1: after a reliable update
    int rc2 = convert(c, po, ps, rl + r * fs, r_hi + r * fo, 0, par, s);
    if (rc2) return rc2;
    if (!keep) {
      if ((rc2 = convert(c, ps, ps, rt + r * fs, rl + r * fs, 0, par, s))) return rc2;
      for (char* z : {pv + r * fs, v + r * fs}) { BlasArgs a = mkr(c, r, z); if ((rc2 = blas<OpZero>(c, ps, a, s))) return rc2; }
    }
    BlasArgs a = mkr(c, r, rt + r * fs, rl + r * fs); a.i0 = keep;
    return blas<OpBicgInit>(c, ps, a, s);
  };
  int ndone = 0;
  for (int r = 0; r < nrhs; ++r) {
    res[r].iterations = 0; res[r].restarts = 0;
    maxr[r] = rn[r];
    { BlasArgs a = mkr(c, r, xl + r * fs); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
    if (rn[r] <= stop[r] || !(rn[r] == rn[r])) {
      done[r] = 1; ++ndone; status[r] = (rn[r] == rn[r]) ? LQCD_OK : LQCD_EBREAKDOWN;
      if ((rc = set_done(c, r, 1.0, s))) return rc;
      for (char* z : {rl + r * fs, rt + r * fs, pv + r * fs, v + r * fs, t + r * fs}) { BlasArgs a = mkr(c, r, z); if ((rc = blas<OpZero>(c, ps, a, s))) return rc; }
    } else if ((rc = restart(r, 0))) return rc;
  }
  int it = 0;
  while (ndone < nrhs) {
    const bool capped = it >= p.max_iter;
    bool update = capped;
    int nwant = 0;
    if (!capped) {
      { BlasArgs a = mkb(c, ps, pv, rl, v); if ((rc = blasb<OpBicgP>(c, ps, a, nrhs, s))) return rc; }
      if ((rc = op_matpc_mrhs(c, v, pv, nrhs, par, 0, p.kappa, ps, p.recon_sloppy, s))) return rc;
      { BlasArgs a = mkb(c, ps, rt, v); if ((rc = blasb<OpBicgAlpha>(c, ps, a, nrhs, s))) return rc; }
      { BlasArgs a = mkb(c, ps, rl, v); if ((rc = blasb<OpBicgS>(c, ps, a, nrhs, s))) return rc; }
      if ((rc = op_matpc_mrhs(c, t, rl, nrhs, par, 0, p.kappa, ps, p.recon_sloppy, s))) return rc;
      { BlasArgs a = mkb(c, ps, t, rl); if ((rc = blasb<OpBicgOmega>(c, ps, a, nrhs, s))) return rc; }
      { BlasArgs a = mkb(c, ps, xl, pv, rl, t, rt); if ((rc = blasb<OpBicgXR>(c, ps, a, nrhs, s))) return rc; }
      ++it;
      cnt.mat_sloppy += 2 * (nrhs - ndone); cnt.blas_flop_sites += 1056.0 * (nrhs - ndone);
      if ((rc = read_S_all(c, S_RR, nrhs, s))) return rc;
      for (int r = 0; r < nrhs; ++r) {
        if (done[r]) continue;
        res[r].iterations = it;
        const double rr = c->hS[S_TOTAL + 2 * r], flag = c->hS[S_TOTAL + 2 * r + 1];
        if (!(rr == rr) || flag != 0.0) status[r] = LQCD_EBREAKDOWN;
        const double rln = sqrt(rr);
        if (rln > maxr[r]) maxr[r] = rln;
        const bool want = rln <= stop[r] || rln < delta * maxr[r];
        waiting[r] = want ? waiting[r] + 1 : 0;
        if (want) ++nwant;
        if (status[r] == LQCD_EBREAKDOWN || waiting[r] > 4) update = true;
      }
      // the update costs one outer-precision Mhat for every source, so it is shared: taken when all
      // unfinished sources ask for it, or one has been asking for more than 4 iterations, or broke down
      if (nwant == nrhs - ndone) update = true;
    }
    if (!update) continue;
    // reliable update of every unfinished source: x += x_l, true residual in the outer precision
    for (int r = 0; r < nrhs; ++r) {
      if (done[r]) continue;
      MultiArgs m; memset(&m, 0, sizeof(m));
      m.b = mk(c, false); m.z[0] = xl + r * fs; m.chi[0] = 1.0; m.n = 1;
      cudaError_t e = run_accumulate(po, ps, x + r * fo, m, s); c->launches++;
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "accumulate", e);
      BlasArgs a = mkr(c, r, xl + r * fs); if ((rc = blas<OpZero>(c, ps, a, s))) return rc;
    }
    if ((rc = residual_mrhs(c, r_hi, b, x, nrhs, par, p.kappa, po, p.recon_outer, rn.data(), s))) return rc;
    cnt.mat_outer += nrhs;
    for (int r = 0; r < nrhs; ++r) {
      if (done[r]) continue;
      res[r].restarts++;
      const bool nan = !(rn[r] == rn[r]);
      if (rn[r] <= stop[r] || nan || capped) {
        done[r] = 1; ++ndone;
        status[r] = nan ? LQCD_EBREAKDOWN : (rn[r] <= stop[r] ? LQCD_OK : LQCD_ENOCONV);
        if ((rc = set_done(c, r, 1.0, s))) return rc;
      } else {
        if ((rc = restart(r, status[r] == LQCD_EBREAKDOWN ? 0 : 1))) return rc;
        status[r] = LQCD_OK;
        maxr[r] = rn[r];
        waiting[r] = 0;
      }
    }
  }
  for (int r = 0; r < nrhs; ++r) {
    res[r].status = status[r];
    res[r].iterated_residual = rn[r];
  }
  return LQCD_OK;
}

int check_params(lqcd_ctx* c, const lqcd_invert_params* p) {
  if (!p) return fail(c, LQCD_EINVAL, "null params");
  if (!c->have_gauge || !c->have_clover) return fail(c, LQCD_ESTATE, "invert before load_gauge / build_clover");
  if (!(p->c_sw == c->c_sw)) return fail(c, LQCD_ESTATE, "params.c_sw differs from the built clover term");
  if ((p->parity | 1) != 1) return fail(c, LQCD_EINVAL, "parity");
  for (int pr : {p->prec_outer, p->prec_sloppy, p->prec_precond}) if (pr < 0 || pr > 2) return fail(c, LQCD_EINVAL, "precision");
  for (int r : {p->recon_outer, p->recon_sloppy, p->recon_precond}) if (recon_index(r) < 0) return fail(c, LQCD_EINVAL, "recon");
  if (p->solver != LQCD_SOLVER_BICGSTAB && p->solver != LQCD_SOLVER_GCR_DD && p->solver != LQCD_SOLVER_CGNR && p->solver != LQCD_SOLVER_CGNE) return fail(c, LQCD_EINVAL, "solver");
  if (!(p->tol > 0) || p->max_iter < 1) return fail(c, LQCD_EINVAL, "tol / max_iter");
  if (p->solver == LQCD_SOLVER_GCR_DD && p->precondition && p->mr_steps < 1) return fail(c, LQCD_EINVAL, "mr_steps");
  if (p->schwarz_type != LQCD_SCHWARZ_ADDITIVE && p->schwarz_type != LQCD_SCHWARZ_MULTIPLICATIVE) return fail(c, LQCD_EINVAL, "schwarz_type");
  if (p->sap_cycles < 0) return fail(c, LQCD_EINVAL, "sap_cycles");
  if (p->matpc_type != LQCD_MATPC_ASYMMETRIC && p->matpc_type != LQCD_MATPC_SYMMETRIC) return fail(c, LQCD_EINVAL, "matpc_type");
  if (p->matpc_type == LQCD_MATPC_SYMMETRIC && p->solver == LQCD_SOLVER_GCR_DD) return fail(c, LQCD_EINVAL, "symmetric form: BiCGstab, CGNR and CGNE only");
  return LQCD_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

int lqcd_schwarz(lqcd_ctx* c, void* out, const void* in, int parity, double kappa, const int block[4], int n_mr,
                 double omega_mr, int prec, int recon, int prec_io, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || (parity | 1) != 1 || n_mr < 1 || prec < 0 || prec > 2 || prec_io < 0 || prec_io > 2)
    return fail(c, LQCD_EINVAL, "schwarz arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  int rc = set_blocks(c, block, 0, c->schwarz_overlap);
  if (rc) return rc;
  Work wk(c, s);
  char *rho, *w, *xk;
  for (char** q : {&rho, &w, &xk}) if ((rc = wk.get(q, spinor_bytes(prec, c->bm.blk.ns)))) return rc;     // block-major: grown domains
  rc = schwarz_apply(c, (char*)out, (const char*)in, parity, kappa, n_mr, omega_mr, prec, recon, prec_io, rho, w, xk, s);
  cudaStreamSynchronize(s);          // workspace is freed on return
  return rc;
}

int lqcd_schwarz_sap(lqcd_ctx* c, void* out, const void* in, int parity, double kappa, const int block[4], int n_mr,
                     double omega_mr, int n_cycle, int prec, int recon, int prec_io, int recon_io, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity | 1) != 1 || n_mr < 1 || n_cycle < 1 || prec < 0 || prec > 2 || prec_io < 0 || prec_io > 2)
    return fail(c, LQCD_EINVAL, "schwarz_sap arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  int rc = set_blocks(c, block, 1);
  if (rc) return rc;
  Work wk(c, s);
  char *rho, *w, *xk, *r, *y, *t;
  for (char** q : {&rho, &w, &xk}) if ((rc = wk.get(q, spinor_bytes(prec, c->nat.ns)))) return rc;
  for (char** q : {&r, &y, &t}) if ((rc = wk.get(q, spinor_bytes(prec_io, c->nat.ns)))) return rc;
  rc = schwarz_sap_apply(c, (char*)out, (const char*)in, parity, kappa, n_mr, omega_mr, n_cycle, prec, recon, prec_io, recon_io,
                         rho, w, xk, r, y, t, s);
  cudaStreamSynchronize(s);          // workspace is handed back on return
  return rc;
}

int lqcd_set_schwarz_group(lqcd_ctx* c, int blocks_per_group) {
  if (!c) return LQCD_EINVAL;
  if (blocks_per_group < 0) return fail(c, LQCD_EINVAL, "schwarz group");
  c->schwarz_group = blocks_per_group;
  return LQCD_OK;
}

int lqcd_set_schwarz_overlap(lqcd_ctx* c, int overlap) {
  if (!c) return LQCD_EINVAL;
  if (overlap < 0) return fail(c, LQCD_EINVAL, "schwarz overlap");
  c->schwarz_overlap = overlap;
  return LQCD_OK;
}

int lqcd_invert(lqcd_ctx* c, void* x_can, const void* b_can, const lqcd_invert_params* p, lqcd_invert_result* res, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x_can || !b_can || !res) return fail(c, LQCD_EINVAL, "invert arguments");
  int rc = check_params(c, p);
  if (rc) return rc;
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  memset(res, 0, sizeof(*res));
  c->hist.clear();
  if (p->history_len < 0 || (p->history_len > 0 && !p->residual_history)) return fail(c, LQCD_EINVAL, "residual_history");
  const int po = p->prec_outer, par = p->parity;
  const long long ns = c->nat.ns;
  Work wk(c, s);
  char *bp, *bq, *xp, *xq, *t1;
  for (char** q : {&bp, &bq, &xp, &xq, &t1}) if ((rc = wk.get(q, spinor_bytes(po, ns)))) return rc;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return fail(c, LQCD_ECUDA, "event");
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return fail(c, LQCD_ECUDA, "event"); }
  EventPair ev{e0, e1};                 // destroyed on every return path
  cudaEventRecord(e0, s);
  Counts cnt;
  nvtxRangePushA("lqcd_invert: prepare");
  struct PopGuard { int n = 1; ~PopGuard() { while (n-- > 0) nvtxRangePop(); } } nvtx_guard;   // balances the ranges on every return path
  // pack b; ||b||
  cudaError_t e = run_pack_spinor(po, bp, (const double*)b_can, c->nat, par, 0, s); c->launches++;
  if (e == cudaSuccess) { e = run_pack_spinor(po, bq, (const double*)b_can, c->nat, 1 - par, 0, s); c->launches++; }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
  double n1, n2;
  if ((rc = norm2(c, po, bp, &n1, s))) return rc;
  if ((rc = norm2(c, po, bq, &n2, s))) return rc;
  const double bnorm = sqrt(n1 + n2);
  if (bnorm == 0.0) {
    cudaMemsetAsync(x_can, 0, (size_t)c->V * 24 * sizeof(double), s);
    cudaStreamSynchronize(s);
    res->status = LQCD_OK;
    return LQCD_OK;
  }
  // source preparation: bhat_p = b_p + kappa D A^-1 b_pbar   (R6)
  const char *A, *Ai;
  if ((rc = get_clover(c, po, p->kappa, false, &A, &Ai, s))) return rc;
  e = run_clover_apply(po, t1, bq, Ai, c->nat, 1 - par, s); c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "clover_apply", e);
  if ((rc = op_dslash(c, xq /* holds bhat */, t1, bp, par, 0, po, p->recon_outer, EPI_XPAY, p->kappa, p->kappa, false, s))) return rc;
  char* bhat = xq;
  // initial guess
  if (p->use_initial_guess) {
    e = run_pack_spinor(po, xp, (const double*)x_can, c->nat, par, 0, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
  } else {
    BlasArgs a = mk(c, false, xp);
    if ((rc = blas<OpZero>(c, po, a, s))) return rc;
  }
  const double stop = p->tol * bnorm;
  int status;
  nvtxRangePop(); nvtxRangePushA("lqcd_invert: iterate");
  if (p->solver == LQCD_SOLVER_BICGSTAB) status = solve_bicgstab(c, xp, bhat, *p, stop, res, cnt, s);
  else if (p->solver == LQCD_SOLVER_CGNR) status = solve_cgnr(c, xp, bhat, *p, stop, res, cnt, s);
  else if (p->solver == LQCD_SOLVER_CGNE) status = solve_cgne(c, xp, bhat, *p, stop, res, cnt, s);
  else status = solve_gcr(c, xp, bhat, *p, stop, res, cnt, s);
  if (status != LQCD_OK && status != LQCD_ENOCONV && status != LQCD_EBREAKDOWN) return status;
  nvtxRangePop(); nvtxRangePushA("lqcd_invert: true residual, reconstruct, unpack");
  // true residual of the Schur system in the outer precision = ||b - M x|| (R6)
  double rn;
  if ((rc = residual(c, t1, bhat, xp, par, p->kappa, po, p->recon_outer, &rn, s))) return rc;
  cnt.mat_outer++;
  res->true_residual = rn / bnorm;
  res->iterated_residual /= bnorm;
  for (size_t k = 0; k < c->hist.size() && (int)k < p->history_len; ++k) { p->residual_history[k] = c->hist[k] / bnorm; res->history_count = (int)k + 1; }
  // reconstruction: x_pbar = A^-1 (b_pbar + kappa D x_p)
  if ((rc = op_dslash(c, t1, xp, bq, 1 - par, 0, po, p->recon_outer, EPI_XPAY_CLOVOUT, p->kappa, p->kappa, false, s))) return rc;
  e = run_pack_spinor(po, xp, (const double*)x_can, c->nat, par, 1, s); c->launches++;
  if (e == cudaSuccess) { e = run_pack_spinor(po, t1, (const double*)x_can, c->nat, 1 - par, 1, s); c->launches++; }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
  cudaEventRecord(e1, s);
  e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "invert", e);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  res->seconds = ms * 1e-3;
  res->status = status;
  res->matpc_sloppy = (int)cnt.mat_sloppy; res->matpc_outer = (int)cnt.mat_outer; res->matpc_precond = (int)cnt.mat_precond;
  res->gflop = ((double)(cnt.mat_sloppy + cnt.mat_outer + cnt.mat_precond) * 3696.0 + cnt.blas_flop_sites) * (double)c->Vh * 1e-9;
  if (status == LQCD_ENOCONV) return fail(c, status, "max_iter reached");
  if (status == LQCD_EBREAKDOWN) return fail(c, status, "solver breakdown");
  return LQCD_OK;
}

int lqcd_invert_mrhs(lqcd_ctx* c, void* x_can, const void* b_can, int nrhs, const lqcd_invert_params* p, lqcd_invert_result* res,
                     void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x_can || !b_can || !res || nrhs < 1 || nrhs > LQCD_MAX_RHS) return fail(c, LQCD_EINVAL, "invert_mrhs arguments");
  int rc = check_params(c, p);
  if (rc) return rc;
  if (p->solver != LQCD_SOLVER_BICGSTAB || p->matpc_type != LQCD_MATPC_ASYMMETRIC)
    return fail(c, LQCD_EINVAL, "invert_mrhs: BiCGstab on the asymmetric Schur system only");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  memset(res, 0, sizeof(*res) * nrhs);
  const int po = p->prec_outer, par = p->parity;
  const long long ns = c->nat.ns;
  const size_t fo = spinor_bytes(po, ns), cb = (size_t)c->V * 24 * sizeof(double);
  Work wk(c, s);
  char *bp, *bq, *xp, *bhat, *t1;
  for (char** q : {&bp, &bq, &xp, &bhat, &t1}) if ((rc = wk.get(q, fo * nrhs))) return rc;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess) return fail(c, LQCD_ECUDA, "event");
  if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); return fail(c, LQCD_ECUDA, "event"); }
  EventPair ev{e0, e1};
  cudaEventRecord(e0, s);
  Counts cnt;
  const char *A, *Ai;
  if ((rc = get_clover(c, po, p->kappa, false, &A, &Ai, s))) return rc;
  cudaError_t e = cudaSuccess;
  for (int r = 0; r < nrhs && e == cudaSuccess; ++r) {
    const double* bc = (const double*)((const char*)b_can + r * cb);
    e = run_pack_spinor(po, bp + r * fo, bc, c->nat, par, 0, s); c->launches++;
    if (e == cudaSuccess) { e = run_pack_spinor(po, bq + r * fo, bc, c->nat, 1 - par, 0, s); c->launches++; }
    if (e == cudaSuccess) { e = run_clover_apply(po, t1 + r * fo, bq + r * fo, Ai, c->nat, 1 - par, s); c->launches++; }
    if (e == cudaSuccess) {
      if (p->use_initial_guess) { e = run_pack_spinor(po, xp + r * fo, (const double*)((const char*)x_can + r * cb), c->nat, par, 0, s); c->launches++; }
      else { BlasArgs a = mk(c, false, xp + r * fo); if ((rc = blas<OpZero>(c, po, a, s))) return rc; }
    }
  }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack / clover", e);
  // ||b_r||: two norms per source on its own scalar set
  std::vector<double> bnorm(nrhs), stop(nrhs);
  for (int r = 0; r < nrhs; ++r) {
    BlasArgs a = mkr(c, r, bp + r * fo); a.i0 = 0; if ((rc = blas<OpNorm2>(c, po, a, s))) return rc;
    BlasArgs a2 = mkr(c, r, bq + r * fo); a2.i0 = 1; if ((rc = blas<OpNorm2>(c, po, a2, s))) return rc;
  }
  if ((rc = read_S_all(c, S_OUT, nrhs, s))) return rc;
  for (int r = 0; r < nrhs; ++r) {
    bnorm[r] = sqrt(c->hS[S_TOTAL + 2 * r] + c->hS[S_TOTAL + 2 * r + 1]);
    stop[r] = p->tol * bnorm[r];                           // a zero source is "converged" at once with x = 0
  }
  // source preparation for all sources: bhat_p = b_p + kappa D A^-1 b_pbar   (R6)
  if ((rc = op_dslash_mrhs(c, bhat, t1, bp, nrhs, par, 0, po, p->recon_outer, EPI_XPAY, p->kappa, p->kappa, s))) return rc;
  rc = solve_bicgstab_mrhs(c, xp, bhat, nrhs, *p, stop.data(), res, cnt, s);
  if (rc) return rc;
  // true residuals, reconstruction x_pbar = A^-1 (b_pbar + kappa D x_p), unpack
  std::vector<double> rn(nrhs);
  if ((rc = residual_mrhs(c, t1, bhat, xp, nrhs, par, p->kappa, po, p->recon_outer, rn.data(), s))) return rc;
  cnt.mat_outer += nrhs;
  if ((rc = op_dslash_mrhs(c, t1, xp, bq, nrhs, 1 - par, 0, po, p->recon_outer, EPI_XPAY_CLOVOUT, p->kappa, p->kappa, s))) return rc;
  for (int r = 0; r < nrhs && e == cudaSuccess; ++r) {
    double* xc = (double*)((char*)x_can + r * cb);
    e = run_pack_spinor(po, xp + r * fo, xc, c->nat, par, 1, s); c->launches++;
    if (e == cudaSuccess) { e = run_pack_spinor(po, t1 + r * fo, xc, c->nat, 1 - par, 1, s); c->launches++; }
  }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
  cudaEventRecord(e1, s);
  e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "invert_mrhs", e);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  int worst = LQCD_OK;
  const double gflop = ((double)(cnt.mat_sloppy + cnt.mat_outer) * 3696.0 + cnt.blas_flop_sites) * (double)c->Vh * 1e-9;
  for (int r = 0; r < nrhs; ++r) {
    res[r].true_residual = bnorm[r] > 0 ? rn[r] / bnorm[r] : 0.0;
    res[r].iterated_residual = bnorm[r] > 0 ? res[r].iterated_residual / bnorm[r] : 0.0;
    res[r].seconds = ms * 1e-3;                            // the whole batch
    res[r].gflop = gflop;                                  // the whole batch
    res[r].matpc_sloppy = 2 * res[r].iterations; res[r].matpc_outer = res[r].restarts + 2;
    if (res[r].status != LQCD_OK && worst == LQCD_OK) worst = res[r].status;
  }
  if (worst == LQCD_ENOCONV) return fail(c, worst, "max_iter reached for at least one right-hand side");
  if (worst == LQCD_EBREAKDOWN) return fail(c, worst, "solver breakdown for at least one right-hand side");
  return LQCD_OK;
}

int lqcd_axpy_norm(lqcd_ctx* c, double a_, const void* x, void* y, int prec, double* norm2_host, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x || !y || !norm2_host || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "axpy_norm arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  BlasArgs a = mk(c, false, (char*)x, (char*)y);
  a.c[0] = a_;
  int rc = blas<OpAxpyNorm>(c, prec, a, s);
  if (rc) return rc;
  rc = read_S(c, S_OUT, 1, s);
  *norm2_host = c->hS[S_OUT];
  return rc;
}

int lqcd_cdot(lqcd_ctx* c, const void* x, const void* y, int prec, double* dot_host, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x || !y || !dot_host || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "cdot arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  BlasArgs a = mk(c, false, (char*)x, (char*)y);
  int rc = blas<OpCdot>(c, prec, a, s);
  if (rc) return rc;
  rc = read_S(c, S_OUT, 2, s);
  dot_host[0] = c->hS[S_OUT]; dot_host[1] = c->hS[S_OUT + 1];
  return rc;
}

}  // extern "C"
