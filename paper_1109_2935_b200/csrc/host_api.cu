// host_api.cu -- end-to-end entry points taking HOST buffers (include/lqcd.h): the
// host->device copy of the inputs, the computation and the device->host copy of the result all
// happen inside the call.
//
// lqcd_apply_host is a slab pipeline over the slowest lattice index t: the canonical input is cut
// into n <= 16 slabs of T/n time slices; slab k+1 is copied host->device on one copy stream while
// slab k is packed and the operator is applied to slab k-1 on the caller's stream (a slab of outputs
// needs its two neighbour slabs of inputs, periodic in t), and finished slabs are unpacked and
// copied device->host on a second copy stream.  PCIe is full duplex, so the call costs about one
// direction's transfer time instead of two plus the kernels.  The kernels are the ordinary ones
// launched on the slab's site range (t is the slowest checkerboard index, so a slab is one
// contiguous range of every packed field); results are bit-identical to whole-lattice launches.
#include <cstring>
#include "ops.h"

using namespace lq;

namespace {
// grow-only staging buffer `slot` of the context (freed by lqcd_destroy)
int hbuf(lqcd_ctx* c, int slot, size_t bytes, void** out) {
  if (c->hws_bytes[slot] < bytes) {
    if (c->hws[slot]) { cudaFree(c->hws[slot]); c->hws[slot] = nullptr; c->hws_bytes[slot] = 0; }
    int rc = dev_alloc(c, &c->hws[slot], bytes);
    if (rc) return rc;
    c->hws_bytes[slot] = bytes;
  }
  *out = c->hws[slot];
  return LQCD_OK;
}

int hpipe(lqcd_ctx* c) {
  if (c->have_hpipe) return LQCD_OK;
  bool ok = cudaStreamCreateWithFlags(&c->hs_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->hs_out, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->hev_sync, cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; ok && i < LQ_HOST_SLABS; ++i)
    ok = cudaEventCreateWithFlags(&c->hev_in[i], cudaEventDisableTiming) == cudaSuccess &&
         cudaEventCreateWithFlags(&c->hev_out[i], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) return fail(c, LQCD_ECUDA, "apply_host: stream / event creation", cudaGetLastError());
  c->have_hpipe = true;
  return LQCD_OK;
}
}  // namespace

// creal = bytes of one real of the canonical host arrays: 8 (complex128) or 4 (complex64)
static int apply_host(lqcd_ctx* c, void* out_host, const void* in_host, int op, int parity, int dagger, double kappa,
                      int prec, int recon, void* stream, int creal) {
  if (!c) return LQCD_EINVAL;
  if (!out_host || !in_host || (op != 0 && op != 1) || (parity | 1) != 1 || prec < 0 || prec > 2 || recon_index(recon) < 0)
    return fail(c, LQCD_EINVAL, "apply_host arguments");
  if (!c->have_gauge || (op == 1 && !c->have_clover)) return fail(c, LQCD_ESTATE, "apply_host before load_gauge / build_clover");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t cbytes = (size_t)c->V * 24 * creal, pbytes = spinor_bytes(prec, c->nat.ns);
  const int c32 = creal == 4;
  int rc;
  if ((rc = hpipe(c))) return rc;
  void *can_in, *can_out, *pk[4];
  if ((rc = hbuf(c, 0, cbytes, &can_in)) || (rc = hbuf(c, 1, cbytes, &can_out))) return rc;
  for (int i = 0; i < 4; ++i) if ((rc = hbuf(c, 2 + i, pbytes, &pk[i]))) return rc;
  char *pin[2] = {(char*)pk[0], (char*)pk[1]}, *pout[2] = {(char*)pk[2], (char*)pk[3]};
  // slabs: n = largest divisor of T that is <= LQ_HOST_SLABS; a slab needs distinct neighbours (n >= 3)
  const int T = c->dims[3];
  int n = T < LQ_HOST_SLABS ? T : LQ_HOST_SLABS;
  while (T % n) --n;
  if (n < 3) n = 1;
  const long long sl_sites = c->Vh / n;                 // sites of one parity per slab
  const size_t sl_bytes = cbytes / n;                   // canonical bytes per slab
  const int dg = dagger ? 1 : 0;
  cudaError_t e = cudaSuccess;
#define LQ_CK(call, what) do { e = (call); if (e != cudaSuccess) return fail(c, LQCD_ECUDA, what, e); } while (0)
  // the copy streams start after everything already queued on the caller's stream
  LQ_CK(cudaEventRecord(c->hev_sync, s), "event");
  LQ_CK(cudaStreamWaitEvent(c->hs_in, c->hev_sync, 0), "wait");
  LQ_CK(cudaStreamWaitEvent(c->hs_out, c->hev_sync, 0), "wait");
  for (int k = 0; k < n; ++k) {
    LQ_CK(cudaMemcpyAsync((char*)can_in + k * sl_bytes, (const char*)in_host + k * sl_bytes, sl_bytes, cudaMemcpyHostToDevice, c->hs_in), "H2D");
    LQ_CK(cudaEventRecord(c->hev_in[k], c->hs_in), "event");
  }
  if (op == 1) LQ_CK(cudaMemsetAsync(can_out, 0, cbytes, s), "memset");     // the other parity of the result is zero
  bool packed[LQ_HOST_SLABS] = {false}, st1[LQ_HOST_SLABS] = {false}, st2[LQ_HOST_SLABS] = {false};
  auto ready = [&](const bool* f, int k) { return f[(k + n - 1) % n] && f[k] && f[(k + 1) % n]; };
  auto finish = [&](int k) -> int {                     // unpack slab k and send it home
    const long long i0 = k * sl_sites, i1 = i0 + sl_sites;
    for (int p = 0; p < 2; ++p) {
      if (op == 1 && p != parity) continue;
      e = run_pack_spinor(prec, op == 1 ? pout[0] : pout[p], (const double*)can_out, c->nat, p, 1, s, i0, i1, c32); c->launches++;
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
    }
    if ((e = cudaEventRecord(c->hev_out[k], s)) != cudaSuccess || (e = cudaStreamWaitEvent(c->hs_out, c->hev_out[k], 0)) != cudaSuccess ||
        (e = cudaMemcpyAsync((char*)out_host + k * sl_bytes, (char*)can_out + k * sl_bytes, sl_bytes, cudaMemcpyDeviceToHost, c->hs_out)) != cudaSuccess)
      return fail(c, LQCD_ECUDA, "D2H", e);
    return LQCD_OK;
  };
  for (int j = 0; j < n; ++j) {
    LQ_CK(cudaStreamWaitEvent(s, c->hev_in[j], 0), "wait");
    const long long i0 = j * sl_sites, i1 = i0 + sl_sites;
    for (int p = 0; p < 2; ++p) {
      if (op == 1 && p != parity) continue;
      e = run_pack_spinor(prec, op == 1 ? pin[0] : pin[p], (const double*)can_in, c->nat, p, 0, s, i0, i1, c32); c->launches++;
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
    }
    packed[j] = true;
    for (int k = 0; k < n; ++k) {
      if (st1[k] || !ready(packed, k)) continue;
      const int c0 = (int)(k * sl_sites), c1 = (int)(c0 + sl_sites);
      if (op == 0) {                                    // out_p = D in_pbar on both parities
        for (int p = 0; p < 2; ++p)
          if ((rc = op_dslash(c, pout[p], pin[1 - p], nullptr, p, dg, prec, recon, EPI_NONE, 0, 0, false, s, c0, c1))) return rc;
        if ((rc = finish(k))) return rc;
      } else {                                          // tmp_pbar = A^-1 D in_p
        if ((rc = op_dslash(c, pout[1], pin[0], nullptr, 1 - parity, dg, prec, recon, EPI_CLOVOUT, 0.0, kappa, false, s, c0, c1))) return rc;
      }
      st1[k] = true;
    }
    if (op == 1) {
      for (int k = 0; k < n; ++k) {
        if (st2[k] || !ready(st1, k)) continue;         // out_p = A in_p - kappa^2 D tmp_pbar
        const int c0 = (int)(k * sl_sites), c1 = (int)(c0 + sl_sites);
        if ((rc = op_dslash(c, pout[0], pout[1], pin[0], parity, dg, prec, recon, EPI_CLOVX_XPAY, -kappa * kappa, kappa, false, s, c0, c1))) return rc;
        if ((rc = finish(k))) return rc;
        st2[k] = true;
      }
    }
  }
  LQ_CK(cudaEventRecord(c->hev_sync, c->hs_out), "event");
  LQ_CK(cudaStreamWaitEvent(s, c->hev_sync, 0), "wait");
  LQ_CK(cudaStreamSynchronize(s), "apply_host");
#undef LQ_CK
  return LQCD_OK;
}

extern "C" {

int lqcd_apply_host(lqcd_ctx* c, void* out_host, const void* in_host, int op, int parity, int dagger, double kappa,
                    int prec, int recon, void* stream) {
  return apply_host(c, out_host, in_host, op, parity, dagger, kappa, prec, recon, stream, 8);
}

int lqcd_apply_host_c64(lqcd_ctx* c, void* out_host, const void* in_host, int op, int parity, int dagger, double kappa,
                        int prec, int recon, void* stream) {
  if (c && prec == 0) return fail(c, LQCD_EINVAL, "apply_host_c64: single-precision host arrays serve fp32 / half compute only");
  return apply_host(c, out_host, in_host, op, parity, dagger, kappa, prec, recon, stream, 4);
}

int lqcd_invert_host(lqcd_ctx* c, void* x_host, const void* b_host, const lqcd_invert_params* p, lqcd_invert_result* res, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x_host || !b_host || !p || !res) return fail(c, LQCD_EINVAL, "invert_host arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t cbytes = (size_t)c->V * 24 * sizeof(double);
  struct Ws { lqcd_ctx* c; cudaStream_t s; size_t n; void* p = nullptr; ~Ws() { ws_put(c, p, n, s); } } xb{c, s, cbytes}, bb{c, s, cbytes};
  int rc;
  if ((rc = ws_get(c, &xb.p, cbytes, s))) return rc;
  if ((rc = ws_get(c, &bb.p, cbytes, s))) return rc;
  cudaError_t e = cudaMemcpyAsync(bb.p, b_host, cbytes, cudaMemcpyHostToDevice, s);
  if (e == cudaSuccess && p->use_initial_guess) e = cudaMemcpyAsync(xb.p, x_host, cbytes, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "H2D", e);
  rc = lqcd_invert(c, xb.p, bb.p, p, res, stream);
  if (rc != LQCD_OK && rc != LQCD_ENOCONV && rc != LQCD_EBREAKDOWN) return rc;
  e = cudaMemcpyAsync(x_host, xb.p, cbytes, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "D2H", e);
  return rc;
}

}  // extern "C"
