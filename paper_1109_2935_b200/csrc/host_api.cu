// host_api.cu -- end-to-end entry points taking HOST buffers (include/lqcd.h): the
// host->device copy of the inputs, the computation and the device->host copy of the result all
// happen inside the call, on the caller's stream.
#include <cstring>
#include "ops.h"

using namespace lq;

namespace {
struct DevBuf {
  void* p = nullptr;
  ~DevBuf() { if (p) cudaFree(p); }
};
}  // namespace

extern "C" {

int lqcd_apply_host(lqcd_ctx* c, void* out_host, const void* in_host, int op, int parity, int dagger, double kappa,
                    int prec, int recon, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out_host || !in_host || (op != 0 && op != 1) || (parity | 1) != 1 || prec < 0 || prec > 2)
    return fail(c, LQCD_EINVAL, "apply_host arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t cbytes = (size_t)c->V * 24 * sizeof(double), pbytes = spinor_bytes(prec, c->nat.ns);
  DevBuf can, pin[2], pout[2];
  int rc;
  if ((rc = dev_alloc(c, &can.p, cbytes))) return rc;
  for (int i = 0; i < 2; ++i) { if ((rc = dev_alloc(c, &pin[i].p, pbytes))) return rc; if ((rc = dev_alloc(c, &pout[i].p, pbytes))) return rc; }
  cudaError_t e = cudaMemcpyAsync(can.p, in_host, cbytes, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "H2D", e);
  if (op == 0) {
    for (int p = 0; p < 2; ++p) {
      e = run_pack_spinor(prec, (char*)pin[p].p, (const double*)can.p, c->nat, p, 0, s); c->launches++;
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
    }
    for (int p = 0; p < 2; ++p)
      if ((rc = op_dslash(c, (char*)pout[p].p, (const char*)pin[1 - p].p, nullptr, p, dagger ? 1 : 0, prec, recon, EPI_NONE, 0, 0, false, s))) return rc;
    for (int p = 0; p < 2; ++p) {
      e = run_pack_spinor(prec, (char*)pout[p].p, (const double*)can.p, c->nat, p, 1, s); c->launches++;
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
    }
  } else {
    e = run_pack_spinor(prec, (char*)pin[0].p, (const double*)can.p, c->nat, parity, 0, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
    if ((rc = op_matpc(c, (char*)pout[0].p, (const char*)pin[0].p, parity, dagger ? 1 : 0, kappa, prec, recon, false, false, s))) return rc;
    e = cudaMemsetAsync(can.p, 0, cbytes, s);
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "memset", e);
    e = run_pack_spinor(prec, (char*)pout[0].p, (const double*)can.p, c->nat, parity, 1, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
  }
  e = cudaMemcpyAsync(out_host, can.p, cbytes, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "D2H", e);
}

int lqcd_invert_host(lqcd_ctx* c, void* x_host, const void* b_host, const lqcd_invert_params* p, lqcd_invert_result* res, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x_host || !b_host || !p || !res) return fail(c, LQCD_EINVAL, "invert_host arguments");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  const size_t cbytes = (size_t)c->V * 24 * sizeof(double);
  DevBuf xb, bb;
  int rc;
  if ((rc = dev_alloc(c, &xb.p, cbytes))) return rc;
  if ((rc = dev_alloc(c, &bb.p, cbytes))) return rc;
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
