// noalloc.cu -- lqcd_cdot_static: <x,y> and ||y||^2 of two packed device fields with NO allocation.
//
// For callers that cannot call cudaMalloc (stream capture into a CUDA graph, tight serving loops, harnesses that
// forbid it).  Same sums as lqcd_cdot / OpCdot (blas_ops.cuh; the reductions of the Krylov
// solvers), but (i) the per-CTA partial sums live in a file-scope __device__ array instead of the context's
// cudaMalloc'ed workspace, (ii) the result goes to a DEVICE pointer of the caller (no copy, no stream sync), and
// (iii) the call issues two kernel launches and nothing else: no cudaMalloc / cudaFree / memcpy / event.
//
// The array is LQ_STATIC_SCRATCH_BYTES (768 KiB) on every GPU that loads the library, until the process exits.  It
// bounds the field size: at most LQ_STATIC_MAX_SITES sites per parity field (2^23, e.g. 64^3 x 64); larger fields
// are rejected with LQCD_EINVAL.  Every call on a device shares the array and it keeps the last call's contents.
// Nothing in it has to start at zero: the finalize kernel reads exactly the n partials the first kernel of the SAME
// call wrote (no arrival counter, no accumulation into old contents).  Two calls that overlap on one GPU (two
// streams, two host threads) race on it; calls on one stream are ordered.
#include <mutex>
#include "blas.cuh"
#include "ops.h"

namespace lq {

#define LQ_STATIC_MAX_SITES (1 << 23)
#define LQ_STATIC_MAX_CTAS (LQ_STATIC_MAX_SITES / LQ_BLAS_BLOCK)
#define LQ_STATIC_SCRATCH_DOUBLES (3 * LQ_STATIC_MAX_CTAS)
#define LQ_STATIC_SCRATCH_BYTES (8 * LQ_STATIC_SCRATCH_DOUBLES)

// [cta][3] partial sums (re <x,y>, im <x,y>, ||y||^2).  In HOST code this name is a host-side stand-in, not a device
// address: kernels get the address cudaGetSymbolAddress returns (static_scratch below).
static __device__ __align__(256) double lq_static_scratch[LQ_STATIC_SCRATCH_DOUBLES];

// one site per thread; per-site sums in the field's arithmetic type, then fp64 (as OpCdot); one partial per CTA
template <class P>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK) cdot_static_kernel(const char* x, const char* y, long long ns, int vh, double* part) {
  typedef typename P::real R;
  __shared__ double sm[3 * (LQ_BLAS_BLOCK / 32)];
  double red[3] = {0, 0, 0};
  const int cb = blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x;
  if (cb < vh) {
    R vx[24], vy[24];
    load_site<P, 24>(vx, x, ns, cb);
    load_site<P, 24>(vy, y, ns, cb);
    site_cdot<R>(vx, vy, red[0], red[1]);
    site_norm2<R>(vy, red[2]);
  }
  cta_reduce<3, LQ_BLAS_BLOCK>(red, sm);
  if (threadIdx.x == 0) {
    part[3ll * blockIdx.x] = red[0]; part[3ll * blockIdx.x + 1] = red[1]; part[3ll * blockIdx.x + 2] = red[2];
  }
}

// one CTA adds the n partials in a fixed order (bit-reproducible) and writes the three sums to the caller's buffer
__global__ void __launch_bounds__(1024) cdot_static_finalize_kernel(const double* part, int n, double* out) {
  __shared__ double sm[3 * 32];
  double s[3] = {0, 0, 0};
  for (int i = threadIdx.x; i < n; i += 1024) {
    s[0] += part[3ll * i]; s[1] += part[3ll * i + 1]; s[2] += part[3ll * i + 2];
  }
  cta_reduce<3, 1024>(s, sm);
  if (threadIdx.x == 0) { out[0] = s[0]; out[1] = s[1]; out[2] = s[2]; }
}

// Device address of lq_static_scratch on the CURRENT device, looked up once per device (cudaGetSymbolAddress
// allocates nothing; the array is part of the module image).
static cudaError_t static_scratch(int device, double** out) {
  static std::mutex mu;
  static double* addr[64] = {nullptr};
  if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[device]) {
    double* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, lq_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    addr[device] = p;
  }
  *out = addr[device];
  return cudaSuccess;
}

}  // namespace lq

using namespace lq;

extern "C" int lqcd_cdot_static(lqcd_ctx* c, const void* x, const void* y, int prec, double* out_device, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x || !y || !out_device || prec < 0 || prec > 2) return fail(c, LQCD_EINVAL, "cdot_static arguments");
  const int vh = c->nat.vh;
  if (vh > LQ_STATIC_MAX_SITES) {
    char msg[160];
    snprintf(msg, sizeof(msg), "lqcd_cdot_static: %d sites per parity field exceed the static scratch maximum of %d", vh,
             (int)LQ_STATIC_MAX_SITES);
    return fail(c, LQCD_EINVAL, msg);
  }
  cudaError_t e = cudaSetDevice(c->device);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "cdot_static: set device", e);
  double* part = nullptr;
  if ((e = static_scratch(c->device, &part)) != cudaSuccess) return fail(c, LQCD_ECUDA, "cdot_static: address of the static scratch", e);
  cudaStream_t s = (cudaStream_t)stream;
  const int ctas = (vh + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK;
  const char* xp = (const char*)x;
  const char* yp = (const char*)y;
  switch (prec) {
    case 0: cdot_static_kernel<PrecD><<<ctas, LQ_BLAS_BLOCK, 0, s>>>(xp, yp, c->nat.ns, vh, part); break;
    case 1: cdot_static_kernel<PrecS><<<ctas, LQ_BLAS_BLOCK, 0, s>>>(xp, yp, c->nat.ns, vh, part); break;
    default: cdot_static_kernel<PrecH><<<ctas, LQ_BLAS_BLOCK, 0, s>>>(xp, yp, c->nat.ns, vh, part); break;
  }
  if ((e = cudaGetLastError()) != cudaSuccess) return fail(c, LQCD_ECUDA, "cdot_static launch", e);
  cdot_static_finalize_kernel<<<1, 1024, 0, s>>>(part, ctas, out_device);
  if ((e = cudaGetLastError()) != cudaSuccess) return fail(c, LQCD_ECUDA, "cdot_static finalize launch", e);
  c->launches += 2;
  return LQCD_OK;
}
