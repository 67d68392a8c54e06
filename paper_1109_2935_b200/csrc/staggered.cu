// staggered.cu -- improved staggered (asqtad) path: link loading, colour-vector
// pack / unpack, the hopping term and M^dag M on one parity, and the paper's
// solver for the shifted systems (M^dag M + sigma_i) x_i = b of Eq. 4: single-precision multi-shift CG
// followed by sequential mixed-precision CG refinement of every x_i.
#include <cmath>
#include <cstring>
#include <vector>
#include "blas_ops.cuh"
#include "ops.h"
#include "staggered.cuh"

using namespace lq;

namespace {

// canonical chi[t][z][y][x][3] (complex128) <-> packed parity field of precision P
template <class P>
__global__ void pack_colour_kernel(char* packed, double* canonical, const Geom g, int parity, int unpack) {
  typedef typename P::real R;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.ns) return;
  int c[4];
  cb_to_coords(g, (int)i, parity, c);
  const long long site = c[0] + (long long)g.X[0] * (c[1] + (long long)g.X[1] * (c[2] + (long long)g.X[2] * c[3]));
  double* p = canonical + site * 6;
  R v[6];
  if (!unpack) {
#pragma unroll
    for (int k = 0; k < 6; ++k) v[k] = (R)p[k];
    Colour<P>::store(v, packed, g.ns >> 2, i);
  } else {
    Colour<P>::load(v, packed, g.ns >> 2, i);
#pragma unroll
    for (int k = 0; k < 6; ++k) p[k] = (double)v[k];
  }
}

cudaError_t run_pack_colour(int prec, char* packed, const double* canonical, const Geom& nat, int parity, int unpack, cudaStream_t s) {
  dim3 grid((unsigned)((nat.ns + 127) / 128)), block(128);
  double* c = const_cast<double*>(canonical);
  if (prec == 0) pack_colour_kernel<PrecD><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack);
  else if (prec == 1) pack_colour_kernel<PrecS><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack);
  else return cudaErrorInvalidValue;
  return cudaGetLastError();
}

template <class P>
cudaError_t launch_stag(const StagArgs& a, bool xpay, cudaStream_t s) {
  dim3 grid((a.g.vh + LQ_STAG_BLOCK - 1) / LQ_STAG_BLOCK), block(LQ_STAG_BLOCK);
  if (xpay) stag_dslash_kernel<P, true><<<grid, block, 0, s>>>(a);
  else stag_dslash_kernel<P, false><<<grid, block, 0, s>>>(a);
  return cudaGetLastError();
}

size_t colour_bytes(int prec, long long vh) { return (size_t)vh * 6 * (prec == 0 ? 8 : 4); }

int stag_check(lqcd_ctx* c, int prec) {
  if (prec != LQCD_PREC_DOUBLE && prec != LQCD_PREC_SINGLE) return fail(c, LQCD_EINVAL, "staggered fields are fp64 or fp32");
  if (!c->have_stag) return fail(c, LQCD_ESTATE, "staggered links not loaded");
  return LQCD_OK;
}

// fp64 masters -> links of precision prec (recon-18 records), on first use
int stag_links(lqcd_ctx* c, int prec, const char** fat, const char** lng, cudaStream_t s) {
  if (prec == 0) { *fat = (const char*)c->sfat64; *lng = (const char*)c->slng64; return LQCD_OK; }
  if (!c->sfat32) {
    int rc = dev_alloc(c, (void**)&c->sfat32, gauge_bytes(1, 18, c->nat.ns));
    if (!rc) rc = dev_alloc(c, (void**)&c->slng32, gauge_bytes(1, 18, c->nat.ns));
    if (rc) return rc;
    cudaError_t e = run_convert_gauge(1, 18, c->sfat32, c->sfat64, c->bm, 0, s); c->launches++;
    if (e == cudaSuccess) { e = run_convert_gauge(1, 18, c->slng32, c->slng64, c->bm, 0, s); c->launches++; }
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "convert staggered links", e);
  }
  *fat = c->sfat32; *lng = c->slng32;
  return LQCD_OK;
}

// out = a*y + b*(D in) (y != nullptr) or out = D in, output parity p
int op_stag_dslash(lqcd_ctx* c, char* out, const char* in, const char* y, double a, double b, int p, int prec, cudaStream_t s) {
  StagArgs d;
  memset(&d, 0, sizeof(d));
  d.g = c->nat;
  d.out = out; d.in = in; d.y = y; d.a = a; d.b = b; d.parity = p;
  int rc = stag_links(c, prec, &d.fat, &d.lng, s);
  if (rc) return rc;
  cudaError_t e = prec == 0 ? launch_stag<PrecD>(d, y != nullptr, s) : launch_stag<PrecS>(d, y != nullptr, s);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "staggered dslash launch", e);
}

// out = (M^dag M + sigma) in on parity p = (m^2 + sigma) in - 1/4 D_{p,pbar} D_{pbar,p} in   (R14)
int op_stag_mdagm(lqcd_ctx* c, char* out, const char* in, int p, double mass, double sigma, int prec, cudaStream_t s) {
  char*& tmp = c->stmp[prec];
  if (!tmp) { int rc = dev_alloc(c, (void**)&tmp, colour_bytes(prec, c->Vh)); if (rc) return rc; }
  int rc = op_stag_dslash(c, tmp, in, nullptr, 0, 0, 1 - p, prec, s);
  if (rc) return rc;
  return op_stag_dslash(c, out, tmp, in, mass * mass + sigma, -0.25, p, prec, s);
}

}  // namespace

// ================================================================================================
extern "C" {

int lqcd_load_staggered_links(lqcd_ctx* c, const void* fat, const void* lng, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!fat || !lng) return fail(c, LQCD_EINVAL, "null link pointer");
  for (int m = 0; m < 4; ++m) if (c->dims[m] < 4) return fail(c, LQCD_EINVAL, "the three-hop term needs every extent >= 4");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  int rc;
  if (!c->sfat64 && (rc = dev_alloc(c, (void**)&c->sfat64, gauge_bytes(0, 18, c->nat.ns)))) return rc;
  if (!c->slng64 && (rc = dev_alloc(c, (void**)&c->slng64, gauge_bytes(0, 18, c->nat.ns)))) return rc;
  if (c->sfat32) { cudaFree(c->sfat32); c->sfat32 = nullptr; }
  if (c->slng32) { cudaFree(c->slng32); c->slng32 = nullptr; }
  cudaError_t e = run_pack_gauge(c->sfat64, (const double*)fat, c->nat, s); c->launches++;
  if (e == cudaSuccess) { e = run_pack_gauge(c->slng64, (const double*)lng, c->nat, s); c->launches++; }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack staggered links", e);
  c->have_stag = true;
  return LQCD_OK;
}

int lqcd_pack_staggered(lqcd_ctx* c, void* packed, const void* canonical, int parity, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!packed || !canonical || (parity | 1) != 1 || (prec != 0 && prec != 1)) return fail(c, LQCD_EINVAL, "pack_staggered arguments");
  cudaSetDevice(c->device);
  cudaError_t e = run_pack_colour(prec, (char*)packed, (const double*)canonical, c->nat, parity, 0, (cudaStream_t)stream);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "pack_staggered", e);
}

int lqcd_unpack_staggered(lqcd_ctx* c, void* canonical, const void* packed, int parity, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!packed || !canonical || (parity | 1) != 1 || (prec != 0 && prec != 1)) return fail(c, LQCD_EINVAL, "unpack_staggered arguments");
  cudaSetDevice(c->device);
  cudaError_t e = run_pack_colour(prec, (char*)packed, (const double*)canonical, c->nat, parity, 1, (cudaStream_t)stream);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "unpack_staggered", e);
}

int lqcd_staggered_dslash(lqcd_ctx* c, void* out, const void* in, int parity_out, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity_out | 1) != 1) return fail(c, LQCD_EINVAL, "staggered_dslash arguments");
  int rc = stag_check(c, prec);
  if (rc) return rc;
  cudaSetDevice(c->device);
  return op_stag_dslash(c, (char*)out, (const char*)in, nullptr, 0, 0, parity_out, prec, (cudaStream_t)stream);
}

int lqcd_staggered_mdagm(lqcd_ctx* c, void* out, const void* in, int parity, double mass, double sigma, int prec, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!out || !in || out == in || (parity | 1) != 1) return fail(c, LQCD_EINVAL, "staggered_mdagm arguments");
  int rc = stag_check(c, prec);
  if (rc) return rc;
  cudaSetDevice(c->device);
  return op_stag_mdagm(c, (char*)out, (const char*)in, parity, mass, sigma, prec, (cudaStream_t)stream);
}

}  // extern "C"
