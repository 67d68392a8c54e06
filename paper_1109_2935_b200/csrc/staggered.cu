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
cudaError_t launch_stag(const StagArgs& a, bool xpay, bool long12, cudaStream_t s) {
  dim3 grid((a.g.vh + LQ_STAG_BLOCK - 1) / LQ_STAG_BLOCK), block(LQ_STAG_BLOCK);
  if (long12) {
    if (xpay) stag_dslash_kernel<P, true, 12><<<grid, block, 0, s>>>(a);
    else stag_dslash_kernel<P, false, 12><<<grid, block, 0, s>>>(a);
  } else {
    if (xpay) stag_dslash_kernel<P, true, 18><<<grid, block, 0, s>>>(a);
    else stag_dslash_kernel<P, false, 18><<<grid, block, 0, s>>>(a);
  }
  return cudaGetLastError();
}

// max over links of || L L^dag / scale^2 - 1 ||_max and |det L / scale^3 - 1| : is every long link scale x SU(3)?
__global__ void long_link_check_kernel(const double* __restrict__ lng, long long nlinks, double inv2, double inv3, double* out) {
  double worst = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nlinks; i += (long long)gridDim.x * blockDim.x) {
    const double* u = lng + i * 18;
    for (int r = 0; r < 3; ++r)
      for (int q = 0; q < 3; ++q) {
        double re = 0, im = 0;
        for (int k = 0; k < 3; ++k) {
          re += u[6 * r + 2 * k] * u[6 * q + 2 * k] + u[6 * r + 2 * k + 1] * u[6 * q + 2 * k + 1];
          im += u[6 * r + 2 * k + 1] * u[6 * q + 2 * k] - u[6 * r + 2 * k] * u[6 * q + 2 * k + 1];
        }
        worst = fmax(worst, fmax(fabs(re * inv2 - (r == q ? 1.0 : 0.0)), fabs(im * inv2)));
      }
    // det L = scale^3 (row 2 = conj(row0 x row1) / scale needs det = 1 as well as unitarity)
    double dr = 0, di = 0;
    for (int c0 = 0; c0 < 3; ++c0) {
      const int j = (c0 + 1) % 3, k = (c0 + 2) % 3;
      const double cr = u[6 + 2 * j] * u[12 + 2 * k] - u[6 + 2 * j + 1] * u[12 + 2 * k + 1] - u[6 + 2 * k] * u[12 + 2 * j] + u[6 + 2 * k + 1] * u[12 + 2 * j + 1];
      const double ci = u[6 + 2 * j] * u[12 + 2 * k + 1] + u[6 + 2 * j + 1] * u[12 + 2 * k] - u[6 + 2 * k] * u[12 + 2 * j + 1] - u[6 + 2 * k + 1] * u[12 + 2 * j];
      dr += u[2 * c0] * cr - u[2 * c0 + 1] * ci;
      di += u[2 * c0] * ci + u[2 * c0 + 1] * cr;
    }
    worst = fmax(worst, fmax(fabs(dr * inv3 - 1.0), fabs(di * inv3)));
  }
  for (int o = 16; o > 0; o >>= 1) worst = fmax(worst, __shfl_down_sync(0xffffffffu, worst, o));
  if ((threadIdx.x & 31) == 0 && worst > 0) atomicMax((unsigned long long*)out, (unsigned long long)__double_as_longlong(worst));
}

size_t colour_bytes(int prec, long long vh) { return (size_t)vh * 6 * (prec == 0 ? 8 : 4); }

int stag_check(lqcd_ctx* c, int prec) {
  if (prec != LQCD_PREC_DOUBLE && prec != LQCD_PREC_SINGLE) return fail(c, LQCD_EINVAL, "staggered fields are fp64 or fp32");
  if (!c->have_stag) return fail(c, LQCD_ESTATE, "staggered links not loaded");
  return LQCD_OK;
}

// fp64 masters -> links of precision prec (recon-18 records), on first use
// (the long links are 12-real records when the caller declared them long_scale x SU(3))
int stag_links(lqcd_ctx* c, int prec, const char** fat, const char** lng, cudaStream_t s) {
  const int lr = c->slong_scale != 0.0 ? 12 : 18;
  if (prec == 0 && lr == 18) { *fat = (const char*)c->sfat64; *lng = (const char*)c->slng64; return LQCD_OK; }
  char*& f = c->sfatp[prec];
  char*& l = c->slngp[prec];
  if (!l) {
    int rc = LQCD_OK;
    if (prec == 1) rc = dev_alloc(c, (void**)&f, gauge_bytes(1, 18, c->nat.ns));
    if (!rc) rc = dev_alloc(c, (void**)&l, gauge_bytes(prec, lr, c->nat.ns));
    if (rc) return rc;
    cudaError_t e = cudaSuccess;
    if (prec == 1) { e = run_convert_gauge(1, 18, f, c->sfat64, c->bm, 0, s); c->launches++; }
    if (e == cudaSuccess) { e = run_convert_gauge(prec, lr, l, c->slng64, c->bm, 0, s); c->launches++; }
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "convert staggered links", e);
  }
  *fat = prec == 0 ? (const char*)c->sfat64 : f;
  *lng = l;
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
  const bool l12 = c->slong_scale != 0.0;
  d.linv = l12 ? 1.0 / c->slong_scale : 0.0;
  cudaError_t e = prec == 0 ? launch_stag<PrecD>(d, y != nullptr, l12, s) : launch_stag<PrecS>(d, y != nullptr, l12, s);
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

// ---------------------------------------------------------------- solver for Eq. 4
struct MsArgs {
  const char* r;
  char* x[LQ_MS_MAX];
  char* p[LQ_MS_MAX];
  const double* S;
  long long ns;         // records (= Vh/4)
  int n;                // active shifts (a prefix: shifts are sorted ascending, larger ones converge first)
};

// one pass over r: x_i += alpha_i p_i ; p_i = zeta_i r + beta_i p_i for every active shift
template <class P>
__global__ void __launch_bounds__(LQ_BLAS_BLOCK) ms_update_kernel(const MsArgs m) {
  typedef typename P::real R;
  const long long i = (long long)blockIdx.x * LQ_BLAS_BLOCK + threadIdx.x;
  if (i >= m.ns) return;
  R r[24];
  load_site<P, 24>(r, m.r, m.ns, i);
  for (int k = 0; k < m.n; ++k) {
    const double* sc = m.S + S_MS + LQ_MS_STRIDE * k;
    const R z = (R)sc[0], al = (R)sc[2], be = (R)sc[3];
    R x[24], p[24];
    load_site<P, 24>(x, m.x[k], m.ns, i);
    load_site<P, 24>(p, m.p[k], m.ns, i);
#pragma unroll
    for (int j = 0; j < 24; ++j) { x[j] = fma_(al, p[j], x[j]); p[j] = fma_(be, p[j], z * r[j]); }
    store_site<P, 24>(x, m.x[k], m.ns, i);
    store_site<P, 24>(p, m.p[k], m.ns, i);
  }
}

BlasArgs mks(lqcd_ctx* c, char* v0 = nullptr, char* v1 = nullptr, char* v2 = nullptr, char* v3 = nullptr) {
  BlasArgs a;
  memset(&a, 0, sizeof(a));
  a.v[0] = v0; a.v[1] = v1; a.v[2] = v2; a.v[3] = v3;
  a.ns = c->Vh / 4; a.vh = (int)(c->Vh / 4); a.nb = 1;      // quad-site records (staggered.cuh)
  a.S = c->S; a.partials = c->partials; a.counters = c->counters;
  return a;
}
template <class Op> int sblas(lqcd_ctx* c, int prec, const BlasArgs& a, cudaStream_t s) {
  cudaError_t e = run_blas<Op>(prec, a, c->n_sm * LQ_BLAS_CTAS_PER_SM, s, 1);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "staggered blas launch", e);
}
int sread(lqcd_ctx* c, int off, int n, cudaStream_t s) {
  cudaError_t e = cudaMemcpyAsync(c->hS + off, c->S + off, n * sizeof(double), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "scalar read-back", e);
}
int sconvert(lqcd_ctx* c, int pa, int pb, char* dst, const char* src, cudaStream_t s) {
  BlockMap bm = c->bm;
  bm.nat.ns = c->Vh / 4; bm.nat.vh = (int)(c->Vh / 4);
  cudaError_t e = run_convert(pa, pb, dst, src, bm, 0, 0, s);
  c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "convert", e);
}
// y (fp64) += x (fp32)
int saccumulate(lqcd_ctx* c, char* y, char* x, cudaStream_t s) {
  MultiArgs m; memset(&m, 0, sizeof(m));
  m.b = mks(c); m.z[0] = x; m.chi[0] = 1.0; m.n = 1;
  cudaError_t e = run_accumulate(0, 1, y, m, s); c->launches++;
  return e == cudaSuccess ? LQCD_OK : fail(c, LQCD_ECUDA, "accumulate", e);
}
// r = b - (M^dag M + sigma) x in fp64 ; *rn = ||r||
int sresidual(lqcd_ctx* c, char* r, const char* b, const char* x, int par, double mass, double sigma, double* rn, cudaStream_t s) {
  int rc = op_stag_mdagm(c, r, x, par, mass, sigma, 0, s);
  if (rc) return rc;
  BlasArgs a = mks(c, const_cast<char*>(b), r);
  if ((rc = sblas<OpXmyNorm>(c, 0, a, s))) return rc;
  if ((rc = sread(c, S_OUT, 1, s))) return rc;
  *rn = sqrt(c->hS[S_OUT]);
  return LQCD_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

int lqcd_load_staggered_links(lqcd_ctx* c, const void* fat, const void* lng, double long_scale, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!fat || !lng) return fail(c, LQCD_EINVAL, "null link pointer");
  for (int m = 0; m < 4; ++m) if (c->dims[m] < 4) return fail(c, LQCD_EINVAL, "the three-hop term needs every extent >= 4");
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  int rc;
  if (!c->sfat64 && (rc = dev_alloc(c, (void**)&c->sfat64, gauge_bytes(0, 18, c->nat.ns)))) return rc;
  if (!c->slng64 && (rc = dev_alloc(c, (void**)&c->slng64, gauge_bytes(0, 18, c->nat.ns)))) return rc;
  for (int i = 0; i < 2; ++i) {
    if (c->sfatp[i]) { cudaFree(c->sfatp[i]); c->sfatp[i] = nullptr; }
    if (c->slngp[i]) { cudaFree(c->slngp[i]); c->slngp[i] = nullptr; }
  }
  c->have_stag = false;
  if (long_scale != 0.0) {
    // the caller says every long link is long_scale x SU(3): check it before trusting a 12-real encoding
    cudaError_t e = cudaMemsetAsync(c->S + S_OUT, 0, sizeof(double), s);
    if (e == cudaSuccess) {
      long_link_check_kernel<<<c->n_sm * 4, 256, 0, s>>>((const double*)lng, 4 * c->V, 1.0 / (long_scale * long_scale), 1.0 / (long_scale * long_scale * long_scale), c->S + S_OUT);
      c->launches++;
      e = cudaMemcpyAsync(c->hS + S_OUT, c->S + S_OUT, sizeof(double), cudaMemcpyDeviceToHost, s);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "long link check", e);
    if (!(c->hS[S_OUT] <= 1e-10)) return fail(c, LQCD_EINVAL, "long links are not long_scale x SU(3); pass long_scale = 0");
  }
  cudaError_t e = run_pack_gauge(c->sfat64, (const double*)fat, c->nat, s); c->launches++;
  if (e == cudaSuccess) { e = run_pack_gauge(c->slng64, (const double*)lng, c->nat, s); c->launches++; }
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack staggered links", e);
  c->slong_scale = long_scale;
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

// (M^dag M + sigma_i) x_i = b on one parity, i < nshift (Eq. 4), by the paper's strategy
// (PAPER.md:296): a pure single-precision multi-shift CG for all shifts at once, then sequential
// mixed-precision CG (fp64 outer with reliable updates, fp32 inner) refining every x_i to `tol`.
// multishift_prec = LQCD_PREC_DOUBLE runs the multi-shift phase in fp64 to `tol` instead (the memory and
// fp64 rate that ruled it out on the paper's GPUs, are not a constraint on B200).
int lqcd_staggered_multishift(lqcd_ctx* c, void* x_can, const void* b_can, int parity, double mass, const double* sigma,
                              int nshift, double tol, int max_iter, int multishift_prec, lqcd_invert_result* res, void* stream) {
  if (!c) return LQCD_EINVAL;
  if (!x_can || !b_can || !sigma || !res || (parity | 1) != 1 || nshift < 1 || nshift > LQ_MS_MAX || !(tol > 0) || max_iter < 1 ||
      (multishift_prec != LQCD_PREC_SINGLE && multishift_prec != LQCD_PREC_DOUBLE))
    return fail(c, LQCD_EINVAL, "staggered_multishift arguments");
  for (int i = 0; i < nshift; ++i) if (!(sigma[i] >= 0.0)) return fail(c, LQCD_EINVAL, "shifts must be >= 0");
  for (int i = 1; i < nshift; ++i) if (!(sigma[i] > sigma[i - 1])) return fail(c, LQCD_EINVAL, "shifts must be strictly ascending");
  int rc = stag_check(c, 0);
  if (rc) return rc;
  cudaSetDevice(c->device);
  cudaStream_t s = (cudaStream_t)stream;
  memset(res, 0, sizeof(*res) * nshift);
  const size_t f64 = colour_bytes(0, c->Vh), f32 = colour_bytes(1, c->Vh), cbytes = (size_t)c->V * 6 * sizeof(double);
  struct Bufs {                                           // workspace from / back to the context's cache
    lqcd_ctx* c; cudaStream_t s; std::vector<std::pair<void*, size_t>> v;
    ~Bufs() { for (auto& b : v) ws_put(c, b.first, b.second, s); }
  } bufs{c, s, {}};
  auto get = [&](char** out, size_t bytes) -> int {
    void* p = nullptr;
    int rc2 = ws_get(c, &p, bytes, s);
    if (rc2) return rc2;
    bufs.v.push_back({p, bytes}); *out = (char*)p;
    return LQCD_OK;
  };
  char *b_hi, *x_hi, *r_hi, *r, *ap, *xs, *ps;
  const int pm = multishift_prec;
  const size_t fm = pm == 0 ? f64 : f32;
  if ((rc = get(&b_hi, f64)) || (rc = get(&x_hi, f64)) || (rc = get(&r_hi, f64)) || (rc = get(&r, fm)) || (rc = get(&ap, fm)) ||
      (rc = get(&xs, fm * nshift)) || (rc = get(&ps, fm * nshift))) return rc;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  struct Ev { cudaEvent_t a, b; ~Ev() { cudaEventDestroy(a); cudaEventDestroy(b); } } ev{e0, e1};
  cudaEventRecord(e0, s);
  cudaError_t e = run_pack_colour(0, b_hi, (const double*)b_can, c->nat, parity, 0, s); c->launches++;
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "pack", e);
  double bn;
  { BlasArgs a = mks(c, b_hi); a.i0 = 0; if ((rc = sblas<OpNorm2>(c, 0, a, s))) return rc; }
  if ((rc = sread(c, S_OUT, 1, s))) return rc;
  bn = sqrt(c->hS[S_OUT]);
  e = cudaMemsetAsync(x_can, 0, cbytes * nshift, s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "memset", e);
  long long n_lo = 0, n_hi = 0;
  double blas_sites = 0;
  int ms_iters = 0, worst = LQCD_OK;
  if (bn > 0.0) {
    // ---- phase 1: multi-shift CG in precision pm (single = the paper's strategy), all x_i = 0, r = p_i = b
    if ((rc = sconvert(c, 0, pm, r, b_hi, s))) return rc;
    for (int i = 0; i < nshift; ++i) {
      if ((rc = sconvert(c, pm, pm, ps + i * fm, r, s))) return rc;
      BlasArgs a = mks(c, xs + i * fm); if ((rc = sblas<OpZero>(c, pm, a, s))) return rc;
    }
    { BlasArgs a = mks(c, r); a.i0 = 0; if ((rc = sblas<OpCgInit>(c, pm, a, s))) return rc; }      // rr -> S_RHO, flag = 0
    {
      double* h = c->hS;                                  // initial multi-shift state
      for (int i = 0; i < nshift; ++i) {
        double* m = h + S_MS + LQ_MS_STRIDE * i;
        m[0] = 1; m[1] = 1; m[2] = 0; m[3] = 0; m[4] = sigma[i] - sigma[0];
      }
      h[S_MS_AOLD] = 1; h[S_MS_BOLD] = 0; h[S_MS_N] = nshift;
      e = cudaMemcpyAsync(c->S + S_MS, h + S_MS, (S_MS_N + 1 - S_MS) * sizeof(double), cudaMemcpyHostToDevice, s);
      if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "multi-shift state", e);
    }
    // single precision cannot resolve more than ~1e-6 of the source; the refinement takes over from there
    const double ms_stop = (pm == 0 ? tol : (tol > 2e-6 ? tol : 2e-6)) * bn;
    int active = nshift;
    double rn = bn, best = bn;
    int stall = 0;
    while (rn > ms_stop && ms_iters < max_iter) {
      if ((rc = op_stag_mdagm(c, ap, ps, parity, mass, sigma[0], pm, s))) return rc;
      { BlasArgs a = mks(c, ps, ap); if ((rc = sblas<OpCgPAp>(c, pm, a, s))) return rc; }
      { BlasArgs a = mks(c, r, ap); if ((rc = sblas<OpMsR>(c, pm, a, s))) return rc; }
      MsArgs m; memset(&m, 0, sizeof(m));
      m.r = r; m.S = c->S; m.ns = c->Vh / 4; m.n = active;
      for (int i = 0; i < active; ++i) { m.x[i] = xs + i * fm; m.p[i] = ps + i * fm; }
      if (pm == 0) ms_update_kernel<PrecD><<<(unsigned)((m.ns + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK), LQ_BLAS_BLOCK, 0, s>>>(m);
      else ms_update_kernel<PrecS><<<(unsigned)((m.ns + LQ_BLAS_BLOCK - 1) / LQ_BLAS_BLOCK), LQ_BLAS_BLOCK, 0, s>>>(m);
      c->launches++;
      if ((e = cudaGetLastError()) != cudaSuccess) return fail(c, LQCD_ECUDA, "ms_update", e);
      ++ms_iters; if (pm == 0) ++n_hi; else ++n_lo; blas_sites += 6.0 * (2 + 3 + 5 * active);
      if ((rc = sread(c, 0, S_MS_N + 1, s))) return rc;
      const double rr = c->hS[S_RR];
      if (!(rr == rr) || c->hS[S_FLAG] != 0.0) { worst = LQCD_EBREAKDOWN; break; }
      rn = sqrt(rr);
      // a shift whose own residual |zeta_i| ||r|| is below the target is finished: drop it (it is a suffix)
      while (active > 1 && fabs(c->hS[S_MS + LQ_MS_STRIDE * (active - 1)]) * rn <= ms_stop) --active;
      if (rn < 0.999 * best) { best = rn; stall = 0; } else if (++stall > 50) break;     // precision floor reached
    }
  }
  // ---- phase 2: sequential mixed-precision CG refinement of every shift (fp64 outer, fp32 inner)
  const double stop = tol * bn, delta = 0.1;
  worst = LQCD_OK;                                         // a breakdown of the single-precision phase is repaired below
  char *xl = r, *rl = ap;                                  // fp32 work fields reused: x_l, r_l ; p and A p below
  char *pl, *apl;
  if ((rc = get(&pl, f32)) || (rc = get(&apl, f32))) return rc;
  for (int i = 0; i < nshift; ++i) {
    lqcd_invert_result& R = res[i];
    if (bn == 0.0) { R.status = LQCD_OK; continue; }
    if ((rc = sconvert(c, pm, 0, x_hi, xs + i * fm, s))) return rc;
    double rn;
    if ((rc = sresidual(c, r_hi, b_hi, x_hi, parity, mass, sigma[i], &rn, s))) return rc;
    ++n_hi; R.matpc_outer++;
    int status = LQCD_OK;
    if (!(rn == rn)) {                                     // the single-precision phase broke down: start from zero
      BlasArgs a = mks(c, x_hi); if ((rc = sblas<OpZero>(c, 0, a, s))) return rc;
      if ((rc = sresidual(c, r_hi, b_hi, x_hi, parity, mass, sigma[i], &rn, s))) return rc;
      ++n_hi; R.matpc_outer++; status = LQCD_OK;
    }
    int it = 0;
    bool fresh = true;                                      // start (or restart) the direction p = r
    double maxr = rn;
    while (rn > stop) {
      if (fresh) {
        if ((rc = sconvert(c, 0, 1, rl, r_hi, s))) return rc;
        { BlasArgs a = mks(c, xl); if ((rc = sblas<OpZero>(c, 1, a, s))) return rc; }
        { BlasArgs a = mks(c, pl); if ((rc = sblas<OpZero>(c, 1, a, s))) return rc; }
        { BlasArgs a = mks(c, rl); a.i0 = 0; if ((rc = sblas<OpCgInit>(c, 1, a, s))) return rc; }
        { BlasArgs a = mks(c, pl, rl); if ((rc = sblas<OpCgP>(c, 1, a, s))) return rc; }
        fresh = false;
      }
      if (it >= max_iter) { status = LQCD_ENOCONV; break; }
      if ((rc = op_stag_mdagm(c, apl, pl, parity, mass, sigma[i], 1, s))) return rc;
      { BlasArgs a = mks(c, pl, apl); if ((rc = sblas<OpCgPAp>(c, 1, a, s))) return rc; }
      { BlasArgs a = mks(c, xl, pl, rl, apl); if ((rc = sblas<OpCgXRB>(c, 1, a, s))) return rc; }
      { BlasArgs a = mks(c, pl, rl); if ((rc = sblas<OpCgP>(c, 1, a, s))) return rc; }
      ++it; ++n_lo; R.matpc_sloppy++; blas_sites += 6.0 * (2 + 6 + 3);
      if ((rc = sread(c, S_RR, 2, s))) return rc;
      const double rr = c->hS[S_RR];
      const bool bad = !(rr == rr) || c->hS[S_FLAG] != 0.0;
      const double rln = sqrt(rr);
      if (rln > maxr) maxr = rln;
      if (bad || rln <= stop || rln < delta * maxr) {
        // reliable update: x += x_l, true residual in fp64; the direction is kept (beta from the new residual)
        if ((rc = saccumulate(c, x_hi, xl, s))) return rc;
        { BlasArgs a = mks(c, xl); if ((rc = sblas<OpZero>(c, 1, a, s))) return rc; }
        if ((rc = sresidual(c, r_hi, b_hi, x_hi, parity, mass, sigma[i], &rn, s))) return rc;
        ++n_hi; R.matpc_outer++; R.restarts++;
        if (!(rn == rn)) { status = LQCD_EBREAKDOWN; break; }
        if (rn <= stop) break;
        maxr = rn;
        if (bad) { fresh = true; continue; }
        if ((rc = sconvert(c, 0, 1, rl, r_hi, s))) return rc;
        { BlasArgs a = mks(c, rl); a.i0 = 2; if ((rc = sblas<OpCgInit>(c, 1, a, s))) return rc; }   // beta = rr_new / rr_old
        { BlasArgs a = mks(c, pl, rl); if ((rc = sblas<OpCgP>(c, 1, a, s))) return rc; }
      }
    }
    if (status == LQCD_ENOCONV) {                          // fold what the inner iteration has and report its true residual
      if ((rc = saccumulate(c, x_hi, xl, s))) return rc;
      if ((rc = sresidual(c, r_hi, b_hi, x_hi, parity, mass, sigma[i], &rn, s))) return rc;
      ++n_hi; R.matpc_outer++;
    }
    R.status = status; R.iterations = it;
    R.true_residual = rn / bn; R.iterated_residual = rn / bn;
    if (status != LQCD_OK && worst == LQCD_OK) worst = status;
    e = run_pack_colour(0, x_hi, (const double*)((const char*)x_can + i * cbytes), c->nat, parity, 1, s); c->launches++;
    if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "unpack", e);
  }
  res[0].matpc_sloppy += ms_iters;
  res[0].matpc_precond = ms_iters;                          // iterations of the multi-shift phase
  cudaEventRecord(e1, s);
  e = cudaStreamSynchronize(s);
  if (e != cudaSuccess) return fail(c, LQCD_ECUDA, "staggered_multishift", e);
  float ms = 0;
  cudaEventElapsedTime(&ms, e0, e1);
  const double gflop = ((double)(n_lo + n_hi) * (2.0 * 1146 + 12) + blas_sites) * (double)c->Vh * 1e-9;
  for (int i = 0; i < nshift; ++i) { res[i].seconds = ms * 1e-3; res[i].gflop = gflop; }
  if (worst == LQCD_ENOCONV) return fail(c, worst, "max_iter reached for at least one shift");
  if (worst == LQCD_EBREAKDOWN) return fail(c, worst, "breakdown for at least one shift");
  return LQCD_OK;
}

}  // extern "C"
