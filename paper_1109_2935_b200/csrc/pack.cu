// pack.cu -- boundary kernels: canonical (lexicographic AoS complex128) <-> packed fields.
// Setup path: the gauge field "must only be transferred once at the
// beginning of a solve"; compression 18 -> 12 / 8 reals per link.
#include "host.h"

namespace lq {

// canonical U[mu][t][z][y][x][3][3] -> fp64 recon-18 checkerboarded SoA [parity][mu]
__global__ void pack_gauge_kernel(double* g64, const double* __restrict__ U, const Geom g) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.ns) return;
  const int pm = blockIdx.y, parity = pm >> 2, mu = pm & 3;
  int c[4];
  cb_to_coords(g, (int)i, parity, c);
  const long long V = 2 * g.ns;
  const long long site = c[0] + (long long)g.X[0] * (c[1] + (long long)g.X[1] * (c[2] + (long long)g.X[2] * c[3]));
  const double* src = U + ((long long)mu * V + site) * 18;
  alignas(16) double u[18];
#pragma unroll
  for (int k = 0; k < 18; ++k) u[k] = src[k];
  Rec<double, 18>::store(u, (char*)g64 + (long long)pm * 144 * g.ns, g.ns, i);
}

cudaError_t run_pack_gauge(double* g64, const double* U, const Geom& nat, cudaStream_t s) {
  dim3 grid((unsigned)((nat.ns + 127) / 128), 8), block(128);
  pack_gauge_kernel<<<grid, block, 0, s>>>(g64, U, nat);
  return cudaGetLastError();
}

// fp64 recon-18 natural -> (P, RECON), natural or block-major
template <class P, int RECON>
__global__ void convert_gauge_kernel(char* dst, const double* __restrict__ g64, const BlockMap bm, int blocked) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= bm.nat.ns) return;
  const int pm = blockIdx.y, parity = pm >> 2;
  long long is = i;
  if (blocked) is = block_to_natural(bm, (int)(i / bm.blk.vh), (int)(i % bm.blk.vh), parity);
  alignas(16) double u[18];
  Rec<double, 18>::load(u, (const char*)g64 + (long long)pm * 144 * bm.nat.ns, bm.nat.ns, is);
  double v[RECON];
  compress_link<RECON>(u, v);
  alignas(16) typename P::store_t q[RECON];
  quantize_link<P, RECON>(v, q);
  Rec<typename P::store_t, RECON>::store(q, dst + (long long)pm * RECON * sizeof(typename P::store_t) * bm.nat.ns, bm.nat.ns, i);
}

template <class P>
static cudaError_t convert_gauge_p(int recon, char* dst, const double* g64, const BlockMap& bm, int blocked, cudaStream_t s) {
  dim3 grid((unsigned)((bm.nat.ns + 127) / 128), 8), block(128);
  switch (recon) {
    case 18: convert_gauge_kernel<P, 18><<<grid, block, 0, s>>>(dst, g64, bm, blocked); break;
    case 12: convert_gauge_kernel<P, 12><<<grid, block, 0, s>>>(dst, g64, bm, blocked); break;
    case 8:  convert_gauge_kernel<P, 8><<<grid, block, 0, s>>>(dst, g64, bm, blocked); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_convert_gauge(int prec, int recon, char* dst, const double* g64, const BlockMap& bm, int blocked, cudaStream_t s) {
  switch (prec) {
    case 0: return convert_gauge_p<PrecD>(recon, dst, g64, bm, blocked, s);
    case 1: return convert_gauge_p<PrecS>(recon, dst, g64, bm, blocked, s);
    case 2: return convert_gauge_p<PrecH>(recon, dst, g64, bm, blocked, s);
  }
  return cudaErrorInvalidValue;
}

// canonical psi[t][z][y][x][4][3] (complex128) <-> packed parity field of precision P
template <class P>
__global__ void pack_spinor_kernel(char* packed, double* canonical, const Geom g, int parity, int unpack, long long i0, long long i1) {
  const long long i = i0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= i1) return;
  int c[4];
  cb_to_coords(g, (int)i, parity, c);
  const long long site = c[0] + (long long)g.X[0] * (c[1] + (long long)g.X[1] * (c[2] + (long long)g.X[2] * c[3]));
  double* p = canonical + site * 24;
  typename P::real v[24];
  if (!unpack) {
#pragma unroll
    for (int k = 0; k < 24; ++k) v[k] = (typename P::real)p[k];
    store_site<P, 24>(v, packed, g.ns, i);
  } else {
    load_site<P, 24>(v, packed, g.ns, i);
#pragma unroll
    for (int k = 0; k < 24; ++k) p[k] = (double)v[k];
  }
}

cudaError_t run_pack_spinor(int prec, char* packed, const double* canonical, const Geom& nat, int parity, int unpack, cudaStream_t s,
                            long long i0, long long i1) {
  if (i1 < 0) i1 = nat.ns;
  dim3 grid((unsigned)((i1 - i0 + 127) / 128)), block(128);
  double* c = const_cast<double*>(canonical);
  switch (prec) {
    case 0: pack_spinor_kernel<PrecD><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    case 1: pack_spinor_kernel<PrecS><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    case 2: pack_spinor_kernel<PrecH><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace lq
