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

// fp64 recon-18 natural -> (P, RECON), natural or block-major.
// Compressed forms hold SU(3) links only (PAPER.md:164 (a); R10), and recon-8 cannot hold a link whose first row is
// (a1, 0, 0) (N = |a2|^2 + |a3|^2 = 0, e.g. U = 1: the lower 2x2 block is then not determined by the 8 stored reals).
// `bad` (device word, may be null) collects: bit 0 = a link is not SU(3) to 1e-9 (unitarity or determinant),
// bit 1 = a recon-8 link has N = 0 in the stored precision (the in-kernel reconstruction would divide by zero).
template <class P, int RECON>
__global__ void convert_gauge_kernel(char* dst, const double* __restrict__ g64, const BlockMap bm, int blocked, unsigned* bad) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long ns_d = blocked ? bm.blk.ns : bm.nat.ns;      // block-major copies have their own size with overlapping domains (host.h)
  if (i >= ns_d) return;
  const int pm = blockIdx.y, parity = pm >> 2;
  long long is = i;
  if (blocked) is = block_to_natural(bm, (int)(i / bm.blk.vh), (int)(i % bm.blk.vh), parity);
  alignas(16) double u[18];
  Rec<double, 18>::load(u, (const char*)g64 + (long long)pm * 144 * bm.nat.ns, bm.nat.ns, is);
  double v[RECON];
  compress_link<RECON>(u, v);
  alignas(16) typename P::store_t q[RECON];
  quantize_link<P, RECON>(v, q);
  Rec<typename P::store_t, RECON>::store(q, dst + (long long)pm * RECON * sizeof(typename P::store_t) * ns_d, ns_d, i);
  if (RECON != 18 && bad) {
    unsigned f = 0;
    // rows orthonormal, row2 = conj(row0 x row1)  <=>  U in SU(3)
    double defect = 0;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = a; b < 2; ++b) {
        double re = 0, im = 0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          re += u[6 * a + 2 * k] * u[6 * b + 2 * k] + u[6 * a + 2 * k + 1] * u[6 * b + 2 * k + 1];
          im += u[6 * a + 2 * k + 1] * u[6 * b + 2 * k] - u[6 * a + 2 * k] * u[6 * b + 2 * k + 1];
        }
        defect = fmax(defect, fmax(fabs(re - (a == b ? 1.0 : 0.0)), fabs(im)));
      }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const int j = (c + 1) % 3, k = (c + 2) % 3;
      const double re = u[2 * j] * u[6 + 2 * k] - u[2 * j + 1] * u[6 + 2 * k + 1] - u[2 * k] * u[6 + 2 * j] + u[2 * k + 1] * u[6 + 2 * j + 1];
      const double im = u[2 * j] * u[6 + 2 * k + 1] + u[2 * j + 1] * u[6 + 2 * k] - u[2 * k] * u[6 + 2 * j + 1] - u[2 * k + 1] * u[6 + 2 * j];
      defect = fmax(defect, fmax(fabs(re - u[12 + 2 * c]), fabs(-im - u[12 + 2 * c + 1])));
    }
    if (!(defect <= 1e-9)) f |= 1u;
    if (RECON == 8) {
      double n = 0;      // N as the Dslash kernels will see it (stored precision)
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const double x = P::HALF ? (double)((int)(unsigned short)q[k] - 32768) : (double)q[k];
        n += x * x;
      }
      if (!(n > (P::HALF ? 0.5 : (sizeof(typename P::real) == 8 ? 1e-290 : 1e-36)))) f |= 2u;
    }
    if (f) atomicOr(bad, f);
  }
}

template <class P>
static cudaError_t convert_gauge_p(int recon, char* dst, const double* g64, const BlockMap& bm, int blocked, unsigned* bad, cudaStream_t s) {
  dim3 grid((unsigned)(((blocked ? bm.blk.ns : bm.nat.ns) + 127) / 128), 8), block(128);
  switch (recon) {
    case 18: convert_gauge_kernel<P, 18><<<grid, block, 0, s>>>(dst, g64, bm, blocked, bad); break;
    case 12: convert_gauge_kernel<P, 12><<<grid, block, 0, s>>>(dst, g64, bm, blocked, bad); break;
    case 8:  convert_gauge_kernel<P, 8><<<grid, block, 0, s>>>(dst, g64, bm, blocked, bad); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_convert_gauge(int prec, int recon, char* dst, const double* g64, const BlockMap& bm, int blocked, cudaStream_t s, unsigned* bad) {
  switch (prec) {
    case 0: return convert_gauge_p<PrecD>(recon, dst, g64, bm, blocked, bad, s);
    case 1: return convert_gauge_p<PrecS>(recon, dst, g64, bm, blocked, bad, s);
    case 2: return convert_gauge_p<PrecH>(recon, dst, g64, bm, blocked, bad, s);
  }
  return cudaErrorInvalidValue;
}

// canonical psi[t][z][y][x][4][3] (complex128, or complex64 for the single-precision host entry point) <-> packed
// parity field of precision P
template <class P, typename C>
__global__ void pack_spinor_kernel(char* packed, C* canonical, const Geom g, int parity, int unpack, long long i0, long long i1) {
  const long long i = i0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= i1) return;
  int c[4];
  cb_to_coords(g, (int)i, parity, c);
  const long long site = c[0] + (long long)g.X[0] * (c[1] + (long long)g.X[1] * (c[2] + (long long)g.X[2] * c[3]));
  C* p = canonical + site * 24;
  typename P::real v[24];
  if (!unpack) {
#pragma unroll
    for (int k = 0; k < 24; ++k) v[k] = (typename P::real)p[k];
    store_site<P, 24>(v, packed, g.ns, i);
  } else {
    load_site<P, 24>(v, packed, g.ns, i);
#pragma unroll
    for (int k = 0; k < 24; ++k) p[k] = (C)v[k];
  }
}

template <typename C>
static cudaError_t pack_spinor_c(int prec, char* packed, C* c, const Geom& nat, int parity, int unpack, cudaStream_t s, long long i0, long long i1) {
  dim3 grid((unsigned)((i1 - i0 + 127) / 128)), block(128);
  switch (prec) {
    case 0: pack_spinor_kernel<PrecD, C><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    case 1: pack_spinor_kernel<PrecS, C><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    case 2: pack_spinor_kernel<PrecH, C><<<grid, block, 0, s>>>(packed, c, nat, parity, unpack, i0, i1); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

cudaError_t run_pack_spinor(int prec, char* packed, const double* canonical, const Geom& nat, int parity, int unpack, cudaStream_t s,
                            long long i0, long long i1, int canonical_single) {
  if (i1 < 0) i1 = nat.ns;
  if (canonical_single) return pack_spinor_c<float>(prec, packed, reinterpret_cast<float*>(const_cast<double*>(canonical)), nat, parity, unpack, s, i0, i1);
  return pack_spinor_c<double>(prec, packed, const_cast<double*>(canonical), nat, parity, unpack, s, i0, i1);
}

}  // namespace lq
