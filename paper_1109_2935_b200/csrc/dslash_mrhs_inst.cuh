// dslash_mrhs_inst.cuh -- host dispatch over (recon, epilogue) of the multi-right-hand-side
// Dslash for one precision; included by dslash_mrhs_{fp64,fp32,half}.cu.
#pragma once
#include "dslash_mrhs.cuh"

namespace lq {

template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int NR, int DAG>
static cudaError_t launch_mrhs_nr(const DslashArgs& a, int nrhs, cudaStream_t s) {
#ifndef LQ_MRHS_PIPE
#define LQ_MRHS_PIPE 3   /* measured: 2 -> 200, 3 -> 195, 4 -> 214 us per source for the fp32/r12 Mhat at 32^3x64 */
#endif
  constexpr int NST = P::HALF ? 4 : LQ_MRHS_PIPE;   // depth of the spinor cp.async ring
  constexpr int SMEM = LinkTile<typename P::real>::BYTES + NST * SpinStage<P, NR>::BYTES;
  dim3 grid((a.range.cb1 - a.range.cb0 + 31) / 32, a.g.nb, (nrhs + NR - 1) / NR);
  auto kern = dslash_mrhs_kernel<P, RECON, XPAY, CLOVX, CLOVOUT, NST, NR, DAG>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
  if (e != cudaSuccess) return e;
  cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  kern<<<grid, dim3(32 * NR), SMEM, s>>>(a);
  return cudaGetLastError();
}

template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT>
static cudaError_t launch_mrhs_one(const DslashArgs& a, int nrhs, cudaStream_t s) {
  if constexpr (P::HALF) {
    if (a.dagger & 1) return launch_mrhs_nr<P, RECON, XPAY, CLOVX, CLOVOUT, 4, 1>(a, nrhs, s);
    return launch_mrhs_nr<P, RECON, XPAY, CLOVX, CLOVOUT, 4, 0>(a, nrhs, s);
  } else {
    return launch_mrhs_nr<P, RECON, XPAY, CLOVX, CLOVOUT, 4, -1>(a, nrhs, s);
  }
}

template <class P, int RECON>
static cudaError_t launch_mrhs_r(const DslashArgs& a, int nrhs, int epi, cudaStream_t s) {
  switch (epi) {
    case EPI_NONE:         return launch_mrhs_one<P, RECON, false, false, false>(a, nrhs, s);
    case EPI_CLOVOUT:      return launch_mrhs_one<P, RECON, false, false, true>(a, nrhs, s);
    case EPI_CLOVX_XPAY:   return launch_mrhs_one<P, RECON, true, true, false>(a, nrhs, s);
    case EPI_XPAY:         return launch_mrhs_one<P, RECON, true, false, false>(a, nrhs, s);
    case EPI_XPAY_CLOVOUT: return launch_mrhs_one<P, RECON, true, false, true>(a, nrhs, s);
  }
  return cudaErrorInvalidValue;
}

template <class P>
cudaError_t launch_dslash_mrhs(const DslashArgs& a, int nrhs, int recon, int epi, cudaStream_t s) {
  switch (recon) {
    case 18: return launch_mrhs_r<P, 18>(a, nrhs, epi, s);
    case 12: return launch_mrhs_r<P, 12>(a, nrhs, epi, s);
    case 8:  return launch_mrhs_r<P, 8>(a, nrhs, epi, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace lq
