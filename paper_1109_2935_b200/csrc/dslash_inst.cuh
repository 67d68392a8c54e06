// dslash_inst.cuh -- host dispatch over (recon, epilogue) for one precision; included by
// dslash_fp64.cu / dslash_fp32.cu / dslash_half.cu so the three precisions compile in parallel.
#pragma once
#include "dslash.cuh"

namespace lq {

template <class P, int RECON>
static cudaError_t launch_dslash_r(const DslashArgs& a, int epi, cudaStream_t s) {
  dim3 grid((a.g.vh + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK, a.g.nb);
  dim3 block(LQ_DSLASH_BLOCK);
  switch (epi) {
    case EPI_NONE:            dslash_kernel<P, RECON, false, false, false, false><<<grid, block, 0, s>>>(a); break;
    case EPI_CLOVOUT:         dslash_kernel<P, RECON, false, false, true,  false><<<grid, block, 0, s>>>(a); break;
    case EPI_CLOVX_XPAY:      dslash_kernel<P, RECON, true,  true,  false, false><<<grid, block, 0, s>>>(a); break;
    case EPI_XPAY:            dslash_kernel<P, RECON, true,  false, false, false><<<grid, block, 0, s>>>(a); break;
    case EPI_XPAY_CLOVOUT:    dslash_kernel<P, RECON, true,  false, true,  false><<<grid, block, 0, s>>>(a); break;
    case EPI_CLOVX_XPAY_DOTS: dslash_kernel<P, RECON, true,  true,  false, true ><<<grid, block, 0, s>>>(a); break;
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

template <class P>
cudaError_t launch_dslash(const DslashArgs& a, int recon, int epi, cudaStream_t s) {
  switch (recon) {
    case 18: return launch_dslash_r<P, 18>(a, epi, s);
    case 12: return launch_dslash_r<P, 12>(a, epi, s);
    case 8:  return launch_dslash_r<P, 8>(a, epi, s);
  }
  return cudaErrorInvalidValue;
}

}  // namespace lq
