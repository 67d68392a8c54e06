// dslash_inst.cuh -- host dispatch over (recon, epilogue) for one precision; included by
// dslash_fp64.cu / dslash_fp32.cu / dslash_half.cu so the three precisions compile in parallel.
#pragma once
#include <cstdlib>
#include <mutex>
#include "dslash.cuh"
#include "dslash_tile.cuh"

namespace lq {

// fp64: the ring pays for the plain hopping term (32^3x64 r18 272 -> 246 us, r12 222 -> 212, r8 323 -> 282) but
// not with a clover epilogue (Mhat r18 696 -> 730 us), which keeps loading straight into registers
#ifndef LQ_PIPE_FP64
#define LQ_PIPE_FP64 2
#endif
#ifndef LQ_PIPE_FP32
#define LQ_PIPE_FP32 2
#endif
#ifndef LQ_PIPE_HALF
#define LQ_PIPE_HALF 4
#endif

template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int DOTS, int DAG>
static void launch_dag(const DslashArgs& a, dim3 grid, dim3 block, cudaStream_t s) {
  constexpr int NST = sizeof(typename P::real) == 8 ? ((CLOVX || CLOVOUT) ? 0 : LQ_PIPE_FP64) : (P::HALF ? LQ_PIPE_HALF : LQ_PIPE_FP32);
  constexpr int SMEM = NST * HopStage<P, RECON>::BYTES;
  auto kern = dslash_kernel<P, RECON, XPAY, CLOVX, CLOVOUT, DOTS, NST, DAG>;
  // function attributes are per device: set once per instantiation and device (std::call_once, so that two
  // contexts driven from two host threads cannot race on the flag)
  static std::once_flag configured_dev[64];
  int dev = 0;
  cudaGetDevice(&dev);
  std::call_once(configured_dev[dev & 63], [&] {
    if (NST > 0) {
      cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
      cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    } else {
      // no staging ring: ask for the largest L1.  Without a preference the SM keeps the carve-out of
      // the previous kernel, and after a ring kernel the fp64 clover variants lost 5 % (696 -> 730 us)
      cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxL1);
    }
  });
  kern<<<grid, block, SMEM, s>>>(a);
}

#ifndef LQ_TILE_PIPE
#define LQ_TILE_PIPE 4
#endif
// half precision, tile form (dslash_tile.cuh): T threads per CTA, ring of LQ_TILE_PIPE hops
template <int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int T, int DAG>
static void launch_tile(const DslashArgs& a, TileInfo& ti, cudaStream_t s) {
  constexpr int NST = LQ_TILE_PIPE;
  tile_planes<RECON>(a, ti);
  constexpr int SMEM = NST * TileStage<RECON, T>::BYTES + 2 * NST * 8;
  auto kern = dslash_tile_kernel<RECON, XPAY, CLOVX, CLOVOUT, T, NST, DAG>;
  static std::once_flag configured_dev[64];
  int dev = 0;
  cudaGetDevice(&dev);
  std::call_once(configured_dev[dev & 63], [&] {
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
    cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  });
  const int slice = a.g.Xh * a.g.X[1] * a.g.X[2];
  dim3 grid(a.g.Xh * a.g.X[1] / T, a.g.X[2], (a.range.cb1 - a.range.cb0) / slice), block(T);
  kern<<<grid, block, SMEM, s>>>(a, ti);
}

// LQCD_B200_NO_TILE=1 in the environment keeps every launch on dslash_kernel (A/B timing, the bit-identity test);
// read at every launch so that a test can switch it
static bool tile_enabled() {
  const char* e = getenv("LQCD_B200_NO_TILE");
  return !(e && e[0] == '1');
}

// half precision: the dagger flag selects one of two instantiations (dslash.cuh, hop_fixed)
template <class P, int RECON, bool XPAY, bool CLOVX, bool CLOVOUT, int DOTS>
static void launch_one(const DslashArgs& a, dim3 grid, dim3 block, cudaStream_t s) {
  // Tile form for the plain hopping term only.  Measured at 32^3x64, half r12 / r18: 71.0 -> 67.7 / 76.0 -> 71.6 us;
  // with a clover epilogue the tile form (2,770 SASS instructions, 44 KB: over the 32 KB instruction cache) is no
  // faster than dslash_kernel (Mhat 188.5 vs 189.6 us), so those variants are not instantiated.
  if constexpr (P::HALF && !DOTS && RECON != 8 && !XPAY && !CLOVX && !CLOVOUT) {
    TileInfo ti;
    if (tile_enabled()) {
      if (tile_ok<128>(a, ti)) {
        if (a.dagger & 1) launch_tile<RECON, XPAY, CLOVX, CLOVOUT, 128, 1>(a, ti, s);
        else launch_tile<RECON, XPAY, CLOVX, CLOVOUT, 128, 0>(a, ti, s);
        return;
      }
      if (tile_ok<96>(a, ti)) {
        if (a.dagger & 1) launch_tile<RECON, XPAY, CLOVX, CLOVOUT, 96, 1>(a, ti, s);
        else launch_tile<RECON, XPAY, CLOVX, CLOVOUT, 96, 0>(a, ti, s);
        return;
      }
    }
  }
  if constexpr (P::HALF) {
    if (a.dagger & 1) launch_dag<P, RECON, XPAY, CLOVX, CLOVOUT, DOTS, 1>(a, grid, block, s);
    else launch_dag<P, RECON, XPAY, CLOVX, CLOVOUT, DOTS, 0>(a, grid, block, s);
  } else {
    launch_dag<P, RECON, XPAY, CLOVX, CLOVOUT, DOTS, -1>(a, grid, block, s);
  }
}

template <class P, int RECON>
static cudaError_t launch_dslash_r(const DslashArgs& a, int epi, cudaStream_t s) {
  const bool whole = epi == EPI_CLOVX_XPAY_DOTS || epi == EPI_CLOVX_XPAY_YDOT || epi == EPI_CLOVX_XPAY_QDOT;   // no site range (dslash.cuh)
  const int nsite = whole ? a.g.vh : a.range.cb1 - a.range.cb0;
  dim3 grid((nsite + LQ_DSLASH_BLOCK - 1) / LQ_DSLASH_BLOCK, a.g.nb);   // g.nb = boxes of this launch (g.ns keeps the field stride)
  dim3 block(LQ_DSLASH_BLOCK);
  switch (epi) {
    case EPI_NONE:            launch_one<P, RECON, false, false, false, 0>(a, grid, block, s); break;
    case EPI_CLOVOUT:         launch_one<P, RECON, false, false, true, 0>(a, grid, block, s); break;
    case EPI_CLOVX_XPAY:      launch_one<P, RECON, true, true, false, 0>(a, grid, block, s); break;
    case EPI_XPAY:            launch_one<P, RECON, true, false, false, 0>(a, grid, block, s); break;
    case EPI_XPAY_CLOVOUT:    launch_one<P, RECON, true, false, true, 0>(a, grid, block, s); break;
    case EPI_CLOVX_XPAY_DOTS: launch_one<P, RECON, true, true, false, 1>(a, grid, block, s); break;
    case EPI_CLOVX_XPAY_YDOT: launch_one<P, RECON, true, true, false, 2>(a, grid, block, s); break;
    case EPI_CLOVX_XPAY_QDOT: launch_one<P, RECON, true, true, false, 3>(a, grid, block, s); break;
    case EPI_XPAY_CLOVD:      launch_one<P, RECON, true, true, true, 0>(a, grid, block, s); break;
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
