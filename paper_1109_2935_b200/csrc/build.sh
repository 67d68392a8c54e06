#!/bin/sh
# Builds liblqcd_b200.so in-tree for sm_100a (one nvcc per translation unit, in parallel).
set -e
cd "$(dirname "$0")"
OUT=${LQ_OUT:-../liblqcd_b200.so}
BUILD=${LQ_BUILD_DIR:-build}
# LQ_EXTRA_FLAGS: e.g. -DLQ_BOUNDS_CHECK for the index-checked debug build (remove build/ first)
FLAGS="-gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -std=c++17 -Xcompiler -fPIC --expt-relaxed-constexpr $LQ_EXTRA_FLAGS"
mkdir -p $BUILD
pids=""
for f in dslash_fp64 dslash_fp32 dslash_half dslash_mrhs_fp64 dslash_mrhs_fp32 dslash_mrhs_half staggered blas clover pack api solver host_api noalloc; do
  if [ ! -f $BUILD/$f.o ] || [ $f.cu -nt $BUILD/$f.o ] || [ -n "$(find . -maxdepth 1 \( -name '*.cuh' -o -name '*.h' \) -newer $BUILD/$f.o)" ] || [ ../../include/lqcd.h -nt $BUILD/$f.o ]; then
    nvcc $FLAGS -c $f.cu -o $BUILD/$f.o &
    pids="$pids $!"
  fi
done
for p in $pids; do wait $p; done
nvcc -gencode arch=compute_100a,code=sm_100a -shared -o $OUT $BUILD/*.o -lcudart
echo "built $OUT"
