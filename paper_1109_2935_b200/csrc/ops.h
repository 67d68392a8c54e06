// ops.h -- internal host-side operator layer shared by api.cu and solver.cu.
#pragma once
#include "host.h"

namespace lq {

int fail(lqcd_ctx* c, int code, const char* what, cudaError_t e = cudaSuccess);
int dev_alloc(lqcd_ctx* c, void** p, size_t bytes);
// workspace of a call: taken from the context's cache when a buffer of that size is there, else allocated;
// ws_put hands it back (its pending work on stream `s` is ordered before any reuse on the same stream, and
// waited for before a reuse on another stream)
int ws_get(lqcd_ctx* c, void** p, size_t bytes, cudaStream_t s);
void ws_put(lqcd_ctx* c, void* p, size_t bytes, cudaStream_t s);
int get_gauge(lqcd_ctx* c, int prec, int recon, bool blocked, const char** out, cudaStream_t s);
int get_clover(lqcd_ctx* c, int prec, double kappa, bool blocked, const char** A, const char** Ainv, cudaStream_t s);
int get_tmp(lqcd_ctx* c, int prec, bool blocked, char** out);
int set_blocks(lqcd_ctx* c, const int* blk, int cmaj = 0, int overlap = 0);   // cmaj: colour-major box order (multiplicative Schwarz); overlap: host.h
int op_dslash(lqcd_ctx* c, char* out, const char* in, const char* y, int parity_out, int dagger, int prec, int recon,
              int epi, double a, double kappa, bool blocked, cudaStream_t s, int cb0 = 0, int cb1 = -1, int fin = 0,
              const char* q = nullptr, int box0 = 0, int nbox = 0);
int op_matpc(lqcd_ctx* c, char* out, const char* in, int parity, int dagger, double kappa, int prec, int recon,
             bool blocked, bool dots, cudaStream_t s, int sym = 0, int fin = 0, const char* q = nullptr,
             int box0 = 0, int nbox = 0);

// multi-right-hand-side forms (dslash_mrhs.cuh): in / out / y hold nrhs packed fields back to back
int op_dslash_mrhs(lqcd_ctx* c, char* out, const char* in, const char* y, int nrhs, int parity_out, int dagger, int prec,
                   int recon, int epi, double a, double kappa, cudaStream_t s);
int op_matpc_mrhs(lqcd_ctx* c, char* out, const char* in, int nrhs, int parity, int dagger, double kappa, int prec, int recon,
                  cudaStream_t s);

template <class P> cudaError_t launch_dslash(const DslashArgs& a, int recon, int epi, cudaStream_t s);
template <class P> cudaError_t launch_dslash_mrhs(const DslashArgs& a, int nrhs, int recon, int epi, cudaStream_t s);

}  // namespace lq
