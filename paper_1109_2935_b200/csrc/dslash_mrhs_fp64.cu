// dslash_mrhs_fp64.cu -- instantiates the multi-right-hand-side Dslash kernels for storage precision PrecD.
#include "dslash_mrhs_inst.cuh"
namespace lq {
template cudaError_t launch_dslash_mrhs<PrecD>(const DslashArgs&, int, int, int, cudaStream_t);
}
