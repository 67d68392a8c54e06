// dslash_mrhs_half.cu -- instantiates the multi-right-hand-side Dslash kernels for storage precision PrecH.
#include "dslash_mrhs_inst.cuh"
namespace lq {
template cudaError_t launch_dslash_mrhs<PrecH>(const DslashArgs&, int, int, int, cudaStream_t);
}
