// dslash_mrhs_fp32.cu -- instantiates the multi-right-hand-side Dslash kernels for storage precision PrecS.
#include "dslash_mrhs_inst.cuh"
namespace lq {
template cudaError_t launch_dslash_mrhs<PrecS>(const DslashArgs&, int, int, int, cudaStream_t);
}
