// dslash_fp32.cu -- instantiates the Dslash kernels of dslash.cuh for storage precision PrecS.
#include "dslash_inst.cuh"
namespace lq {
template cudaError_t launch_dslash<PrecS>(const DslashArgs&, int, int, cudaStream_t);
}
