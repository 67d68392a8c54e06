// dslash_half.cu -- instantiates the Dslash kernels of dslash.cuh for storage precision PrecH.
#include "dslash_inst.cuh"
namespace lq {
template cudaError_t launch_dslash<PrecH>(const DslashArgs&, int, int, cudaStream_t);
}
