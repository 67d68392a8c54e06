// dslash_fp64.cu -- instantiates the Dslash kernels of dslash.cuh for storage precision PrecD.
#include "dslash_inst.cuh"
namespace lq {
template cudaError_t launch_dslash<PrecD>(const DslashArgs&, int, int, cudaStream_t);
}
