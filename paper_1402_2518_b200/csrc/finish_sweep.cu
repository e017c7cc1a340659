// finish_sweep.cu -- translation unit of finish_sweep_kernel: compiled on its own so that its register
// budget (12 warps per SM = 3 per scheduler, up to 168 registers) does not bind the other kernels of the library.
#include <algorithm>

#include "finish_sweep.cuh"

namespace linmin {

cudaError_t launch_finish_sweep_tu(const LibView &lv, const SolveParams &prm, int sm_count,
                                   unsigned int *counter, unsigned int *overflow, const unsigned int *list,
                                   unsigned int *defer, cudaStream_t stream) {
    return launch_finish_sweep(lv, prm, sm_count, counter, overflow, list, defer, stream);
}

}  // namespace linmin
