// ipls_r32.cuh -- register-blocked projection + IPLS kernel for R = 32 (placeholder: not built yet).
#pragma once
#include "common.cuh"

namespace linmin {

inline bool ipls_r32_supported(int /*L*/) { return false; }
inline cudaError_t launch_ipls_r32(const LibView &, const SolveParams &, int, cudaStream_t) {
    return cudaErrorNotSupported;
}

}  // namespace linmin
