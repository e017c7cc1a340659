// thresholds_static.cu -- linmin_detection_thresholds_static: the eq. 8 thresholds for callers
// that cannot let this library allocate device memory.
//
// Who that is: an application that handed the whole GPU to its own arena at start-up (a cudaMalloc or a pool
// allocation made here would fail, or eat into memory the application has already planned), and a
// latency-bound loop (an instrument pipeline classifying frames as they arrive) that cannot afford the
// device-wide synchronisation and the unbounded duration an allocation may cost.  linmin_detection_thresholds takes
// its per-block partial sums from the library's staging pool; this variant keeps them in a fixed array that is part
// of the library image, so it calls neither cudaMalloc / cudaFree nor any pool or other allocating routine.
//
// The price, all of it stated in include/linmin.h too:
//   * the array is sized for R <= LINMIN_STATIC_MAX_R endmembers and LINMIN_STATIC_MAX_BLOCKS thread blocks
//     (384 KiB); every GPU on which the library image gets loaded holds those 384 KiB until the process exits;
//   * there is ONE array per device: calls that overlap on a device (two streams, two host threads) race on it;
//   * the first call on each device looks the array's device address up and should come before any stream capture.
//
// Own translation unit: nothing of the existing paths is touched.  The two kernels repeat the arithmetic of
// threshold_partial_kernel / threshold_final_kernel (detect.cuh); the launch differs (at most 128 blocks), so
// the fp64 partial sums are added in another order than on the pooled path: the float32 thresholds agree to
// rounding, not always bit for bit.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <mutex>

#include "../../include/linmin.h"

// [block][endmember][6]: count, sum, sum of squares of the detections on present pixels, then on absent pixels.
// In HOST code this name is only a handle for the symbol -- not an address a kernel could use; host code gets the
// address from cudaGetSymbolAddress (scratch_for_current_device below).
static __device__ __align__(256) double g_threshold_scratch[(size_t)LINMIN_STATIC_MAX_BLOCKS * LINMIN_STATIC_MAX_R * 6];

namespace {

constexpr int kMaxR = LINMIN_STATIC_MAX_R;
constexpr int kMaxBlocks = LINMIN_STATIC_MAX_BLOCKS;
constexpr int kMaxDevices = 64;

std::mutex g_setup_mu;
double *g_scratch_addr[kMaxDevices] = {};     // device address of g_threshold_scratch, per device ordinal

// Once per device, with that device current: the address of this device's copy of the array.
cudaError_t scratch_for_current_device(double **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_setup_mu);
    if (!g_scratch_addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_threshold_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

// Stage 1 (same sums as threshold_partial_kernel): a thread stays on one endmember because blockDim.x is a multiple
// of R; block b leaves its six fp64 sums per endmember in part[b][i][0..5].  Every block of the launch writes all of
// its R x 6 slots, and stage 2 reads exactly the slots of this launch: whatever an earlier call left in the array is
// never read, so nothing has to be cleared between calls.
__global__ void threshold_partial_static_kernel(const float *__restrict__ coeffs, const unsigned char *__restrict__ present,
                                                int64_t N, int R, double *__restrict__ part) {
    extern __shared__ double sh[];          // [blockDim.x][6]
    const int64_t total = N * R;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const float v = coeffs[e];
        if (v > 0.0f) {
            const int o = present[e] ? 0 : 3;
            acc[o] += 1.0; acc[o + 1] += (double)v; acc[o + 2] += (double)v * (double)v;
        }
    }
    for (int k = 0; k < 6; ++k) sh[threadIdx.x * 6 + k] = acc[k];
    __syncthreads();
    if (threadIdx.x < R) {
        double s[6] = {0, 0, 0, 0, 0, 0};
        for (int t = threadIdx.x; t < blockDim.x; t += R)
            for (int k = 0; k < 6; ++k) s[k] += sh[t * 6 + k];
        for (int k = 0; k < 6; ++k) part[((size_t)blockIdx.x * R + threadIdx.x) * 6 + k] = s[k];
    }
}

// Stage 2: blocks added in index order, then eq. 8: C^i = 1/2 (mean(A+) - 2 std(A+) + mean(A-) + 6 std(A-)),
// population std, an empty class contributing 0 (reading R19 of DESIGN.md).
__global__ void threshold_final_static_kernel(const double *__restrict__ part, int nblocks, int R, float *__restrict__ thr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= R) return;
    double s[6] = {0, 0, 0, 0, 0, 0};
    for (int b = 0; b < nblocks; ++b)
        for (int k = 0; k < 6; ++k) s[k] += part[((size_t)b * R + i) * 6 + k];
    double mp = 0, sp = 0, mf = 0, sf = 0;
    if (s[0] > 0) { mp = s[1] / s[0]; sp = sqrt(fmax(s[2] / s[0] - mp * mp, 0.0)); }
    if (s[3] > 0) { mf = s[4] / s[3]; sf = sqrt(fmax(s[5] / s[3] - mf * mf, 0.0)); }
    thr[i] = (float)(0.5 * (mp - 2.0 * sp + mf + 6.0 * sf));
}

}  // namespace

extern "C" int linmin_detection_thresholds_static(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                                  float *thresholds_out, void *stream) {
    if (!coeffs || !present || !thresholds_out || N < 0 || R < 1) return LINMIN_ERR_INVALID_ARGUMENT;
    if (R > kMaxR) return LINMIN_ERR_STATIC_SCRATCH;      // the fixed array has no room for more endmembers
    cudaStream_t st = (cudaStream_t)stream;
    double *part = nullptr;
    if (scratch_for_current_device(&part) != cudaSuccess) { (void)cudaGetLastError(); return LINMIN_ERR_CUDA; }
    const int block = R * std::max(1, 256 / R);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N * R + block - 1) / block, kMaxBlocks));
    threshold_partial_static_kernel<<<grid, block, (size_t)block * 6 * sizeof(double), st>>>(coeffs, present, N, R, part);
    if (cudaGetLastError() != cudaSuccess) return LINMIN_ERR_CUDA;
    threshold_final_static_kernel<<<(R + 63) / 64, 64, 0, st>>>(part, grid, R, thresholds_out);
    if (cudaGetLastError() != cudaSuccess) return LINMIN_ERR_CUDA;
    return LINMIN_OK;
}
