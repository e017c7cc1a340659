// common.cuh -- shared declarations of the LinMin CUDA path (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/linmin.h"

// an endmember belongs to the initial support of the finish when its IPLS coefficient exceeds this
#define LINMIN_SUPPORT_THRESHOLD 1e-4f
// ... and IPLS hands over a_i = 0 where the primal-dual indicator says "inactive": a_i sc <= kappa lambda_i
// (sc = the pixel's gradient scale).  At the stopping point a_i lambda_i ~ mu for every i, so a_i / lambda_i
// separates the two classes by orders of magnitude where a_i alone does not; kappa = 30 halves the support
// repairs of the finish against the plain threshold (numpy model of the iteration on config 4).
#define LINMIN_TAPIA_KAPPA 30.0f

namespace linmin {

// Device-side view of the once-per-library precompute.
struct LibView {
    int L, R;
    const float *A;     // L x R, caller's library (copied into the handle)
    const float *At;    // R x L, the same by endmember (At[r][l] = A[l][r])
    const float *Ac;    // L x R, centred: Ac[l][r] = A[l][r] - c[l], c[l] = mean_r A[l][r]
    const float *c;     // L
    const float *Gc;    // R x R fp32, Gc = Ac' Ac accumulated in fp64 (drives IPLS)
    const double *G64;  // R x R fp64, A'A + t 11' (uncentred, exact data; t: precompute.cuh; drives the finish)
    const float *scal;  // device scalars of the precompute: [0] gdmax = max_i Gc[i][i] (1 if that is 0), [1] sum of Giq
    const int *flags;   // device word: bit 0 = the library holds a non-finite value (every kernel then returns at once)
    int cons;           // 1: the coefficients sum to one (sto, and slo through its slack endmember); 0: positivity only
                        // (pos: no equality constraint, nu == 0, library not centred, G64 not shifted)
    const float *Gi;    // R x R fp32, (Gc + 1e-4 gdmax I)^-1 (start point of IPLS: regularised sum-constrained LS)
    const float *Giq;   // R, row sums of Gi
    const float *Gpad;  // R > 64 only: Gc zero-padded to (32 ceil(R / 32))^2, identity on the padded diagonal (ipls_c256.cuh)
};

struct SolveParams {
    const float *Y;
    const float *sigma;
    int64_t N;
    int64_t ldY;
    int64_t sigma_stride;   // 0 shared, else per pixel
    int has_sigma;
    int max_iter;
    float gap_tol, feas_tol;
    float *coeffs;          // N x R (IPLS iterate in, final coefficients out)
    float *coeff_sigma;     // N x R or NULL
    float *resid;           // N or NULL
    int32_t *info;          // N or NULL
};

// column-major packed lower triangle of an n x n matrix: (i, j), i >= j
__host__ __device__ __forceinline__ int cm(int n, int i, int j) { return j * n - (j * (j - 1)) / 2 + (i - j); }

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_min(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// ---- reductions over a group of W consecutive lanes (W = 4 or 8 lanes cooperate on one pixel)
template <int W> __device__ __forceinline__ float group_sum(float v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
template <int W> __device__ __forceinline__ double group_sum(double v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
template <int W> __device__ __forceinline__ float group_min(float v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
template <int W> __device__ __forceinline__ double group_min(double v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
template <int W> __device__ __forceinline__ float group_max(float v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
template <int W> __device__ __forceinline__ unsigned group_or(unsigned v) {
#pragma unroll
    for (int o = 1; o < W; o <<= 1) v |= __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// ---- packed fp32 arithmetic (sm_100 FFMA2 / FMUL2: the FP32 peak of this part is an FFMA2 peak)
__device__ __forceinline__ unsigned long long pk2(float2 v) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(v.x), "f"(v.y));
    return r;
}
__device__ __forceinline__ float2 upk2(unsigned long long v) {
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
// a * b + c on both halves; the scalar form broadcasts a
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)), "l"(pk2(c)));
    return upk2(d);
}
__device__ __forceinline__ float2 fma2(float a, float2 b, float2 c) { return fma2(make_float2(a, a), b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(pk2(a)), "l"(pk2(b)));
    return upk2(d);
}

}  // namespace linmin
