// precompute.cuh -- once-per-library kernels ("S.S^T").
//
// Because every pixel's coefficients sum to one (eq. 4), y - A a = (y - c) - (A - c 1') a
// for ANY channel vector c.  Taking c = row mean of A removes the component common to all endmembers
// (the flat-dominated continuum), which shrinks the entries of the Gram matrix by 1-2 orders of
// magnitude and with them the absolute fp32 rounding error of the interior-point iteration
// (DESIGN.md "centring").  The finish works on the exact, uncentred data in fp64.
#pragma once
#include "common.cuh"

namespace linmin {

// At[r][l] = A[l][r]: the library by endmember, for the kernels that walk one endmember over the channels
// (the lanes of a warp then read consecutive addresses).  One thread per element, reads coalesced.
__global__ void transpose_library_kernel(const float *__restrict__ A, int L, int R, float *__restrict__ At) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (size_t)L * R) return;
    const int l = (int)(e / R), r = (int)(e - (size_t)l * R);
    At[(size_t)r * L + l] = A[e];
}

// one warp per channel l: c[l] = mean_r A[l][r] (fp64), Ac[l][r] = fl32(A[l][r] - c[l]).
// flags[0] |= 1 when A holds a non-finite value.
__global__ void center_library_kernel(const float *__restrict__ A, int L, int R, float *__restrict__ Ac,
                                      float *__restrict__ c, int *__restrict__ flags) {
    int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (warp >= L) return;
    const float *row = A + (size_t)warp * R;
    double s = 0.0;
    bool bad = false;
    for (int r = lane; r < R; r += 32) {
        float v = row[r];
        bad |= !isfinite(v);
        s += (double)v;
    }
    s = warp_sum(s);
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(flags, 1);
    double mean = s / (double)R;
    for (int r = lane; r < R; r += 32) Ac[(size_t)warp * R + r] = (float)((double)row[r] - mean);
    if (lane == 0) c[warp] = (float)mean;
}

// one thread per (i, j): G64[i][j] = sum_l A[l][i] A[l][j]  (fp64; products of fp32 are exact in fp64),
// Gc[i][j] = fl32( sum_l Ac[l][i] Ac[l][j] ) accumulated in fp64.
__global__ void gram_kernel(const float *__restrict__ A, const float *__restrict__ Ac, int L, int R,
                            double *__restrict__ G64, float *__restrict__ Gc) {
    int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= R * R) return;
    int i = e / R, j = e - i * R;
    double s = 0.0, sc = 0.0;
    for (int l = 0; l < L; ++l) {
        s += (double)A[(size_t)l * R + i] * (double)A[(size_t)l * R + j];
        sc += (double)Ac[(size_t)l * R + i] * (double)Ac[(size_t)l * R + j];
    }
    G64[e] = s;
    Gc[e] = (float)sc;
}

}  // namespace linmin
