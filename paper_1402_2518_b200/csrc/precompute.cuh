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

// one warp per channel l: c[l] = mean_r A[l][r] (fp64), Ac[l][r] = fl32(A[l][r] - c[l]); center == 0 (pos option):
// c = 0, Ac = A.  flags[0] |= 1 when the caller's library Araw (L x Rraw) holds a non-finite value.
__global__ void center_library_kernel(const float *__restrict__ A, const float *__restrict__ Araw, int L, int R, int Rraw,
                                      int center, float *__restrict__ Ac, float *__restrict__ c, int *__restrict__ flags) {
    int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int lane = threadIdx.x & 31;
    if (warp >= L) return;
    const float *row = A + (size_t)warp * R;
    double s = 0.0;
    bool bad = false;
    for (int r = lane; r < R; r += 32) s += (double)row[r];
    for (int r = lane; r < Rraw; r += 32) bad |= !isfinite(Araw[(size_t)warp * Rraw + r]);
    s = warp_sum(s);
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(flags, 1);
    double mean = center ? s / (double)R : 0.0;
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

// Start-point data of IPLS (the "factor data" of north_star's precompute step): Gi = (Gc + 1e-4 gdmax I)^-1, its
// row sums Giq, and gdmax = max_i Gc[i][i] -- on the device, so that the library precompute has no host round
// trip.  ONE CTA; W is an R x R fp64 workspace in global memory (512 KB at R = 256: more than shared memory
// holds).  The regularised matrix is symmetric positive definite with a condition number <= 1e4 R, so the in-place
// Gauss-Jordan inversion needs no pivoting in fp64.  Step j: the pivot row and column go to shared memory, every
// other entry is updated from them.  scal[0] = gdmax (1 when every G_ii is 0: all endmembers identical, any point
// of the simplex is optimal), scal[1] = sum of Giq, scal[2] = t (below).
//
// The finish solves its equality-constrained sub-problems through the fp64 Gram block of the support.  A_F'A_F is
// singular as soon as the members are LINEARLY dependent (an all-zero "dark" endmember, or the slack column of the
// sum-lower-than-one option), although the sub-problem only needs them AFFINELY independent.  Because 1'a = 1
// (eq. 4), a'(G + t 11')a = a'Ga + t on the feasible set: with G64 <- A'A + t 11', t = max_i G_ii, the
// minimiser, the multipliers (taken from the data-space residual) and the projected inverse H = K - K11'K/(1'K1)
// are unchanged, and the block is non-singular exactly when the sub-problem is well posed.  `shift` = 0 skips it.
__global__ void __launch_bounds__(1024, 1)
start_data_kernel(const float *__restrict__ Gc, int R, double *__restrict__ W, float *__restrict__ Gi,
                  float *__restrict__ Giq, float *__restrict__ scal, double *__restrict__ G64, int shift) {
    __shared__ double prow[LINMIN_MAX_R], pcol[LINMIN_MAX_R];
    __shared__ float red[32];
    const int tid = threadIdx.x, nt = blockDim.x;
    float gd = 0.0f;
    for (int i = tid; i < R; i += nt) gd = fmaxf(gd, Gc[(size_t)i * R + i]);
    gd = warp_max(gd);
    if ((tid & 31) == 0) red[tid >> 5] = gd;
    __syncthreads();
    gd = 0.0f;
    for (int w = 0; w < (nt >> 5); ++w) gd = fmaxf(gd, red[w]);
    if (!(gd > 0.0f)) gd = 1.0f;
    const double delta = 1e-4 * (double)gd;
    for (int e = tid; e < R * R; e += nt) {
        const int i = e / R, j = e - i * R;
        // symmetrised read: Gc is symmetric up to the order of its fp64 sums
        W[e] = 0.5 * ((double)Gc[e] + (double)Gc[(size_t)j * R + i]) + (i == j ? delta : 0.0);
    }
    __syncthreads();
    for (int j = 0; j < R; ++j) {
        for (int i = tid; i < R; i += nt) { prow[i] = W[(size_t)j * R + i]; pcol[i] = W[(size_t)i * R + j]; }
        __syncthreads();
        const double d = prow[j];
        const double pv = 1.0 / ((d > 0.0) ? d : delta);
        for (int e = tid; e < R * R; e += nt) {
            const int i = e / R, c = e - i * R;
            double v;
            if (i == j) v = (c == j) ? pv : prow[c] * pv;
            else if (c == j) v = -pcol[i] * pv;
            else v = W[e] - pcol[i] * pv * prow[c];
            W[e] = v;
        }
        __syncthreads();
    }
    // symmetrise, round once to fp32, row sums in fp64
    for (int i = tid; i < R; i += nt) {
        double q = 0.0;
        for (int j = 0; j < R; ++j) {
            const double v = 0.5 * (W[(size_t)i * R + j] + W[(size_t)j * R + i]);
            Gi[(size_t)i * R + j] = (float)v;
            q += v;
        }
        Giq[i] = (float)q;
        prow[i] = (double)(float)q;
    }
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int i = 0; i < R; ++i) s += prow[i];
        scal[0] = gd;
        scal[1] = (float)s;
    }
    // ---- G64 <- A'A + t 11'
    __syncthreads();
    for (int i = tid; i < R; i += nt) pcol[i] = G64[(size_t)i * R + i];
    __syncthreads();
    double tsh = 0.0;
    for (int i = 0; i < R; ++i) tsh = fmax(tsh, pcol[i]);
    if (!shift) tsh = 0.0;
    __syncthreads();
    for (int e = tid; e < R * R; e += nt) G64[e] += tsh;
    if (tid == 0) scal[2] = (float)tsh;
}

// One-shot calls do not wait for the library check: when the library turned out non-finite (flag bit 0) or the noise
// covariance not positive definite (bit 1), every output of the call is overwritten with NaN and every info word with
// LINMIN_INFO_LIBRARY_NONFINITE and / or LINMIN_INFO_COVARIANCE (include/linmin.h).
__global__ void poison_outputs_kernel(const int *__restrict__ flags, int64_t N, int R, float *__restrict__ coeffs,
                                      float *__restrict__ csig, float *__restrict__ resid, int32_t *__restrict__ info) {
    const int f = flags[0];
    if (!f) return;
    const int32_t word = ((f & 1) ? LINMIN_INFO_LIBRARY_NONFINITE : 0) | ((f & 2) ? LINMIN_INFO_COVARIANCE : 0);
    const float qnan = __int_as_float(0x7fc00000);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < N * R; e += stride) {
        coeffs[e] = qnan;
        if (csig) csig[e] = qnan;
    }
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < N; p += stride) {
        if (resid) resid[p] = qnan;
        if (info) info[p] = word;
    }
}

}  // namespace linmin
