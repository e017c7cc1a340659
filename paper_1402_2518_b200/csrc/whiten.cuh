// whiten.cuh -- the renormalised problem (sec. 2.3, eq. 5-6).
//
// One noise covariance C (L x L) for the whole image: "C^-1 = L.L^T ... X' = X.L and S' = S.L.  Thereby, the
// measurement uncertainty is handled by modifying the observation matrix X and the reference spectra S before the
// unmixing process."  Any F with F F^T = C^-1 gives the same criterion (eq. 6); this build takes F^T = W = Rc^-1 with
// C = Rc Rc^T (Cholesky of C itself: no explicit inverse of C), so y' = W y and A' = W A, W lower triangular.
//   once per library (fp64, one CTA each, on the stream):   C -> Rc -> W;   A' = W A (fp64 accumulate, rounded once)
//   per call:  Y' = Y W^T, a real GEMM [N x L].[L x L] -- register-blocked like the projection of start_r32.cuh
//              (a lane owns 4 pixels x 32 output channels, the rows of W^T broadcast from shared memory), or an
//              element-wise scaling when C is diagonal.
// The constrained problem is then solved on (A', Y') by the unweighted path; the coefficient uncertainties are the
// projected inverse Hessian H_w itself (unit noise in whitened space), the residual is the whitened RMS.
#pragma once
#include "common.cuh"

namespace linmin {

// Cd: L x L fp64 workspace.  kind 1: cov = per-channel noise std (L); kind 2: cov = L x L covariance (symmetrised).
// Lower Cholesky factor in place, then W = Rc^-1 (fp64 in Wd, fp32 in W; upper parts zero).  flags |= 2 when C is not
// positive definite or not finite.  ONE CTA.
__global__ void __launch_bounds__(1024, 1)
whitening_matrix_kernel(const float *__restrict__ cov, int kind, int L, double *__restrict__ Cd, double *__restrict__ Wd,
                        float *__restrict__ W, int *__restrict__ flags) {
    const int tid = threadIdx.x, nt = blockDim.x;
    __shared__ double colj[LINMIN_MAX_L];
    __shared__ int bad;
    if (tid == 0) bad = 0;
    for (int e = tid; e < L * L; e += nt) {
        const int i = e / L, j = e - i * L;
        double v;
        if (kind == 1) v = (i == j) ? (double)cov[i] * (double)cov[i] : 0.0;
        else v = 0.5 * ((double)cov[e] + (double)cov[(size_t)j * L + i]);
        Cd[e] = v;
    }
    __syncthreads();
    // right-looking Cholesky: column j is scaled, then the trailing lower triangle is updated
    for (int j = 0; j < L; ++j) {
        const double d = Cd[(size_t)j * L + j];
        if (!(d > 0.0) || !isfinite(d)) { if (tid == 0) bad = 1; }
        const double rd = (d > 0.0) ? 1.0 / sqrt(d) : 0.0;
        for (int i = j + tid; i < L; i += nt) colj[i] = Cd[(size_t)i * L + j] * rd;
        __syncthreads();
        for (int i = j + tid; i < L; i += nt) Cd[(size_t)i * L + j] = colj[i];
        const int n = L - 1 - j;
        for (int e = tid; e < n * n; e += nt) {
            const int a = e / n, b = e - a * n;
            if (b <= a) Cd[(size_t)(j + 1 + a) * L + (j + 1 + b)] -= colj[j + 1 + a] * colj[j + 1 + b];
        }
        __syncthreads();
    }
    // W = Rc^-1 by forward substitution of the unit vectors: one WARP per column, the column in registers (entry k
    // on lane k mod 32), the dot product of row i split over the lanes (coalesced reads of Rc's row) and summed by
    // shuffles -- L steps of L / 32 products per column instead of one thread's chain of L^2 / 2 dependent loads
    {
        const int lane = tid & 31, wid = tid >> 5, nw = nt >> 5;
        constexpr int M = LINMIN_MAX_L / 32;
        for (int c = wid; c < L; c += nw) {
            double x[M];
#pragma unroll
            for (int m = 0; m < M; ++m) x[m] = 0.0;
            for (int i = c; i < L; ++i) {
                const double *row = Cd + (size_t)i * L;
                double v = 0.0;
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    const int k = lane + 32 * m;
                    if (k < i) v += row[k] * x[m];          // (entries above the column's first row are still zero)
                }
                v = warp_sum(v);
                const double xi = (((i == c) ? 1.0 : 0.0) - v) / row[i];
#pragma unroll
                for (int m = 0; m < M; ++m)
                    if (lane + 32 * m == i) x[m] = xi;
            }
#pragma unroll
            for (int m = 0; m < M; ++m) {
                const int k = lane + 32 * m;
                if (k < L) Wd[(size_t)k * L + c] = x[m];
            }
        }
    }
    __syncthreads();
    for (int e = tid; e < L * L; e += nt) W[e] = (float)Wd[e];
    if (tid == 0 && bad) atomicOr(flags, 2);
}

// Aw[l][r] = fl32( sum_{m <= l} W[l][m] A[m][r] ), r < R; columns R .. Ri-1 (the slack endmember of slo) stay zero.
// A == NULL-safe for W: Wd == NULL means "no weighting" (plain copy with zero padding).
__global__ void whiten_library_kernel(const float *__restrict__ A, int L, int R, int Ri, const double *__restrict__ Wd,
                                      float *__restrict__ Aw) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= L * Ri) return;
    const int l = e / Ri, r = e - l * Ri;
    double s = 0.0;
    if (r < R) {
        if (Wd) { for (int m = 0; m <= l; ++m) s += Wd[(size_t)l * L + m] * (double)A[(size_t)m * R + r]; }
        else s = (double)A[(size_t)l * R + r];
    }
    Aw[e] = (float)s;
}

// Diagonal covariance: Y'[p][l] = Y[p][l] * W[l][l]
__global__ void whiten_spectra_diag_kernel(const float *__restrict__ Y, int64_t ldY, int64_t N, int L,
                                           const float *__restrict__ W, float *__restrict__ Yw) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < N * L; e += stride) {
        const int64_t p = e / L;
        const int l = (int)(e - p * L);
        Yw[e] = Y[p * ldY + l] * W[(size_t)l * L + l];
    }
}

namespace wh {
constexpr int WARPS = 8;
constexpr int TP = 128;       // pixels per warp tile (4 per lane)
constexpr int CH = 16;        // channels per staged chunk
constexpr int YST = 20;       // padded row stride of a staged chunk
constexpr int OC = 32;        // output channels per pass
}  // namespace wh

// Full covariance: Y' = Y W^T.  A warp takes a tile of 128 pixels and, pass by pass, 32 output channels o0 .. o0 + 31:
// Y'[p][o] = sum_{m <= o} W[o][m] Y[p][m].  The slab Wt[m][j] = W[o0 + j][m] sits in shared memory (one slab per
// CTA at a time: all warps of the CTA work on the same o0), the spectra are staged as in start_r32.cuh.
__global__ void __launch_bounds__(wh::WARPS * 32, 1)
whiten_spectra_kernel(const float *__restrict__ Y, int64_t ldY, int64_t N, int L, const float *__restrict__ W,
                      float *__restrict__ Yw) {
    using namespace wh;
    extern __shared__ __align__(16) float smem[];
    const int Lp = (L + CH - 1) / CH * CH;
    float *Wt = smem;                                         // [Lp][OC]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *ybuf = Wt + (size_t)Lp * OC + (size_t)warp * (2 * TP * YST);
    const bool vec_ok = ((L & 3) == 0) && ((ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(Y) & 15) == 0);
    const int64_t tiles = (N + TP - 1) / TP;
    const int64_t rounds = (tiles + (int64_t)gridDim.x * WARPS - 1) / ((int64_t)gridDim.x * WARPS);
    for (int o0 = 0; o0 < L; o0 += OC) {
        __syncthreads();
        for (int e = threadIdx.x; e < Lp * OC; e += blockDim.x) {
            const int m = e / OC, j = e - m * OC;
            Wt[e] = (m < L && o0 + j < L && m <= o0 + j) ? W[(size_t)(o0 + j) * L + m] : 0.0f;
        }
        __syncthreads();
        const int nch = min(Lp, o0 + OC + CH - 1) / CH;       // W is lower triangular: channels beyond o0 + 31 add nothing
        for (int64_t rd = 0; rd < rounds; ++rd) {
            const int64_t tile = (rd * gridDim.x + blockIdx.x) * WARPS + warp;
            const int64_t p0 = tile * TP;
            if (p0 >= N) continue;
            auto stage = [&](int cc, float *dst) {
                for (int i = 0; i < 16; ++i) {
                    const int idx = lane + 32 * i, row = idx >> 2, piece = idx & 3;
                    int64_t p = p0 + row;
                    if (p >= N) p = N - 1;
                    const int l = cc * CH + 4 * piece;
                    if (vec_ok) {
                        const float *src = Y + p * ldY + (l < L ? l : 0);
                        const unsigned nbytes = (l < L) ? 16u : 0u;
                        const unsigned sa = (unsigned)__cvta_generic_to_shared(dst + row * YST + 4 * piece);
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(nbytes) : "memory");
                    } else {
                        for (int q = 0; q < 4; ++q) dst[row * YST + 4 * piece + q] = (l + q < L) ? Y[p * ldY + l + q] : 0.0f;
                    }
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
            };
            float2 acc[OC][2];
#pragma unroll
            for (int r = 0; r < OC; ++r) { acc[r][0] = make_float2(0.0f, 0.0f); acc[r][1] = make_float2(0.0f, 0.0f); }
            stage(0, ybuf);
            for (int cc = 0; cc < nch; ++cc) {
                float *cur = ybuf + (cc & 1) * (TP * YST);
                if (cc + 1 < nch) {
                    stage(cc + 1, ybuf + ((cc + 1) & 1) * (TP * YST));
                    asm volatile("cp.async.wait_group 1;" ::: "memory");
                } else {
                    asm volatile("cp.async.wait_group 0;" ::: "memory");
                }
                __syncwarp();
#pragma unroll 1
                for (int l4 = 0; l4 < CH / 4; ++l4) {
                    float yv[4][4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const float4 y4 = *reinterpret_cast<const float4 *>(cur + (lane + 32 * j) * YST + 4 * l4);
                        yv[j][0] = y4.x; yv[j][1] = y4.y; yv[j][2] = y4.z; yv[j][3] = y4.w;
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const float *wrow = Wt + (size_t)(cc * CH + 4 * l4 + q) * OC;
                        const float2 y01 = make_float2(yv[0][q], yv[1][q]), y23 = make_float2(yv[2][q], yv[3][q]);
#pragma unroll
                        for (int r4 = 0; r4 < OC / 4; ++r4) {
                            const float4 a4 = *reinterpret_cast<const float4 *>(wrow + 4 * r4);
                            acc[4 * r4 + 0][0] = fma2(a4.x, y01, acc[4 * r4 + 0][0]); acc[4 * r4 + 0][1] = fma2(a4.x, y23, acc[4 * r4 + 0][1]);
                            acc[4 * r4 + 1][0] = fma2(a4.y, y01, acc[4 * r4 + 1][0]); acc[4 * r4 + 1][1] = fma2(a4.y, y23, acc[4 * r4 + 1][1]);
                            acc[4 * r4 + 2][0] = fma2(a4.z, y01, acc[4 * r4 + 2][0]); acc[4 * r4 + 2][1] = fma2(a4.z, y23, acc[4 * r4 + 2][1]);
                            acc[4 * r4 + 3][0] = fma2(a4.w, y01, acc[4 * r4 + 3][0]); acc[4 * r4 + 3][1] = fma2(a4.w, y23, acc[4 * r4 + 3][1]);
                        }
                    }
                }
                __syncwarp();
            }
            // a lane's pixels: p0 + lane + 32 j; 32 consecutive output channels each
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int64_t p = p0 + lane + 32 * j;
                if (p >= N) continue;
                float *o = Yw + p * L + o0;
#pragma unroll
                for (int r4 = 0; r4 < OC / 4; ++r4) {
                    float v[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float2 a2 = acc[4 * r4 + e][j >> 1];
                        v[e] = (j & 1) ? a2.y : a2.x;
                    }
                    if ((L & 3) == 0) {
                        if (o0 + 4 * r4 < L) *reinterpret_cast<float4 *>(o + 4 * r4) = make_float4(v[0], v[1], v[2], v[3]);
                    } else {
#pragma unroll
                        for (int e = 0; e < 4; ++e) if (o0 + 4 * r4 + e < L) o[4 * r4 + e] = v[e];
                    }
                }
            }
        }
    }
}

inline cudaError_t launch_whiten_spectra(const float *Y, int64_t ldY, int64_t N, int L, const float *W, bool diagonal,
                                         float *Yw, int sm_count, cudaStream_t stream) {
    if (N <= 0) return cudaSuccess;
    if (diagonal) {
        const int grid = (int)std::min<int64_t>((N * L + 255) / 256, (int64_t)sm_count * 16);
        whiten_spectra_diag_kernel<<<grid, 256, 0, stream>>>(Y, ldY, N, L, W, Yw);
        return cudaGetLastError();
    }
    const int Lp = (L + wh::CH - 1) / wh::CH * wh::CH;
    const size_t smem = ((size_t)Lp * wh::OC + (size_t)wh::WARPS * 2 * wh::TP * wh::YST) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(whiten_spectra_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t tiles = (N + wh::TP - 1) / wh::TP;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((tiles + wh::WARPS - 1) / wh::WARPS, sm_count));
    whiten_spectra_kernel<<<grid, wh::WARPS * 32, smem, stream>>>(Y, ldY, N, L, W, Yw);
    return cudaGetLastError();
}

// slo: drop the slack column of the internal (R + 1)-endmember outputs; the slack does not count as a support member.
__global__ void strip_slack_kernel(const float *__restrict__ ci, const float *__restrict__ si, int64_t N, int R, int Ri,
                                   float *__restrict__ coeffs, float *__restrict__ csig, int32_t *__restrict__ info) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < N * R; e += stride) {
        const int64_t p = e / R;
        const int r = (int)(e - p * R);
        coeffs[e] = ci[p * Ri + r];
        if (csig) csig[e] = si[p * Ri + r];
    }
    if (info) {
        for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < N; p += stride) {
            const int w = info[p];
            if (ci[p * Ri + Ri - 1] > 0.0f && ((w >> 24) & 0xff) > 0) info[p] = w - (1 << 24);
        }
    }
}

// slo without a slack endmember (R = 32): the problem is convex, so its minimiser is the pos minimiser where that one has
// sum a <= 1 and the sto minimiser elsewhere (the bound is active there).  One warp per pixel: where the pos result
// qualifies it replaces the sto result already in the caller's arrays.
__global__ void slo_select_kernel(int64_t N, int R, const float *__restrict__ cp, const float *__restrict__ sp,
                                  const float *__restrict__ rp, const int32_t *__restrict__ ip,
                                  float *__restrict__ coeffs, float *__restrict__ csig, float *__restrict__ resid,
                                  int32_t *__restrict__ info) {
    const int lane = threadIdx.x & 31;
    const int64_t stride = (int64_t)gridDim.x * (blockDim.x >> 5);
    for (int64_t p = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); p < N; p += stride) {
        float s = 0.0f;
        for (int r = lane; r < R; r += 32) s += cp[p * R + r];
        s = warp_sum(s);
        if (s <= 1.0f) {            // (a NaN sum, non-finite input, keeps the sto result: it is NaN as well)
            for (int r = lane; r < R; r += 32) {
                coeffs[p * R + r] = cp[p * R + r];
                if (csig) csig[p * R + r] = sp[p * R + r];
            }
            if (lane == 0) {
                if (resid) resid[p] = rp[p];
                if (info) info[p] = ip[p];
            }
        }
    }
}

}  // namespace linmin
