// detect.cuh -- NEXT rows 3 and 4 of SURVEY.md 8(f): library builder, detection layer, autofit.
//
//   additional_spectra_kernel   PAPER.md:112-114 (sec. 2.5), :333-339 (appendix): Flat 1, Flat 0.0001, Slope increasing,
//                               Slope decreasing, then +-cos / +-sin over a quarter and over half a period of the
//                               spectral domain (reading R18 of DESIGN.md).
//   threshold_*                 PAPER.md:149-153 (eq. 8): C^i = 1/2 (mean(A+) - 2 std(A+) + mean(A-) + 6 std(A-)) from a
//                               labelled set (reading R19): fp64 class sums per endmember, summed in a fixed order.
//   detect_kernel               PAPER.md:239-246: coefficient above its threshold, error below the coefficient, RMS
//                               below the noise level.
//   gather / scatter            PAPER.md:294: second pass on the detected sub-library.
//   autofit_ls_kernel           PAPER.md:94-100 (eq. 7), unconstrained: residue of S_n against the other endmembers by
//                               modified Gram-Schmidt (twice) in fp64, data space -- no normal equations.
// All of these are HBM-bound scans over the outputs or once-per-library work; none is on the per-pixel hot path.
#pragma once
#include "common.cuh"

namespace linmin {

// out[l * ld + col0 + j], j < n_extra (4 or 12); wavelength == NULL: position = l / (L - 1)
__global__ void additional_spectra_kernel(const float *__restrict__ wavelength, int L, int n_extra, float *__restrict__ out,
                                          int ld, int col0) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= L) return;
    double x;
    if (wavelength) {
        const double w0 = (double)wavelength[0], w1 = (double)wavelength[L - 1];
        x = ((double)wavelength[l] - w0) / (w1 - w0);
    } else {
        x = (L > 1) ? (double)l / (double)(L - 1) : 0.0;
    }
    float *o = out + (size_t)l * ld + col0;
    o[0] = 1.0f; o[1] = 1e-4f; o[2] = (float)x; o[3] = (float)(1.0 - x);
    if (n_extra == 12) {
        const double pi = 3.14159265358979323846;
        for (int h = 0; h < 2; ++h) {
            const double ph = 2.0 * pi * (h ? 0.5 : 0.25) * x;
            const double c = cos(ph), s = sin(ph);
            o[4 + 4 * h] = (float)c; o[5 + 4 * h] = (float)s; o[6 + 4 * h] = (float)-c; o[7 + 4 * h] = (float)-s;
        }
    }
}

// ---- eq. 8.  Stage 1: block b accumulates, for each endmember, (count, sum, sum of squares) of the detections (> 0;
// with whole_class: of every estimate) on present / absent pixels in fp64; a thread stays on ONE column (blockDim.x is a multiple of R), so the loads are
// coalesced and the per-thread sums need no exchange until the end.  part: [gridDim.x][R][6].
__global__ void threshold_partial_kernel(const float *__restrict__ coeffs, const unsigned char *__restrict__ present,
                                         int64_t N, int R, int whole_class, double *__restrict__ part) {
    extern __shared__ double sh[];          // [blockDim.x][6]
    const int64_t total = N * R;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const float v = coeffs[e];
        if (whole_class || v > 0.0f) {          // whole_class: every pixel of the class, exact zeros included
            const int o = present[e] ? 0 : 3;
            acc[o] += 1.0; acc[o + 1] += (double)v; acc[o + 2] += (double)v * (double)v;
        }
    }
    for (int k = 0; k < 6; ++k) sh[threadIdx.x * 6 + k] = acc[k];
    __syncthreads();
    // stride is a multiple of R (the launcher makes blockDim.x one): thread t always sees column (t mod R)
    if (threadIdx.x < R) {
        double s[6] = {0, 0, 0, 0, 0, 0};
        for (int t = threadIdx.x; t < blockDim.x; t += R)
            for (int k = 0; k < 6; ++k) s[k] += sh[t * 6 + k];
        for (int k = 0; k < 6; ++k) part[((size_t)blockIdx.x * R + threadIdx.x) * 6 + k] = s[k];
    }
}
__global__ void threshold_final_kernel(const double *__restrict__ part, int nblocks, int R, float *__restrict__ thr) {
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

// mask[p][i] = coeff > thr_i  &&  coeff_sigma < coeff  &&  resid_p < rms_max;  counts[i] += detections (integer atomics)
__global__ void detect_kernel(const float *__restrict__ coeffs, const float *__restrict__ csig, const float *__restrict__ resid,
                              const float *__restrict__ thr, float rms_max, int64_t N, int R, unsigned char *__restrict__ mask,
                              unsigned long long *__restrict__ counts) {
    extern __shared__ unsigned int cnt[];       // [R]
    for (int i = threadIdx.x; i < R; i += blockDim.x) cnt[i] = 0u;
    __syncthreads();
    const int64_t total = N * R;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += stride) {
        const int64_t p = e / R;
        const int i = (int)(e - p * R);
        const float c = coeffs[e];
        const bool d = (resid[p] < rms_max) && (c > thr[i]) && (csig[e] < c);
        mask[e] = d ? 1 : 0;
        if (d && counts) atomicAdd(&cnt[i], 1u);
    }
    __syncthreads();
    if (counts)
        for (int i = threadIdx.x; i < R; i += blockDim.x)
            if (cnt[i]) atomicAdd(&counts[i], (unsigned long long)cnt[i]);
}

// sub[l][j] = A[l][idx[j]]
__global__ void gather_columns_kernel(const float *__restrict__ A, int L, int R, const int *__restrict__ idx, int Rs,
                                      float *__restrict__ sub) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= L * Rs) return;
    const int l = e / Rs, j = e - l * Rs;
    sub[e] = A[(size_t)l * R + idx[j]];
}
// full[p][idx[j]] = sub[p][j], zero elsewhere (full is N x R, pre-zeroed by the caller)
__global__ void scatter_columns_kernel(const float *__restrict__ sub, int64_t N, int Rs, const int *__restrict__ idx, int R,
                                       float *__restrict__ full) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < N * Rs; e += stride) {
        const int64_t p = e / Rs;
        const int j = (int)(e - p * Rs);
        full[p * R + idx[j]] = sub[e];
    }
}

// Autofit helpers: Sn[l][j] = A[l][j < n ? j : j + 1] (the library without endmember n), yrow[l] = A[l][n]
__global__ void drop_column_kernel(const float *__restrict__ A, int L, int R, int n, float *__restrict__ Sn, float *__restrict__ yrow) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < L) yrow[e] = A[(size_t)e * R + n];
    if (e >= L * (R - 1)) return;
    const int l = e / (R - 1), j = e - l * (R - 1);
    Sn[e] = A[(size_t)l * R + (j < n ? j : j + 1)];
}
// E[l][n] = A[l][n] - sum_j Sn[l][j] a[j]   (fp64 accumulate; a = the non-negative fit of endmember n by the others)
__global__ void autofit_residue_kernel(const float *__restrict__ A, int L, int R, int n, const float *__restrict__ Sn,
                                       const float *__restrict__ a, float *__restrict__ E) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= L) return;
    double s = (double)A[(size_t)l * R + n];
    for (int j = 0; j < R - 1; ++j) s -= (double)Sn[(size_t)l * (R - 1) + j] * (double)a[j];
    E[(size_t)l * R + n] = (float)s;
}

// Unconstrained autofit, one CTA per endmember n: modified Gram-Schmidt (each column orthogonalised twice) of the other
// endmembers in fp64, columns that lose more than 12 digits dropped (rank deficiency), then the residue of S_n against
// the basis.  Q: workspace [R][L * (R - 1)] doubles; E[l][n] = residue.
__global__ void __launch_bounds__(256)
autofit_ls_kernel(const float *__restrict__ A, int L, int R, double *__restrict__ Qws, float *__restrict__ E) {
    const int n = blockIdx.x, tid = threadIdx.x, nt = blockDim.x;
    double *Q = Qws + (size_t)n * L * (R - 1);
    __shared__ double red[256];
    __shared__ double v[LINMIN_MAX_L];
    auto block_sum = [&](double x) -> double {
        red[tid] = x;
        __syncthreads();
        for (int o = nt >> 1; o > 0; o >>= 1) { if (tid < o) red[tid] += red[tid + o]; __syncthreads(); }
        const double r = red[0];
        __syncthreads();
        return r;
    };
    int nq = 0;
    for (int jj = 0; jj <= R - 1; ++jj) {
        // columns of the others first, S_n itself last
        const int col = (jj == R - 1) ? n : (jj < n ? jj : jj + 1);
        for (int l = tid; l < L; l += nt) v[l] = (double)A[(size_t)l * R + col];
        __syncthreads();
        double n0 = 0.0;
        for (int l = tid; l < L; l += nt) n0 += v[l] * v[l];
        n0 = block_sum(n0);
        for (int pass = 0; pass < 2; ++pass)
            for (int q = 0; q < nq; ++q) {
                double d = 0.0;
                for (int l = tid; l < L; l += nt) d += Q[(size_t)q * L + l] * v[l];
                d = block_sum(d);
                for (int l = tid; l < L; l += nt) v[l] -= d * Q[(size_t)q * L + l];
                __syncthreads();
            }
        if (jj == R - 1) break;
        double n1 = 0.0;
        for (int l = tid; l < L; l += nt) n1 += v[l] * v[l];
        n1 = block_sum(n1);
        if (n1 > 1e-24 * n0 && n1 > 0.0) {
            const double r = 1.0 / sqrt(n1);
            for (int l = tid; l < L; l += nt) Q[(size_t)nq * L + l] = v[l] * r;
            ++nq;
        }
        __syncthreads();
    }
    for (int l = tid; l < L; l += nt) E[(size_t)l * R + n] = (float)v[l];
}

}  // namespace linmin
