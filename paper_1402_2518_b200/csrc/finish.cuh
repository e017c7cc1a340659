// finish.cuh -- exact finish + uncertainty propagation + residual.
//
// IPLS in fp32 on the normal equations lands within ~1e-2 of the minimiser at best (the Gram matrix
// squares the library's condition number).  The tolerances of north_star (1e-4 on coefficients,
// 1e-5 on the objective, 1 % on uncertainties) need the minimiser itself, so each pixel is finished
// exactly: the support F = {i : a_i > 1e-4} of the IPLS iterate warm-starts a primal active-set loop
// whose equality-constrained sub-problems are solved with an fp64 Cholesky factor of G_FF (k x k, from
// the fp64 Gram matrix of the exact data) and right-hand sides formed IN DATA SPACE from the fp64
// residual r = y - A_F a_F.  Mean 0.2 support changes per pixel on the synthetic cubes.
//
//   PAPER.md:54, 63, 68 (eq. 2-4): the minimiser is characterised by  A_F'r = nu 1 on the support,
//       lambda_i = nu - A_i'r >= 0 off it, a_F > 0, 1'a_F = 1.
//   coefficient uncertainty "from the Hessian" (reading R3):
//       K = (A_F'A_F)^-1, H = K - K 1 1'K / (1'K 1), J = H A_F',
//       coeff_sigma_i = sqrt( sum_l J_il^2 sigma_l^2 ) on F, 0 elsewhere.
//   RMS = sqrt( mean_l r_l^2 )  (reading R8).
//
// One warp per pixel.  Everything k-sized lives in shared memory; k <= KMAX (32 for R <= 32, else 64).
#pragma once
#include "common.cuh"
#include "ipls_generic.cuh"

namespace linmin {


__host__ __device__ inline size_t finish_warp_bytes(int L, int R, int KMAX) {
    size_t dbl = (size_t)KMAX * (KMAX + 1) / 2   // Lf
                 + (size_t)L                      // r
                 + (size_t)6 * KMAX;              // aF, atry, gF, q, dinv, tmp
    size_t flt = (size_t)L                        // y
                 + (size_t)L                      // r32
                 + (size_t)KMAX * (KMAX + 1) / 2  // Hs
                 + (size_t)R;                     // g (all endmembers)
    size_t in = (size_t)KMAX + (size_t)((R + 3) / 4);  // idx, state bytes
    return dbl * 8 + flt * 4 + in * 4 + 16;
}

// state[i]: 0 free, 1 in F, 2 blocked (rejected as rank-deficient or degenerate tie)
// list: NULL = all pixels; else [0] = count, [1 + i] = pixel (the overflow list of finish_sweep_kernel)
__global__ void __launch_bounds__(256) finish_kernel(LibView lib, SolveParams prm, int KMAX,
                                                     const unsigned int *__restrict__ list) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (lib.flags[0]) return;
    const int L = lib.L, R = lib.R;
    const int warps = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *basep = smem_raw + (size_t)warp * ((finish_warp_bytes(L, R, KMAX) + 15) & ~(size_t)15);
    double *Lf = (double *)basep;
    double *r = Lf + (size_t)KMAX * (KMAX + 1) / 2;
    double *aF = r + L, *atry = aF + KMAX, *gF = atry + KMAX, *q = gF + KMAX, *dinv = q + KMAX,
           *tmp = dinv + KMAX;
    float *y = (float *)(tmp + KMAX);
    float *r32 = y + L, *Hs = r32 + L, *g = Hs + (size_t)KMAX * (KMAX + 1) / 2;
    int *idx = (int *)(g + R);
    unsigned char *state = (unsigned char *)(idx + KMAX);
    const float *A = lib.A;      // by channel: the multiplier pass walks the endmembers across the lanes
    const float *At = lib.At;    // by endmember: every pass over the channels of one member reads consecutive addresses
    const int max_pivots = 4 * KMAX + 8;
    const bool cons = lib.cons != 0;      // false: positivity only (no equality constraint; the empty support is feasible)

    const int64_t count = list ? (int64_t)list[0] : prm.N;
    for (int64_t pi = (int64_t)blockIdx.x * warps + warp; pi < count; pi += (int64_t)gridDim.x * warps) {
        const int64_t p = list ? (int64_t)list[1 + pi] : pi;
        float *cout = prm.coeffs + p * R;
        int info = prm.info ? prm.info[p] : 0;
        // ---- load y; detect non-finite
        bool bad = false;
        for (int l = lane; l < L; l += 32) {
            float yv = prm.Y[p * prm.ldY + l];
            bad |= !isfinite(yv);
            y[l] = yv;
        }
        if (__any_sync(0xffffffffu, bad)) {
            const float qnan = __int_as_float(0x7fc00000);
            for (int i = lane; i < R; i += 32) {
                cout[i] = qnan;
                if (prm.coeff_sigma) prm.coeff_sigma[p * R + i] = qnan;
            }
            if (lane == 0) {
                if (prm.resid) prm.resid[p] = qnan;
                if (prm.info) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            }
            __syncwarp();
            continue;
        }
        // ---- initial support from the IPLS iterate (largest KMAX entries above the threshold)
        int k = 0;
        float amax = -1.0f; int imax = 0;
        for (int i0 = 0; i0 < R; i0 += 32) {
            int i = i0 + lane;
            float ai = (i < R) ? cout[i] : -1.0f;
            if (ai > amax) { amax = ai; imax = i; }
            bool in = (i < R) && (ai > LINMIN_SUPPORT_THRESHOLD);
            unsigned m = __ballot_sync(0xffffffffu, in);
            int pos = k + __popc(m & ((1u << lane) - 1u));
            if (i < R) state[i] = 0;
            if (in && pos < KMAX) { idx[pos] = i; aF[pos] = (double)ai; state[i] = 1; }
            k = min(KMAX, k + __popc(m));
        }
        if (k == 0 && cons) {   // (can not happen for a point on the simplex; be safe) take the largest entry
            float best = warp_max(amax);
            unsigned m = __ballot_sync(0xffffffffu, amax == best);
            int src = __ffs(m) - 1;
            int ib = __shfl_sync(0xffffffffu, imax, src);
            if (lane == 0) { idx[0] = ib; aF[0] = 1.0; state[ib] = 1; }
            k = 1;
        }
        __syncwarp();
        if (cons) {   // normalise onto the simplex
            double s = 0.0;
            for (int j = lane; j < k; j += 32) s += aF[j];
            s = warp_sum(s);
            for (int j = lane; j < k; j += 32) aF[j] /= s;
        }
        __syncwarp();

        int pivots = 0, last_added = -1;
        bool fallback = false;
        double nu = 0.0;
        while (true) {
            // ---- factor G_FF (fp64)
            for (int j = 0; j < k; ++j)
                for (int i = j + lane; i < k; i += 32) Lf[cm(k, i, j)] = lib.G64[(size_t)idx[i] * R + idx[j]];
            __syncwarp();
            // rank test per column inside the factorisation: pivot <= 1e-13 * G_jj -> reject index
            int rej = -1;
            for (int j = 0; j < k && rej < 0; ++j) {
                double gjj = Lf[cm(k, j, j)];
                double sj = gjj;
                for (int kk = 0; kk < j; ++kk) { double l = Lf[cm(k, j, kk)]; sj -= l * l; }
                if (!(sj > 1e-13 * gjj)) { rej = j; break; }
                double dj = 1.0 / sqrt(sj);
                for (int i = j + lane; i < k; i += 32) {
                    if (i == j) dinv[j] = dj;
                    else {
                        double s = Lf[cm(k, i, j)];
                        for (int kk = 0; kk < j; ++kk) s -= Lf[cm(k, i, kk)] * Lf[cm(k, j, kk)];
                        Lf[cm(k, i, j)] = s * dj;
                    }
                }
                __syncwarp();
            }
            if (rej >= 0) {
                // A_F lost rank at column rej (R9): drop that member, block it, continue at the same point
                __syncwarp();
                int ridx = idx[rej];
                double arej = aF[rej];
                __syncwarp();
                if (lane == 0) {
                    state[ridx] = 2;
                    for (int j = rej; j + 1 < k; ++j) { idx[j] = idx[j + 1]; aF[j] = aF[j + 1]; }
                }
                --k; last_added = -1;
                __syncwarp();
                if (k == 0 && cons) { fallback = true; break; }
                if (arej != 0.0 && cons) {
                    double s = 0.0;
                    for (int j = lane; j < k; j += 32) s += aF[j];
                    s = warp_sum(s);
                    for (int j = lane; j < k; j += 32) aF[j] /= s;
                    __syncwarp();
                }
                if (++pivots > max_pivots) { fallback = true; break; }
                continue;
            }
            // ---- q = K 1
            for (int j = lane; j < k; j += 32) q[j] = 1.0;
            __syncwarp();
            team_solve<32, 1, double>(Lf, dinv, k, q, nullptr);
            double sq = 0.0;
            for (int j = lane; j < k; j += 32) sq += q[j];
            sq = warp_sum(sq);
            // ---- data-space residual at the current point and its projection on the support
            for (int l = lane; l < L; l += 32) {
                double s = (double)y[l];
                for (int j = 0; j < k; ++j) s -= (double)At[(size_t)idx[j] * L + l] * aF[j];
                r[l] = s;
            }
            __syncwarp();
            double suma = 0.0;
            for (int j = 0; j < k; ++j) {
                double s = 0.0;
                for (int l = lane; l < L; l += 32) s += (double)At[(size_t)idx[j] * L + l] * r[l];
                s = warp_sum(s);
                if (lane == 0) { gF[j] = s; atry[j] = s; }
                suma += aF[j];
            }
            __syncwarp();
            // ---- Newton step to the sub-problem solution: G_FF d + mu 1 = g_F, 1'd = 1 - 1'a_F
            team_solve<32, 1, double>(Lf, dinv, k, atry, nullptr);   // atry = K g_F
            double sp = 0.0;
            for (int j = lane; j < k; j += 32) sp += atry[j];
            sp = warp_sum(sp);
            double mu = cons ? (sp - (1.0 - suma)) / sq : 0.0;
            double amin = INFINITY;
            for (int j = lane; j < k; j += 32) {
                double an = aF[j] + atry[j] - mu * q[j];
                atry[j] = an;
                amin = fmin(amin, an);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) amin = fmin(amin, __shfl_xor_sync(0xffffffffu, amin, o));
            __syncwarp();
            if (!(amin > 0.0)) {
                // ---- ratio step: move towards atry until the first coefficient reaches zero
                double alpha = 1.0;
                for (int j = lane; j < k; j += 32) {
                    if (!(atry[j] > 0.0)) {
                        double den = aF[j] - atry[j];
                        double tt = den > 0.0 ? aF[j] / den : 0.0;
                        alpha = fmin(alpha, tt);
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) alpha = fmin(alpha, __shfl_xor_sync(0xffffffffu, alpha, o));
                if (alpha < 0.0) alpha = 0.0;
                __syncwarp();
                int nk = 0;
                if (lane == 0) {
                    double s = 0.0;
                    for (int j = 0; j < k; ++j) {
                        double an = aF[j] + alpha * (atry[j] - aF[j]);
                        double den = aF[j] - atry[j];
                        bool blocking = !(atry[j] > 0.0) && ((den > 0.0 ? aF[j] / den : 0.0) <= alpha);
                        if (blocking || !(an > 0.0)) {
                            state[idx[j]] = (idx[j] == last_added && alpha == 0.0) ? 2 : 0;
                        } else {
                            idx[nk] = idx[j]; aF[nk] = an; s += an; ++nk;
                        }
                    }
                    if (cons) for (int j = 0; j < nk; ++j) aF[j] /= s;
                }
                k = __shfl_sync(0xffffffffu, nk, 0);
                last_added = -1;
                __syncwarp();
                if ((k == 0 && cons) || ++pivots > max_pivots) { fallback = true; break; }
                continue;
            }
            // ---- accept; residual and gradient at the new point
            for (int j = lane; j < k; j += 32) aF[j] = atry[j];
            __syncwarp();
            for (int l = lane; l < L; l += 32) {
                double s = (double)y[l];
                for (int j = 0; j < k; ++j) s -= (double)At[(size_t)idx[j] * L + l] * aF[j];
                r[l] = s;
                r32[l] = (float)s;
            }
            __syncwarp();
            nu = 0.0;
            for (int j = 0; j < k; ++j) {
                double s = 0.0;
                for (int l = lane; l < L; l += 32) s += (double)At[(size_t)idx[j] * L + l] * r[l];
                s = warp_sum(s);
                nu += s * aF[j];
            }
            if (!cons) nu = 0.0;
            // multipliers lambda_i = nu - A_i'r off the support (fp32 dot products of the fp64 residual)
            float lmin = INFINITY; int jmin = -1; float gmax = 0.0f;
            for (int i = lane; i < R; i += 32) {
                float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;      // four chains: the loads of a chain overlap
                int l = 0;
                for (; l + 3 < L; l += 4) {
                    s0 = fmaf(A[(size_t)(l + 0) * R + i], r32[l + 0], s0);
                    s1 = fmaf(A[(size_t)(l + 1) * R + i], r32[l + 1], s1);
                    s2 = fmaf(A[(size_t)(l + 2) * R + i], r32[l + 2], s2);
                    s3 = fmaf(A[(size_t)(l + 3) * R + i], r32[l + 3], s3);
                }
                for (; l < L; ++l) s0 = fmaf(A[(size_t)l * R + i], r32[l], s0);
                const float s = (s0 + s1) + (s2 + s3);
                gmax = fmaxf(gmax, fabsf(s));
                if (state[i] == 0) {
                    float li = (float)nu - s;
                    if (li < lmin) { lmin = li; jmin = i; }
                }
            }
            gmax = warp_max(gmax);
            float lbest = warp_min(lmin);
            unsigned mm = __ballot_sync(0xffffffffu, lmin == lbest && jmin >= 0);
            if (!(lbest < -1e-6f * gmax) || mm == 0u) break;          // optimal
            if (k >= KMAX || pivots >= max_pivots) { fallback = true; break; }
            int src = __ffs(mm) - 1;
            int jadd = __shfl_sync(0xffffffffu, jmin, src);
            if (lane == 0) { idx[k] = jadd; aF[k] = 0.0; state[jadd] = 1; }
            ++k; ++pivots; last_added = jadd;
            __syncwarp();
        }

        // ---- outputs: coefficients (exact zeros off the support), residual
        for (int i = lane; i < R; i += 32) cout[i] = 0.0f;
        __syncwarp();
        for (int j = lane; j < k; j += 32) cout[idx[j]] = (float)aF[j];
        if (fallback) {
            // residual at the current feasible point
            for (int l = lane; l < L; l += 32) {
                double s = (double)y[l];
                for (int j = 0; j < k; ++j) s -= (double)At[(size_t)idx[j] * L + l] * aF[j];
                r[l] = s;
            }
            __syncwarp();
            info |= LINMIN_INFO_FINISH_FALLBACK;
        }
        if (prm.resid) {
            double s = 0.0;
            for (int l = lane; l < L; l += 32) s += r[l] * r[l];
            s = warp_sum(s);
            if (lane == 0) prm.resid[p] = (float)sqrt(s / (double)L);
        }
        // ---- uncertainty propagation
        if (prm.coeff_sigma) {
            float *sout = prm.coeff_sigma + p * R;
            for (int i = lane; i < R; i += 32) sout[i] = 0.0f;
            __syncwarp();
            bool sbad = false;
            if (prm.has_sigma) {
                const float *sg = prm.sigma + p * prm.sigma_stride;
                for (int l = lane; l < L; l += 32) { float sv = sg[l]; sbad |= !(sv > 0.0f) || !isfinite(sv); }
            }
            sbad = __any_sync(0xffffffffu, sbad);
            if (sbad) {
                const float qnan = __int_as_float(0x7fc00000);
                for (int i = lane; i < R; i += 32) sout[i] = qnan;
                info |= LINMIN_INFO_BAD_SIGMA;
            } else if (k > (cons ? 1 : 0) && !fallback) {
                // Lf, dinv, q hold the factor of the FINAL support (last loop pass ended in `break`
                // right after an accepted solve).  W = L^-1 in place (column by column from the end).
                double sq = 0.0;
                for (int j = lane; j < k; j += 32) sq += q[j];
                sq = warp_sum(sq);
                for (int j = k - 1; j >= 0; --j) {
                    for (int i = j + 1 + lane; i < k; i += 32) tmp[i] = Lf[cm(k, i, j)];
                    __syncwarp();
                    double wjj = dinv[j];
                    for (int i = j + 1 + lane; i < k; i += 32) {
                        double s = 0.0;
                        for (int m = j + 1; m <= i; ++m) s += ((m == i) ? dinv[i] : Lf[cm(k, i, m)]) * tmp[m];
                        Lf[cm(k, i, j)] = -s * wjj;
                    }
                    __syncwarp();
                }
                // H = W'W - q q'/(1'q)  (packed lower, fp32)
                for (int j = 0; j < k; ++j)
                    for (int i = j + lane; i < k; i += 32) {
                        double s = 0.0;
                        for (int m = i; m < k; ++m) {
                            double wmi = (m == i) ? dinv[i] : Lf[cm(k, m, i)];
                            double wmj = (m == j) ? dinv[j] : Lf[cm(k, m, j)];
                            s += wmi * wmj;
                        }
                        Hs[cm(k, i, j)] = (float)(cons ? s - q[i] * q[j] / sq : s);     // pos: H = K, no projection
                    }
                __syncwarp();
                const float *sg = prm.has_sigma ? prm.sigma + p * prm.sigma_stride : nullptr;
                // J = H A_F' as a small matrix product per chunk of 256 channels (8 per lane): four rows of H at a
                // time, so that a member's library values are loaded once per four rows and H once per 8 channels
                for (int i = lane; i < k; i += 32) tmp[i] = 0.0;
                __syncwarp();
                for (int l0 = 0; l0 < L; l0 += 256) {
                    float sv[8];
#pragma unroll
                    for (int c = 0; c < 8; ++c) {
                        const int l = l0 + lane + 32 * c;
                        sv[c] = (l < L) ? (sg ? sg[l] : 1.0f) : 0.0f;
                    }
                    for (int i0 = 0; i0 < k; i0 += 4) {
                        float d[4][8];
#pragma unroll
                        for (int ii = 0; ii < 4; ++ii)
#pragma unroll
                            for (int c = 0; c < 8; ++c) d[ii][c] = 0.0f;
                        for (int j = 0; j < k; ++j) {
                            const float *row = At + (size_t)idx[j] * L + l0 + lane;
                            float a[8], h[4];
#pragma unroll
                            for (int c = 0; c < 8; ++c) a[c] = (l0 + lane + 32 * c < L) ? row[32 * c] : 0.0f;
#pragma unroll
                            for (int ii = 0; ii < 4; ++ii) {
                                const int i = i0 + ii;
                                h[ii] = (i < k) ? ((i >= j) ? Hs[cm(k, i, j)] : Hs[cm(k, j, i)]) : 0.0f;
                            }
#pragma unroll
                            for (int ii = 0; ii < 4; ++ii)
#pragma unroll
                                for (int c = 0; c < 8; ++c) d[ii][c] = fmaf(h[ii], a[c], d[ii][c]);
                        }
#pragma unroll
                        for (int ii = 0; ii < 4; ++ii) {
                            float acc = 0.0f;
#pragma unroll
                            for (int c = 0; c < 8; ++c) {
                                const float dv = d[ii][c] * sv[c];
                                acc = fmaf(dv, dv, acc);
                            }
                            acc = warp_sum(acc);
                            if (lane == 0 && i0 + ii < k) tmp[i0 + ii] += (double)acc;
                        }
                    }
                }
                __syncwarp();
                for (int i = lane; i < k; i += 32) sout[idx[i]] = sqrtf((float)tmp[i]);
            }
        }
        if (prm.info && lane == 0) {
            int pv = pivots > 255 ? 255 : pivots;
            prm.info[p] = (info & 0xffff) | (pv << 16) | (k << 24);
        }
        __syncwarp();
    }
}

}  // namespace linmin
