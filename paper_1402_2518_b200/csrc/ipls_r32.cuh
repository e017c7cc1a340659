// ipls_r32.cuh -- register-blocked projection + IPLS kernel for R = 32 endmembers (sm_100a).
//
// Same iteration as ipls_generic.cuh (Mehrotra predictor-corrector on the centred normal equations;
// PAPER.md:71-73 names IPLS and prints no steps -- DESIGN.md reading R1), mapped to the hardware:
//
//   * 8 lanes cooperate on one pixel, 4 pixels per warp.  Lane t of a group owns rows
//     i = t + 8 s (s = 0..3, cyclic) of the 32 x 32 Newton matrix M = G + diag(lambda/a): row i is
//     kept in REGISTERS up to column 8 s + 7 (80 registers for the lower triangle plus the
//     upper part of the diagonal blocks, which is kept at zero).
//   * Right-looking Cholesky, fully unrolled (static register indices).  Column k of L is broadcast
//     to the group through a double-buffered, bank-padded shared-memory line (<= 4 STS.32, one
//     __syncwarp, <= 8 LDS.128 per step): 16 FMAs per LDS.128 instead of 1 per shuffle.
//   * Forward substitution in broadcast form (one shuffle per row and right-hand side), backward
//     substitution in reduction form (3-shuffle group sum per row), both on the register-resident L.
//     The sum-to-one multiplier is eliminated through w = L^-1 1, so an iteration needs three
//     forward and two backward substitutions.
//   * G (padded rows), the centred library (re-laid out so that a lane's four rows are one LDS.128)
//     and the channel means live in shared memory, loaded once per CTA; warps then run independently
//     and fetch groups of 4 pixels from a global atomic counter (per-pixel iteration counts vary).
//
// Algorithmic work per pixel: 2 L R + it (R^3/3 + 8 R^2 + 30 R) flops.
#pragma once
#include "common.cuh"

namespace linmin {

namespace r32 {

constexpr int R = 32;
constexpr int GST = 36;        // padded row stride of G in shared memory (bank-conflict-free LDS.128)
constexpr int XST = 40;        // per-pixel stride of the exchange lines (4 pixels -> 4 x 8 banks)
constexpr int WARPS = 4;       // warps per CTA
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float gsum(float v) {   // sum over the 8 lanes of a pixel group
    v += __shfl_xor_sync(FULL, v, 1);
    v += __shfl_xor_sync(FULL, v, 2);
    v += __shfl_xor_sync(FULL, v, 4);
    return v;
}
__device__ __forceinline__ float gmax(float v) {
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 1));
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 2));
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 4));
    return v;
}

// shared-memory footprint in floats
__host__ __device__ inline int lpad(int L) { return (L + 3) & ~3; }
__host__ __device__ inline int ystride(int L) { return lpad(L) + 8; }
__host__ __device__ inline size_t smem_floats(int L) {
    return (size_t)R * GST + R                 // Gp, row sums
           + (size_t)lpad(L) * R + lpad(L)      // Acp, c
           + (size_t)WARPS * (4 * ystride(L) + 2 * 4 * XST);
}

// L z = r for NR right-hand sides (in place; r[q][s] ends as z at row t + 8 s)
template <int NR>
__device__ __forceinline__ void forward_subst(const float (&m)[4][32], const float (&dinv)[4],
                                              float (&r)[NR][4], int t) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {
        const int s0 = j >> 3, t0 = j & 7;
#pragma unroll
        for (int q = 0; q < NR; ++q) {
            float z = r[q][s0] * dinv[s0];
            float zj = __shfl_sync(FULL, z, t0, 8);
            // rows above j in this slot have m[s0][j] == 0 (upper part kept at zero): unchanged
            float upd = fmaf(-m[s0][j], zj, r[q][s0]);
            r[q][s0] = (t == t0) ? zj : upd;
#pragma unroll
            for (int s = s0 + 1; s < 4; ++s) r[q][s] = fmaf(-m[s][j], zj, r[q][s]);
        }
    }
}

// L' x = z (reduction form); x[s] at row t + 8 s
__device__ __forceinline__ void backward_subst(const float (&m)[4][32], const float (&dinv)[4],
                                               const float (&z)[4], float (&x)[4], int t) {
#pragma unroll
    for (int s = 0; s < 4; ++s) x[s] = 0.0f;
#pragma unroll
    for (int i = 31; i >= 0; --i) {
        const int s0 = i >> 3, t0 = i & 7;
        float part = 0.0f;
#pragma unroll
        for (int s = s0; s < 4; ++s) part = fmaf(m[s][i], x[s], part);
        float tot = gsum(part);
        float xi = (z[s0] - tot) * dinv[s0];
        x[s0] = (t == t0) ? xi : x[s0];
    }
}

}  // namespace r32

__global__ void __launch_bounds__(r32::WARPS * 32, 3)
ipls_r32_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter) {
    using namespace r32;
    extern __shared__ __align__(16) float smem[];
    const int L = lib.L;
    const int Lp = lpad(L), YST = ystride(L);
    float *Gp = smem;                        // [32][GST]
    float *Grs = Gp + R * GST;               // [32] row sums of G
    float *Acp = Grs + R;                    // [Lp][32]: Acp[l][t*4+s] = Ac[l][t+8s]
    float *cv = Acp + (size_t)Lp * R;        // [Lp]
    float *wbase = cv + Lp + (size_t)(threadIdx.x >> 5) * (4 * YST + 2 * 4 * XST);
    const int lane = threadIdx.x & 31, g = lane >> 3, t = lane & 7;
    float *ybuf = wbase + g * YST;                         // this pixel's centred spectrum
    float *xb0 = wbase + 4 * YST + g * XST;                // exchange line, buffer 0
    float *xb1 = xb0 + 4 * XST;                            // buffer 1

    // ---- once per CTA: stage the library data
    for (int e = threadIdx.x; e < R * R; e += blockDim.x) Gp[(e >> 5) * GST + (e & 31)] = lib.Gc[e];
    for (int e = threadIdx.x; e < Lp * R; e += blockDim.x) {
        int l = e >> 5, c = e & 31, tt = c >> 2, s = c & 3;
        Acp[e] = (l < L) ? lib.Ac[(size_t)l * R + tt + 8 * s] : 0.0f;
    }
    for (int l = threadIdx.x; l < Lp; l += blockDim.x) cv[l] = (l < L) ? lib.c[l] : 0.0f;
    __syncthreads();
    if (threadIdx.x < R) {
        float s = 0.0f;
        for (int j = 0; j < R; ++j) s += Gp[threadIdx.x * GST + j];
        Grs[threadIdx.x] = s;
    }
    __syncthreads();

    const float gdmax = lib.gdmax;
    const float tau = 0.995f;
    const float pivot_floor = 1e-12f * gdmax;

    while (true) {
        unsigned int grp = 0;
        if (lane == 0) grp = atomicAdd(counter, 1u);
        grp = __shfl_sync(FULL, grp, 0);
        const int64_t p0 = (int64_t)grp * 4;
        if (p0 >= prm.N) break;
        const bool valid = (p0 + g) < prm.N;
        const int64_t p = valid ? (p0 + g) : (prm.N - 1);

        // ---- load the spectrum (8 lanes x 4 B = one 32 B sector per step), centre, flag non-finite
        const float *y = prm.Y + p * prm.ldY;
        bool bad = false;
        for (int l = t; l < Lp; l += 8) {
            float yv = (l < L) ? y[l] : 0.0f;
            bad |= !isfinite(yv);
            ybuf[l] = yv - cv[l];
        }
        bad = __any_sync(0xffu << (8 * g), bad);
        __syncwarp();
        if (bad) for (int l = t; l < Lp; l += 8) ybuf[l] = 0.0f;
        __syncwarp();

        // ---- projection b = Ac'(y - c)
        float b[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        for (int l4 = 0; l4 < Lp; l4 += 4) {
            float4 y4 = *reinterpret_cast<const float4 *>(ybuf + l4);
            float4 a0 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 0) * R + t * 4);
            float4 a1 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 1) * R + t * 4);
            float4 a2 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 2) * R + t * 4);
            float4 a3 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 3) * R + t * 4);
            b[0] = fmaf(a0.x, y4.x, b[0]); b[1] = fmaf(a0.y, y4.x, b[1]); b[2] = fmaf(a0.z, y4.x, b[2]); b[3] = fmaf(a0.w, y4.x, b[3]);
            b[0] = fmaf(a1.x, y4.y, b[0]); b[1] = fmaf(a1.y, y4.y, b[1]); b[2] = fmaf(a1.z, y4.y, b[2]); b[3] = fmaf(a1.w, y4.y, b[3]);
            b[0] = fmaf(a2.x, y4.z, b[0]); b[1] = fmaf(a2.y, y4.z, b[1]); b[2] = fmaf(a2.z, y4.z, b[2]); b[3] = fmaf(a2.w, y4.z, b[3]);
            b[0] = fmaf(a3.x, y4.w, b[0]); b[1] = fmaf(a3.y, y4.w, b[1]); b[2] = fmaf(a3.z, y4.w, b[2]); b[3] = fmaf(a3.w, y4.w, b[3]);
        }
        float bmax = gmax(fmaxf(fmaxf(fabsf(b[0]), fabsf(b[1])), fmaxf(fabsf(b[2]), fabsf(b[3]))));
        const float sc = fmaxf(bmax, 1e-3f * gdmax);

        // ---- start: a = 1/R, nu = 0, lambda = max(||G a - b||_inf, 1e-3 gdmax)
        float a[4], lam[4], w[4];
        float g0 = 0.0f;
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            a[s] = 1.0f / 32.0f;
            g0 = fmaxf(g0, fabsf(Grs[t + 8 * s] * (1.0f / 32.0f) - b[s]));
        }
        const float lam0 = fmaxf(gmax(g0), 1e-3f * gdmax);
#pragma unroll
        for (int s = 0; s < 4; ++s) lam[s] = lam0;
        float nu = 0.0f;
        int iters = 0, flags = bad ? LINMIN_INFO_NONFINITE_INPUT : 0;
        bool done = false;

        for (int it = 0;; ++it) {
            // ---- exchange a; G a and the Newton matrix rows from shared memory
            float *xe = (it & 1) ? xb1 : xb0;      // this iteration's "even" line
            float *xo = (it & 1) ? xb0 : xb1;
            __syncwarp();
#pragma unroll
            for (int s = 0; s < 4; ++s) xe[t + 8 * s] = a[s];
            __syncwarp();
            float m[4][32];
            float Ga[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                float4 a4 = *reinterpret_cast<const float4 *>(xe + 4 * c);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    float4 g4 = *reinterpret_cast<const float4 *>(Gp + (t + 8 * s) * GST + 4 * c);
                    Ga[s] = fmaf(g4.x, a4.x, Ga[s]); Ga[s] = fmaf(g4.y, a4.y, Ga[s]);
                    Ga[s] = fmaf(g4.z, a4.z, Ga[s]); Ga[s] = fmaf(g4.w, a4.w, Ga[s]);
                    if (4 * c < 8 * s + 8) {
                        m[s][4 * c + 0] = g4.x; m[s][4 * c + 1] = g4.y; m[s][4 * c + 2] = g4.z; m[s][4 * c + 3] = g4.w;
                    }
                }
            }
            // ---- residuals and stopping rule (per pixel group)
            float rdm = 0.0f, sa = 0.0f, gp = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                w[s] = Ga[s] - b[s] + nu;
                rdm = fmaxf(rdm, fabsf(w[s] - lam[s]));
                sa += a[s];
                gp = fmaf(a[s], lam[s], gp);
            }
            rdm = gmax(rdm); sa = gsum(sa); gp = gsum(gp);
            const float rp = sa - 1.0f;
            if (!done) {
                if (gp <= prm.gap_tol * sc && rdm <= prm.feas_tol * sc && fabsf(rp) <= prm.feas_tol) {
                    done = true; flags |= LINMIN_INFO_CONVERGED;
                } else if (it >= prm.max_iter) {
                    done = true; flags |= LINMIN_INFO_MAX_ITER;
                }
            }
            if (__all_sync(FULL, done)) break;
            if (!done) ++iters;
            const float mu = gp * (1.0f / 32.0f);

            // ---- M = G + diag(lambda / a); upper part of the diagonal blocks := 0
            float ainv[4], d[4], dinv[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                ainv[s] = rcp_approx(a[s]);
                d[s] = lam[s] * ainv[s];
                dinv[s] = 0.0f;
#pragma unroll
                for (int jj = 0; jj < 8; ++jj) {
                    float v = m[s][8 * s + jj];
                    v = (jj == t) ? v + d[s] : v;
                    m[s][8 * s + jj] = (jj <= t) ? v : 0.0f;
                }
            }
            // ---- Cholesky, right-looking, column broadcast through shared memory
            bool clamped = false;
#pragma unroll
            for (int k = 0; k < 32; ++k) {
                const int s0 = k >> 3, t0 = k & 7;
                float *cb = (k & 1) ? xe : xo;       // alternate lines: no WAR hazard with one sync per step
                float piv = __shfl_sync(FULL, m[s0][k], t0, 8);
                if (!(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
                float rinv = rsqrtf(piv);
                float lcol[4];
#pragma unroll
                for (int s = s0; s < 4; ++s) {
                    // slot s0: rows above k hold 0 (stay 0), row k itself becomes L_kk
                    lcol[s] = m[s][k] * rinv;
                    m[s][k] = lcol[s];
                    cb[t + 8 * s] = lcol[s];
                }
                dinv[s0] = (t == t0) ? rinv : dinv[s0];
                if (k == 31) break;
                __syncwarp();
                // rows of slot s0 at or above k must not be touched by the update
                float lrow0 = (t > t0) ? lcol[s0] : 0.0f;
#pragma unroll
                for (int c = (k + 1) >> 2; c < 8; ++c) {
                    float4 l4 = *reinterpret_cast<const float4 *>(cb + 4 * c);
                    const float lj[4] = {l4.x, l4.y, l4.z, l4.w};
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int j = 4 * c + q;
                        if (j > k) {
#pragma unroll
                            for (int s = s0; s < 4; ++s) {
                                if (j < 8 * s + 8) {
                                    float li = (s == s0) ? lrow0 : lcol[s];
                                    m[s][j] = fmaf(-li, lj[q], m[s][j]);
                                }
                            }
                        }
                    }
                }
            }
            if (clamped) flags |= LINMIN_INFO_CHOL_REGULARISED;
            // the in-block upper entries were updated with li = 0 only for rows <= k of slot s0 at
            // step k; entries (i, j), j > i, of LATER steps k < i still received updates: clear them
#pragma unroll
            for (int s = 0; s < 4; ++s)
#pragma unroll
                for (int jj = 1; jj < 8; ++jj) m[s][8 * s + jj] = (jj <= t) ? m[s][8 * s + jj] : 0.0f;

            // ---- predictor: w1 = L^-1 1, z = L^-1 (-w)
            float r2[2][4];
#pragma unroll
            for (int s = 0; s < 4; ++s) { r2[0][s] = 1.0f; r2[1][s] = -w[s]; }
            forward_subst<2>(m, dinv, r2, t);
            float sww = 0.0f, swz = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) { sww = fmaf(r2[0][s], r2[0][s], sww); swz = fmaf(r2[0][s], r2[1][s], swz); }
            sww = gsum(sww); swz = gsum(swz);
            const float rsww = 1.0f / sww;
            float dnu = (swz + rp) * rsww;
            float zz[4], da[4], dl[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) zz[s] = fmaf(-r2[0][s], dnu, r2[1][s]);
            backward_subst(m, dinv, zz, da, t);
            float mp = 0.0f, md = 0.0f;     // max of -da/a and -dl/lambda
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                dl[s] = -lam[s] - d[s] * da[s];
                mp = fmaxf(mp, -da[s] * ainv[s]);
                md = fmaxf(md, 1.0f + ainv[s] * da[s]);       // -dl/lambda = 1 + da/a
            }
            mp = gmax(mp); md = gmax(md);
            float ap = (mp > 1.0f) ? rcp_approx(mp) : 1.0f;
            float ad = (md > 1.0f) ? rcp_approx(md) : 1.0f;
            float mua = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) mua = fmaf(fmaf(ap, da[s], a[s]), fmaf(ad, dl[s], lam[s]), mua);
            mua = gsum(mua) * (1.0f / 32.0f);
            float sg = mua / mu;
            sg = fminf(1.0f, fmaxf(0.0f, sg * sg * sg));
            // ---- corrector
            float cc[4], r1[1][4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                cc[s] = fmaf(sg, mu, -da[s] * dl[s]);
                r1[0][s] = fmaf(cc[s], ainv[s], -w[s]);
            }
            forward_subst<1>(m, dinv, r1, t);
            swz = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) swz = fmaf(r2[0][s], r1[0][s], swz);
            swz = gsum(swz);
            dnu = (swz + rp) * rsww;
#pragma unroll
            for (int s = 0; s < 4; ++s) zz[s] = fmaf(-r2[0][s], dnu, r1[0][s]);
            backward_subst(m, dinv, zz, da, t);
            mp = 0.0f; md = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                dl[s] = fmaf(cc[s], ainv[s], -lam[s]) - d[s] * da[s];
                mp = fmaxf(mp, -da[s] * ainv[s]);
                md = fmaxf(md, -dl[s] * rcp_approx(lam[s]));
            }
            mp = gmax(mp); md = gmax(md);
            ap = (tau < mp) ? tau * rcp_approx(mp) : 1.0f;     // min(1, tau / mp)
            ad = (tau < md) ? tau * rcp_approx(md) : 1.0f;
            if (done) { ap = 0.0f; ad = 0.0f; }                // converged pixels ride along unchanged
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                a[s] = fmaxf(fmaf(ap, da[s], a[s]), 1e-18f);
                lam[s] = fmaxf(fmaf(ad, dl[s], lam[s]), 1e-18f * lam0);
            }
            nu = fmaf(ad, dnu, nu);
        }

        // ---- store the iterate (coalesced: 8 lanes x float4 = one 128 B row) and the info word
        __syncwarp();
#pragma unroll
        for (int s = 0; s < 4; ++s) xb0[t + 8 * s] = a[s];
        __syncwarp();
        if (valid) {
            float4 o = *reinterpret_cast<const float4 *>(xb0 + 4 * t);
            *reinterpret_cast<float4 *>(prm.coeffs + p * R + 4 * t) = o;
            if (prm.info && t == 0) prm.info[p] = flags | (iters << 8);
        }
        __syncwarp();
    }
}

inline bool ipls_r32_supported(int L) {
    return r32::smem_floats(L) * sizeof(float) <= 200 * 1024;
}

// counter: device word, zero (the caller clears it on the stream before the launch)
inline cudaError_t launch_ipls_r32(const LibView &lv, const SolveParams &prm, int sm_count,
                                   unsigned int *counter, cudaStream_t stream) {
    size_t smem = r32::smem_floats(lv.L) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(ipls_r32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, ipls_r32_kernel, r32::WARPS * 32, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) occ = 1;
    int64_t groups = (prm.N + 3) / 4;
    int64_t need = (groups + r32::WARPS - 1) / r32::WARPS;
    int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, (int64_t)sm_count * occ));
    ipls_r32_kernel<<<grid, r32::WARPS * 32, smem, stream>>>(lv, prm, counter);
    return cudaGetLastError();
}

}  // namespace linmin
