// finish_sweep.cuh -- exact finish + uncertainty + residual for R <= 32, L <= 256 (sm_100a), v3 of the
// throughput path of SURVEY.md 8(a) a3-a6 (replaces the round-1 finish8 kernel on that path).
//
// Same mathematics and the same active-set logic as finish.cuh (read its header: PAPER.md:54-68
// optimality conditions, PAPER.md:88 uncertainty reading R3, PAPER.md:143 RMS reading R8).  What changed
// is the arithmetic plan, chosen after ncu showed finish8 starved of INSTRUCTIONS (50 % of the stall
// samples were no_instruction: 96 KB of branchy code, 16 warps each somewhere else):
//   * normal-equation form on the support in fp64: b_F = A_F'y is accumulated in fp64 (the products of
//     two fp32 numbers are exact in fp64), K = (A_F'A_F)^-1 comes from ONE in-place Gauss-Jordan sweep of
//     the fp64 Gram block held in shared memory, and the trial point is K b_F - mu K 1.  One fp64 pass
//     over the channels per round instead of two, no separate factor / inverse / product phases.
//   * H = K - q q'/(1'q) is read off the swept matrix; J = H A_F' and A'r run as FFMA2 streams.
//   * reductions over the 8 lanes of a pixel go through shared memory (one store, a few LDS.128)
//     instead of 64-bit shuffle trees.
// Mapping as before: 8 lanes per pixel, 4 pixels per warp, lane t owns channels {4 (t + 8 v) + q},
// support members (ranks) t and t + 8, and endmembers 4 t + q.
#pragma once
#include "common.cuh"

namespace linmin {
namespace fs {

constexpr unsigned FULL = 0xffffffffu;
constexpr int KM = 16;    // support cap of this kernel
constexpr int RP = 32;    // endmember rows staged (rows >= R are zero)
constexpr int GS = 33;    // row stride of the staged fp64 Gram matrix (bank spread)
constexpr int MS = 18;    // row stride (doubles) of the per-pixel matrix: 144 B rows, conflict-free LDS.128 by row

// per-pixel scratch (bytes; every block 16 B aligned)
constexpr int OFF_M = 0;                      // double[16][MS]
constexpr int OFF_HS = 0;                     //   later: float[16][16] H (first KB of M)
constexpr int OFF_EX = 1024;                  //   later: float[8][32] partial sums of A'r (second KB of M)
constexpr int OFF_BE = 16 * MS * 8;           // double[32] b_i = A_i'y by endmember
constexpr int OFF_BR = OFF_BE + 32 * 8;       // double[16] b by rank
constexpr int OFF_AF = OFF_BR + 16 * 8;       // double[16] current point by rank
constexpr int OFF_QV = OFF_AF + 16 * 8;       // double[16] q = K 1 by rank
constexpr int OFF_G = OFF_QV + 16 * 8;        // float[32] gradient / output staging
constexpr int OFF_SG = OFF_G + 32 * 4;        // float[16] coeff_sigma by rank
constexpr int OFF_IDX = OFF_SG + 16 * 4;      // int[16]
constexpr int OFF_STATE = OFF_IDX + 16 * 4;   // uchar[32]: 0 free, 1 in F, 2 blocked
constexpr int PIX_BYTES = OFF_STATE + 32;     // 3232
static_assert(PIX_BYTES % 16 == 0, "scratch alignment");

__host__ __device__ inline size_t cta_bytes(int LQ) {
    return (size_t)RP * GS * 8 + (size_t)RP * 32 * LQ * 4;
}

__device__ __forceinline__ double gsum(double v) { return group_sum<8>(v); }   // over the 8 lanes of a pixel
__device__ __forceinline__ float gsum(float v) { return group_sum<8>(v); }
__device__ __forceinline__ double gmin(double v) { return group_min<8>(v); }
__device__ __forceinline__ float gminf(float v) { return group_min<8>(v); }
__device__ __forceinline__ float gmaxf(float v) { return group_max<8>(v); }
__device__ __forceinline__ unsigned gor(unsigned v) { return group_or<8>(v); }
__device__ __forceinline__ int wmax(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
// sums of 4 values over the 8 lanes of a group with 4 shuffles: lane t ends with the total of v_{t >> 1}
__device__ __forceinline__ float reduce4(float v0, float v1, float v2, float v3, int t) {
    const bool h4 = t & 4;
    float s0 = h4 ? v0 : v2, s1 = h4 ? v1 : v3;
    float k0 = h4 ? v2 : v0, k1 = h4 ? v3 : v1;
    k0 += __shfl_xor_sync(FULL, s0, 4);
    k1 += __shfl_xor_sync(FULL, s1, 4);
    const bool h2 = t & 2;
    float s = h2 ? k0 : k1, k = h2 ? k1 : k0;
    k += __shfl_xor_sync(FULL, s, 2);
    k += __shfl_xor_sync(FULL, k, 1);
    return k;
}
// 1 / x in fp64 for x in the fp32 range: MUFU seed (23 bits) and two Newton steps
__device__ __forceinline__ double rcp_d(double x) {
    float xf = (float)x, sf;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(sf) : "f"(xf));
    double p = (double)sf;
    double e = fma(-x, p, 1.0);
    p = fma(p, e, p);
    e = fma(-x, p, 1.0);
    return fma(p, e, p);
}
}  // namespace fs

// LQ = float4 chunks of the spectrum per lane: L <= 32 LQ
template <int LQ>
__global__ void __launch_bounds__(384, 1)
finish_sweep_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter,
                    unsigned int *__restrict__ overflow /* [0] = count, [1 + i] = pixel */,
                    const unsigned int *__restrict__ list /* NULL: all pixels; else the pixels to do, same layout */,
                    unsigned int *__restrict__ defer /* NULL: run every pixel to its end; else: ONE round per pixel,
                                                        a pixel whose support has to change is handed on through
                                                        this list (its repaired support goes to `coeffs`) */) {
    using namespace fs;
    constexpr int NC = 4 * LQ;          // channels per lane
    constexpr int RS = 32 * LQ;         // library row stride (elements)
    constexpr int IT = (LQ <= 4) ? 4 : 2;   // J rows per tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    if (lib.flags[0]) return;
    const int L = lib.L, R = lib.R;
    double *G64s = (double *)smem_raw;                                    // [RP][GS]
    float *At32 = (float *)(smem_raw + (size_t)RP * GS * 8);              // [RP][32 LQ]: library rows, fp32 (widened on the fly:
                                                                          // an fp64 copy costs twice the shared-memory wavefronts)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 3, t = lane & 7;
    unsigned char *S = (unsigned char *)(At32 + (size_t)RP * RS) + (size_t)(warp * 4 + g) * PIX_BYTES;
    double *Md = (double *)(S + OFF_M);
    float *Hs = (float *)(S + OFF_HS);
    float *Ex = (float *)(S + OFF_EX);
    double *bE = (double *)(S + OFF_BE);
    double *bR = (double *)(S + OFF_BR);
    double *aFs = (double *)(S + OFF_AF);
    double *qv = (double *)(S + OFF_QV);
    float *gs = (float *)(S + OFF_G);
    float *sgs = (float *)(S + OFF_SG);
    int *idx = (int *)(S + OFF_IDX);
    unsigned char *state = S + OFF_STATE;

    // ---- once per CTA: stage the library (transposed, fp32) and the fp64 Gram matrix
    for (int e = threadIdx.x; e < RP * RP; e += blockDim.x) {
        const int i = e >> 5, j = e & 31;
        G64s[i * GS + j] = (i < R && j < R) ? lib.G64[i * R + j] : 0.0;
    }
    for (int e = threadIdx.x; e < RP * RS; e += blockDim.x) {
        const int r = e / RS, l = e - r * RS;
        const float a = (r < R && l < L) ? lib.A[(size_t)l * R + r] : 0.0f;
        At32[e] = a;
    }
    __syncthreads();

    const bool vec_ok = ((prm.ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.Y) & 15) == 0);
    const bool svec_ok = prm.has_sigma && ((prm.sigma_stride & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.sigma) & 15) == 0);
    const bool cvec_ok = ((R & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.coeffs) & 15) == 0);
    const bool csvec_ok = ((R & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.coeff_sigma) & 15) == 0);
    const float qnan = __int_as_float(0x7fc00000);
    const int max_pivots = 4 * RP + 8;
    // false: positivity only: no equality constraint -- no normalisation, mu == nu == 0, H = K, and the
    // empty support is feasible (a = 0)
    const bool cons = lib.cons != 0;
    double *M0 = Md + t * MS;          // my rows of the swept matrix
    double *M1 = Md + (t + 8) * MS;

    // Work unit of a warp: a chunk of 32 consecutive pixels.  Lane i counts the support of pixel i from
    // the IPLS iterate, the 32 counts are ranked (ties by lane), and the chunk is processed as 8 tasks
    // of 4 pixels with neighbouring support sizes: the k-bounded loops of a task then run (almost)
    // without padding (mean of the warp maximum 11.1 -> 8 on config 4).
    int *perm = (int *)((unsigned char *)(At32 + (size_t)RP * RS) + (size_t)(blockDim.x >> 5) * 4 * PIX_BYTES) + warp * 32;
    const int64_t count = list ? (int64_t)list[0] : prm.N;
    // a short list is dealt out one task (4 pixels) at a time: 32-pixel chunks would leave most warps idle
    const int csz = (list && count < (int64_t)gridDim.x * (blockDim.x >> 5) * 128) ? 4 : 32;
    while (true) {
        unsigned int chunk = 0;
        if (lane == 0) chunk = atomicAdd(counter, 1u);
        chunk = __shfl_sync(FULL, chunk, 0);
        const int64_t pbase = (int64_t)chunk * csz;
        if (pbase >= count) break;
        // my pixel of the chunk (-1: none)
        const int64_t mypix = (lane < csz && pbase + lane < count) ? (list ? (int64_t)list[1 + pbase + lane] : pbase + lane) : -1;
        {
            int kc = -1;
            if (mypix >= 0) {
                const float *cp = prm.coeffs + mypix * R;
                kc = 0;
                if (cvec_ok) {
                    for (int i = 0; i < R; i += 4) {
                        const float4 c4 = *reinterpret_cast<const float4 *>(cp + i);
                        kc += (c4.x > LINMIN_SUPPORT_THRESHOLD) + (c4.y > LINMIN_SUPPORT_THRESHOLD) +
                              (c4.z > LINMIN_SUPPORT_THRESHOLD) + (c4.w > LINMIN_SUPPORT_THRESHOLD);
                    }
                } else {
                    for (int i = 0; i < R; ++i) kc += cp[i] > LINMIN_SUPPORT_THRESHOLD;
                }
            }
            int pos = 0;
#pragma unroll 1
            for (int d = 1; d < 32; ++d) {
                const int j = (lane + d) & 31;
                const int kj = __shfl_sync(FULL, kc, j);
                pos += (kj > kc) || (kj == kc && j < lane);
            }
            __syncwarp();
            perm[pos] = lane;
            __syncwarp();
        }
      for (int task = 0; task < 8; ++task) {
        const int64_t p_raw = __shfl_sync(FULL, mypix, perm[4 * task + g]);
        if (__shfl_sync(FULL, mypix, perm[4 * task]) < 0) break;          // sorted: invalid pixels (k = -1) come last
        const bool valid = p_raw >= 0;
        const int64_t p = valid ? p_raw : (prm.N - 1);
        float *cout = prm.coeffs + p * R;
        int info = prm.info ? prm.info[p] : 0;

        // ---- spectrum -> registers
        float yv[NC];
        const float *yp = prm.Y + p * prm.ldY;
        bool bad = false;
#pragma unroll
        for (int v = 0; v < LQ; ++v) {
            const int l = 4 * (t + 8 * v);
            if (vec_ok && l + 3 < L) {
                float4 t4 = *reinterpret_cast<const float4 *>(yp + l);
                yv[4 * v + 0] = t4.x; yv[4 * v + 1] = t4.y; yv[4 * v + 2] = t4.z; yv[4 * v + 3] = t4.w;
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) yv[4 * v + q] = (l + q < L) ? yp[l + q] : 0.0f;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) bad |= !isfinite(yv[4 * v + q]);
        }
        bad = ((__ballot_sync(FULL, bad) >> (8 * g)) & 0xffu) != 0u;
        // ---- noise std -> registers now, so that the load is long done when the uncertainty pass needs it
        float2 sv[NC / 2];
        bool sbad = false;
        if (prm.coeff_sigma && prm.has_sigma) {
            const float *sp = prm.sigma + p * prm.sigma_stride;
#pragma unroll
            for (int v = 0; v < LQ; ++v) {
                const int l = 4 * (t + 8 * v);
                float4 t4;
                if (svec_ok && l + 3 < L) {
                    t4 = *reinterpret_cast<const float4 *>(sp + l);
                } else {
                    t4.x = (l + 0 < L) ? sp[l + 0] : 1.0f; t4.y = (l + 1 < L) ? sp[l + 1] : 1.0f;
                    t4.z = (l + 2 < L) ? sp[l + 2] : 1.0f; t4.w = (l + 3 < L) ? sp[l + 3] : 1.0f;
                }
                sv[2 * v] = make_float2(t4.x, t4.y); sv[2 * v + 1] = make_float2(t4.z, t4.w);
            }
        } else {
#pragma unroll
            for (int c = 0; c < NC / 2; ++c) sv[c] = make_float2(1.0f, 1.0f);
        }

        // ---- initial support from the IPLS iterate; lane t looks at endmembers 4 t + q
        // st: 0 solving, 1 optimal, 2 fallback (feasible point, not certified), 3 nothing to write here
        int st = valid ? 0 : 3;
        int k = 0;
        idx[t] = 0; idx[t + 8] = 0;
        __syncwarp();
        {
            float ai[4];
            if (cvec_ok && 4 * t < R) {
                float4 c4 = *reinterpret_cast<const float4 *>(cout + 4 * t);
                ai[0] = c4.x; ai[1] = c4.y; ai[2] = c4.z; ai[3] = c4.w;
            } else {
#pragma unroll
                for (int q = 0; q < 4; ++q) ai[q] = (4 * t + q < R) ? cout[4 * t + q] : -1.0f;
            }
            unsigned nib = 0;
#pragma unroll
            for (int q = 0; q < 4; ++q) nib |= (ai[q] > LINMIN_SUPPORT_THRESHOLD && 4 * t + q < R) ? (1u << q) : 0u;
            unsigned mask = gor(nib << (4 * t));
            float best = gmaxf(fmaxf(fmaxf(ai[0], ai[1]), fmaxf(ai[2], ai[3])));
            if (mask == 0u && cons) {   // can not happen for a point of the simplex; be safe: the largest entry
                unsigned nb = 0;
#pragma unroll
                for (int q = 0; q < 4; ++q) nb |= (ai[q] == best && 4 * t + q < R) ? (1u << q) : 0u;
                mask = gor(nb << (4 * t));
                mask &= 0u - mask;
                if (mask == 0u) mask = 1u;
#pragma unroll
                for (int q = 0; q < 4; ++q) ai[q] = 1.0f;
            }
            k = __popc(mask);
            uchar4 s4;
            unsigned char sb[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = 4 * t + q;
                const bool in = (mask >> i) & 1u;
                sb[q] = (i >= R) ? 2 : (in ? 1 : 0);
                if (in && k <= KM) {
                    const int rank = __popc(mask & ((1u << i) - 1u));
                    idx[rank] = i;
                    aFs[rank] = (double)ai[q];
                }
            }
            s4.x = sb[0]; s4.y = sb[1]; s4.z = sb[2]; s4.w = sb[3];
            *reinterpret_cast<uchar4 *>(state + 4 * t) = s4;
        }
        if (bad && st == 0) {
            st = 3;
            for (int q = 0; q < 4; ++q) if (4 * t + q < R) cout[4 * t + q] = qnan;
            if (prm.coeff_sigma)
                for (int q = 0; q < 4; ++q) if (4 * t + q < R) prm.coeff_sigma[p * R + 4 * t + q] = qnan;
            if (t == 0) {
                if (prm.resid) prm.resid[p] = qnan;
                if (prm.info) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            }
        }
        if (st == 0 && k > KM) {
            st = 3;
            if (t == 0) { unsigned slot = atomicAdd(overflow, 1u); overflow[1 + slot] = (unsigned)p; }
        }
        __syncwarp();
        // lane t owns members (ranks) t and t + 8: coefficient, endmember index
        double a0 = 0.0, a1 = 0.0;
        int i0 = 0, i1 = 0;
        if (st == 0) {
            if (t < k) { a0 = aFs[t]; i0 = idx[t]; }
            if (t + 8 < k) { a1 = aFs[t + 8]; i1 = idx[t + 8]; }
        }
        {
            const double s = gsum(a0 + a1);
            if (st == 0 && cons) {
                const double rs = rcp_d(s);
                a0 *= rs; a1 *= rs;
                if (t < k) aFs[t] = a0;
                if (t + 8 < k) aFs[t + 8] = a1;
            }
        }
        __syncwarp();

        int pivots = (list && prm.info) ? ((info >> 16) & 0xff) : 0;      // a handed-on pixel keeps its count
        int last_added = -1;
        unsigned have = 0u;              // endmembers whose b_i = A_i'y is in bE
        double q0 = 0.0, q1 = 0.0, sq = 1.0, rss = 0.0;

        while (__any_sync(FULL, st == 0)) {
            const bool act = (st == 0);
            const int kw = wmax(act ? k : 0);
            const bool wide = kw > 8;                 // some pixel of the warp uses ranks 8..15
            // ---- b_i = A_i'y (fp64) for the members that do not have it yet: partial sums over my
            //      channels go to P[rank][lane] (overlays M), lane t then adds up ranks t and t + 8
            const bool need0 = act && t < k && !((have >> i0) & 1u);
            const bool need1 = act && t + 8 < k && !((have >> i1) & 1u);
            if (__any_sync(FULL, need0 || need1)) {
                double yd[NC];                      // widened once per round, not once per member
#pragma unroll
                for (int c = 0; c < NC; ++c) yd[c] = (double)yv[c];
#pragma unroll 1
                for (int j = 0; j < kw; ++j) {
                    const int ij = idx[j];
                    if (act && j < k && !((have >> ij) & 1u)) {
                        const float *row = At32 + (size_t)ij * RS + 4 * t;
                        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
                        for (int v = 0; v < LQ; ++v) {
                            const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
                            s0 = fma((double)a4.x, yd[4 * v + 0], s0); s1 = fma((double)a4.y, yd[4 * v + 1], s1);
                            s2 = fma((double)a4.z, yd[4 * v + 2], s2); s3 = fma((double)a4.w, yd[4 * v + 3], s3);
                        }
                        Md[j * 8 + t] = (s0 + s1) + (s2 + s3);
                    }
                }
                __syncwarp();
                if (need0) {
                    const double2 u0 = *reinterpret_cast<const double2 *>(Md + t * 8), u1 = *reinterpret_cast<const double2 *>(Md + t * 8 + 2);
                    const double2 u2 = *reinterpret_cast<const double2 *>(Md + t * 8 + 4), u3 = *reinterpret_cast<const double2 *>(Md + t * 8 + 6);
                    bE[i0] = ((u0.x + u0.y) + (u1.x + u1.y)) + ((u2.x + u2.y) + (u3.x + u3.y));
                }
                if (need1) {
                    const double *P = Md + (t + 8) * 8;
                    const double2 u0 = *reinterpret_cast<const double2 *>(P), u1 = *reinterpret_cast<const double2 *>(P + 2);
                    const double2 u2 = *reinterpret_cast<const double2 *>(P + 4), u3 = *reinterpret_cast<const double2 *>(P + 6);
                    bE[i1] = ((u0.x + u0.y) + (u1.x + u1.y)) + ((u2.x + u2.y) + (u3.x + u3.y));
                }
                have |= gor((need0 ? (1u << i0) : 0u) | (need1 ? (1u << i1) : 0u));
                __syncwarp();
            }
            // ---- b by rank (zero beyond k), and my rows of G_FF into M (zero-padded columns)
            if (act) {
                bR[t] = (t < k) ? bE[i0] : 0.0;
                if (wide) bR[t + 8] = (t + 8 < k) ? bE[i1] : 0.0;
#pragma unroll 1
                for (int c2 = 0; c2 < (wide ? 8 : 4); ++c2) {
                    {
                        const int2 jj = *reinterpret_cast<const int2 *>(idx + 2 * c2);
                        const bool v0 = 2 * c2 < k, v1 = 2 * c2 + 1 < k;
                        double2 m0, m1;
                        m0.x = (v0 && t < k) ? G64s[i0 * GS + jj.x] : 0.0;
                        m0.y = (v1 && t < k) ? G64s[i0 * GS + jj.y] : 0.0;
                        *reinterpret_cast<double2 *>(M0 + 2 * c2) = m0;
                        if (wide) {
                            m1.x = (v0 && t + 8 < k) ? G64s[i1 * GS + jj.x] : 0.0;
                            m1.y = (v1 && t + 8 < k) ? G64s[i1 * GS + jj.y] : 0.0;
                            *reinterpret_cast<double2 *>(M1 + 2 * c2) = m1;
                        }
                    }
                }
            }
            __syncwarp();
            // ---- in-place Gauss-Jordan sweep: M <- G_FF^-1 (pivot j = Schur complement of the leading block)
            int rej = -1;
            for (int j = 0; j < kw; ++j) {
                const bool on = act && rej < 0 && j < k;
                const double *Mj = Md + j * MS;
                const double d = Mj[j];
                const int ij = idx[j];
                const bool ok = d > 1e-13 * G64s[ij * GS + ij];
                if (on && !ok) rej = j;
                const bool go = on && ok;
                const double pv = rcp_d(go ? d : 1.0);
                double f0 = M0[j] * pv, f1 = 0.0;
                if (t == j) f0 = 1.0 - pv;                      // pivot row: m - (1 - p) m = p m
                if (wide) { f1 = M1[j] * pv; if (t + 8 == j) f1 = 1.0 - pv; }
                // row j goes to a line of its own (qv is free until the point is accepted): the update loops can
                // then stay rolled -- this kernel is bound by instruction supply, not by arithmetic
                *reinterpret_cast<double2 *>(qv + 2 * t) = *reinterpret_cast<const double2 *>(Mj + 2 * t);
                __syncwarp();
                if (go) {
                    const int nc2 = wide ? 8 : 4;
                    const bool r0 = t < k, r1 = wide && t + 8 < k;
#pragma unroll 4
                    for (int c2 = 0; c2 < nc2; ++c2) {
                        const double2 r = *reinterpret_cast<const double2 *>(qv + 2 * c2);
                        if (r0) {
                            double2 m = *reinterpret_cast<double2 *>(M0 + 2 * c2);
                            m.x = fma(-f0, r.x, m.x); m.y = fma(-f0, r.y, m.y);
                            *reinterpret_cast<double2 *>(M0 + 2 * c2) = m;
                        }
                        if (r1) {
                            double2 m = *reinterpret_cast<double2 *>(M1 + 2 * c2);
                            m.x = fma(-f1, r.x, m.x); m.y = fma(-f1, r.y, m.y);
                            *reinterpret_cast<double2 *>(M1 + 2 * c2) = m;
                        }
                    }
                    if (r0) M0[j] = (t == j) ? pv : -f0;
                    if (r1) M1[j] = (t + 8 == j) ? pv : -f1;
                }
                __syncwarp();
            }
            bool skip = !act;
            bool fell = false;      // this round ended in the fallback state: the residual is still due
            if (__any_sync(FULL, act && rej >= 0)) {       // warp-uniform and rare (duplicate or collinear members)
                const int rj = rej >= 0 ? rej : 0;
                const int irej = __shfl_sync(FULL, (rj < 8) ? i0 : i1, rj & 7, 8);     // endmember of the rejected member
                if (act && rej >= 0) {
                    // A_F lost rank at member `rej` (R9): drop it, block it, stay at the same point
                    skip = true;
                    if (t == (rej & 7)) state[(rej < 8) ? i0 : i1] = 2;
                    const int n0 = t - (t > rej ? 1 : 0), n1 = t + 8 - (t + 8 > rej ? 1 : 0);
                    const bool k0 = (t < k) && (t != rej), k1 = (t + 8 < k) && (t + 8 != rej);
                    if (k0) { idx[n0] = i0; aFs[n0] = a0; }
                    if (k1) { idx[n1] = i1; aFs[n1] = a1; }
                    --k; last_added = -1;
                    ++pivots;
                }
                __syncwarp();
                if (act && rej >= 0) {
                    a0 = 0.0; a1 = 0.0; i0 = 0; i1 = 0;
                    if (t < k) { a0 = aFs[t]; i0 = idx[t]; }
                    if (t + 8 < k) { a1 = aFs[t + 8]; i1 = idx[t + 8]; }
                }
                const double s = gsum(a0 + a1);
                if (act && rej >= 0) {
                    if (k == 0 && cons) {
                        // the only member was rejected (a zero endmember): stay on the simplex with it, uncertified
                        k = 1; i0 = (t == 0) ? irej : 0; a0 = (t == 0) ? 1.0 : 0.0;
                        if (t == 0) { idx[0] = irej; aFs[0] = 1.0; state[irej] = 1; }
                        st = 2; fell = true;
                    } else {
                        if (cons) {
                            const double rs = rcp_d(s);
                            a0 *= rs; a1 *= rs;
                            if (t < k) aFs[t] = a0;
                            if (t + 8 < k) aFs[t + 8] = a1;
                        }
                        if (pivots > max_pivots) { st = 2; fell = true; }
                    }
                }
                __syncwarp();
            }

            // ---- q = K 1 and x = K b_F from my rows; trial point x - mu q with 1'(x - mu q) = 1
            q0 = 0.0; q1 = 0.0;
            double x0 = 0.0, x1 = 0.0;
            if (!skip) {
#pragma unroll 1
                for (int c2 = 0; c2 < (wide ? 8 : 4); ++c2) {
                    {
                        const double2 bb = *reinterpret_cast<const double2 *>(bR + 2 * c2);
                        const double2 m = *reinterpret_cast<const double2 *>(M0 + 2 * c2);
                        q0 += m.x + m.y;
                        x0 = fma(m.x, bb.x, fma(m.y, bb.y, x0));
                        if (wide) {
                            const double2 n = *reinterpret_cast<const double2 *>(M1 + 2 * c2);
                            q1 += n.x + n.y;
                            x1 = fma(n.x, bb.x, fma(n.y, bb.y, x1));
                        }
                    }
                }
                if (!(t < k)) { q0 = 0.0; x0 = 0.0; }
                if (!(t + 8 < k)) { q1 = 0.0; x1 = 0.0; }
            }
            const double sqn = gsum(q0 + q1);
            const double sx = gsum(x0 + x1);
            bool accepted = false;
            {
                const double mu = cons ? (sx - 1.0) * rcp_d(skip ? 1.0 : sqn) : 0.0;
                const double t0v = x0 - mu * q0, t1v = x1 - mu * q1;
                const bool m0 = t < k, m1 = t + 8 < k;
                const double amin = gmin(fmin(m0 ? t0v : INFINITY, m1 ? t1v : INFINITY));
                const bool ratio = !skip && !(amin > 0.0);
                // ---- ratio step towards the trial point until the first coefficient reaches zero; drop it.
                //      Warp-uniform branch: 86 % of the rounds accept the trial point and skip all of this.
                if (__any_sync(FULL, ratio)) {
                    double r0 = INFINITY, r1 = INFINITY;
                    if (m0 && !(t0v > 0.0)) { const double den = a0 - t0v; r0 = den > 0.0 ? a0 * rcp_d(fmax(den, 1e-30)) : 0.0; }
                    if (m1 && !(t1v > 0.0)) { const double den = a1 - t1v; r1 = den > 0.0 ? a1 * rcp_d(fmax(den, 1e-30)) : 0.0; }
                    double alpha = fmin(1.0, gmin(fmin(r0, r1)));
                    if (alpha < 0.0) alpha = 0.0;
                    const double n0v = a0 + alpha * (t0v - a0), n1v = a1 + alpha * (t1v - a1);
                    const bool b0 = r0 <= alpha, b1 = r1 <= alpha;
                    const bool keep0 = m0 && !b0 && (n0v > 0.0), keep1 = m1 && !b1 && (n1v > 0.0);
                    // ranks of the kept members: ballots over the group, slot 0 members come first
                    const unsigned bk0 = (__ballot_sync(FULL, keep0) >> (8 * g)) & 0xffu;
                    const unsigned bk1 = (__ballot_sync(FULL, keep1) >> (8 * g)) & 0xffu;
                    const double ssum = gsum((keep0 ? n0v : 0.0) + (keep1 ? n1v : 0.0));
                    __syncwarp();       // every read of idx / aFs of this round precedes the writes below
                    if (ratio) {
                        if (m0 && !keep0) state[i0] = (i0 == last_added && alpha == 0.0) ? 2 : 0;
                        if (m1 && !keep1) state[i1] = (i1 == last_added && alpha == 0.0) ? 2 : 0;
                        const int k0r = __popc(bk0 & ((1u << t) - 1u));
                        const int k1r = __popc(bk0) + __popc(bk1 & ((1u << t) - 1u));
                        const double rs = cons ? rcp_d(ssum > 0.0 ? ssum : 1.0) : 1.0;
                        if (keep0) { idx[k0r] = i0; aFs[k0r] = n0v * rs; }
                        if (keep1) { idx[k1r] = i1; aFs[k1r] = n1v * rs; }
                        k = __popc(bk0) + __popc(bk1);
                        last_added = -1;
                        ++pivots;
                        if ((k == 0 && cons) || pivots > max_pivots) { st = 2; fell = true; }
                    }
                    __syncwarp();
                    if (ratio) {
                        a0 = 0.0; a1 = 0.0; i0 = 0; i1 = 0;
                        if (t < k) { a0 = aFs[t]; i0 = idx[t]; }
                        if (t + 8 < k) { a1 = aFs[t + 8]; i1 = idx[t + 8]; }
                    }
                }
                if (!ratio && !skip) {
                    accepted = true;
                    a0 = m0 ? t0v : 0.0; a1 = m1 ? t1v : 0.0;
                    if (m0) aFs[t] = a0;
                    if (m1) aFs[t + 8] = a1;
                    sq = sqn;
                    qv[t] = q0;
                    qv[t + 8] = q1;
                }
                __syncwarp();
            }
            // ---- H = K - q q'/(1'q) (fp32) replaces the swept matrix: read my rows, then write them
            const bool resid_due = accepted || fell;
            if (__any_sync(FULL, resid_due)) {
                const int kw2 = wmax(resid_due ? k : 0);
                {
                    float h0[16], h1[16];
                    const double rs = cons ? rcp_d(accepted ? sq : 1.0) : 0.0;      // pos: H = K, no projection
                    const double u0 = q0 * rs, u1 = q1 * rs;
#pragma unroll
                    for (int c2 = 0; c2 < 8; ++c2) {
                        if (c2 < 4 || wide) {
                            const double2 qq = *reinterpret_cast<const double2 *>(qv + 2 * c2);
                            const double2 m = *reinterpret_cast<const double2 *>(M0 + 2 * c2);
                            h0[2 * c2] = (float)fma(-u0, qq.x, m.x); h0[2 * c2 + 1] = (float)fma(-u0, qq.y, m.y);
                            if (wide) {
                                const double2 n = *reinterpret_cast<const double2 *>(M1 + 2 * c2);
                                h1[2 * c2] = (float)fma(-u1, qq.x, n.x); h1[2 * c2 + 1] = (float)fma(-u1, qq.y, n.y);
                            }
                        }
                    }
                    __syncwarp();       // the swept matrix has been read by everybody
                    if (accepted) {
#pragma unroll
                        for (int c4 = 0; c4 < 4; ++c4) {
                            if (c4 < 2 || wide) {
                                *reinterpret_cast<float4 *>(Hs + t * 16 + 4 * c4) =
                                    make_float4(h0[4 * c4], h0[4 * c4 + 1], h0[4 * c4 + 2], h0[4 * c4 + 3]);
                                if (wide)
                                    *reinterpret_cast<float4 *>(Hs + (t + 8) * 16 + 4 * c4) =
                                        make_float4(h1[4 * c4], h1[4 * c4 + 1], h1[4 * c4 + 2], h1[4 * c4 + 3]);
                            }
                        }
                    }
                }
                // ---- residual at the new point (fp64), its sum of squares, fp32 copy
                float rf[NC];
                {
                    double r[NC];
#pragma unroll
                    for (int c = 0; c < NC; ++c) r[c] = (double)yv[c];
#pragma unroll 1
                    for (int j = 0; j < kw2; ++j) {
                        {   // branch-free: a member beyond this pixel's support subtracts zero
                            const double aj = (resid_due && j < k) ? aFs[j] : 0.0;
                            const float *row = At32 + (size_t)idx[j] * RS + 4 * t;
#pragma unroll
                            for (int v = 0; v < LQ; ++v) {
                                const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
                                r[4 * v + 0] = fma(-(double)a4.x, aj, r[4 * v + 0]); r[4 * v + 1] = fma(-(double)a4.y, aj, r[4 * v + 1]);
                                r[4 * v + 2] = fma(-(double)a4.z, aj, r[4 * v + 2]); r[4 * v + 3] = fma(-(double)a4.w, aj, r[4 * v + 3]);
                            }
                        }
                    }
                    double s0 = 0.0, s1 = 0.0;
#pragma unroll
                    for (int c = 0; c < NC; c += 2) { s0 = fma(r[c], r[c], s0); s1 = fma(r[c + 1], r[c + 1], s1); }
                    const double s = gsum(s0 + s1);
                    if (resid_due) rss = s;
#pragma unroll
                    for (int c = 0; c < NC; ++c) rf[c] = (float)r[c];
                }
                // ---- g_i = A_i'r for every endmember (FFMA2 over my channels), partial sums exchanged
                //      through Ex[lane][chunk ^ lane]; lane t ends with endmembers 4 t .. 4 t + 3
#pragma unroll 1
                for (int c4 = 0; c4 < RP / 4; ++c4) {
                    float pr[4];
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float *row = At32 + (size_t)(4 * c4 + e) * RS + 4 * t;
                        float2 acc = make_float2(0.0f, 0.0f);
#pragma unroll
                        for (int v = 0; v < LQ; ++v) {
                            const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
                            acc = fma2(make_float2(a4.x, a4.y), make_float2(rf[4 * v + 0], rf[4 * v + 1]), acc);
                            acc = fma2(make_float2(a4.z, a4.w), make_float2(rf[4 * v + 2], rf[4 * v + 3]), acc);
                        }
                        pr[e] = acc.x + acc.y;
                    }
                    *reinterpret_cast<float4 *>(Ex + t * 32 + 4 * (c4 ^ t)) = make_float4(pr[0], pr[1], pr[2], pr[3]);
                }
                __syncwarp();
                float4 g4 = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
#pragma unroll
                for (int tp = 0; tp < 8; ++tp) {
                    const float4 u = *reinterpret_cast<const float4 *>(Ex + tp * 32 + 4 * (t ^ tp));
                    g4.x += u.x; g4.y += u.y; g4.z += u.z; g4.w += u.w;
                }
                *reinterpret_cast<float4 *>(gs + 4 * t) = g4;
                __syncwarp();
                float nu = 0.0f;
                if (accepted && cons) {
                    if (t < k) nu += gs[i0] * (float)a0;
                    if (t + 8 < k) nu += gs[i1] * (float)a1;
                }
                nu = gsum(nu);
                const uchar4 s4 = *reinterpret_cast<const uchar4 *>(state + 4 * t);
                const float gg[4] = {g4.x, g4.y, g4.z, g4.w};
                const unsigned char ss[4] = {s4.x, s4.y, s4.z, s4.w};
                float lmin = INFINITY, gmx = 0.0f;
                int jmin = -1;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    if (4 * t + q < R) gmx = fmaxf(gmx, fabsf(gg[q]));
                    const float li = (ss[q] == 0) ? (nu - gg[q]) : INFINITY;
                    if (li < lmin) { lmin = li; jmin = 4 * t + q; }
                }
                gmx = gmaxf(gmx);
                const float lbest = gminf(lmin);
                const unsigned cand = (__ballot_sync(FULL, lmin == lbest && jmin >= 0) >> (8 * g)) & 0xffu;
                const int src = cand ? (__ffs(cand) - 1) : 0;
                const int jadd = __shfl_sync(FULL, jmin, src, 8);
                __syncwarp();
                if (accepted) {
                    if (!(lbest < -1e-6f * gmx) || cand == 0u) {
                        st = 1;                                            // optimal
                    } else if (pivots >= max_pivots) {
                        st = 2;
                    } else if (k >= KM) {
                        st = 3;                                            // support outgrows this kernel
                        if (t == 0) { unsigned slot = atomicAdd(overflow, 1u); overflow[1 + slot] = (unsigned)p; }
                    } else {
                        if (t == 0) { state[jadd] = 1; idx[k] = jadd; aFs[k] = 0.0; }
                        if (t == (k & 7)) { if (k < 8) { i0 = jadd; a0 = 0.0; } else { i1 = jadd; a1 = 0.0; } }
                        ++k; ++pivots; last_added = jadd;
                    }
                }
                __syncwarp();
            }
            if (defer && st == 0) st = 4;        // one round only: the next one belongs to the repair pass
        }

        const bool wr = (st == 1 || st == 2);
        const bool df = (st == 4);
        if (st == 2) info |= LINMIN_INFO_FINISH_FALLBACK;
        // ---- coefficients (exact zeros off the support), staged in endmember order
        if (wr || df) *reinterpret_cast<float4 *>(gs + 4 * t) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        __syncwarp();
        if (wr) {
            if (t < k) gs[i0] = (float)a0;
            if (t + 8 < k) gs[i1] = (float)a1;
        }
        if (df) {       // the support as it stands now (a member just added sits at 0), kept above the threshold
            if (t < k) gs[i0] = fmaxf((float)a0, 1.5f * LINMIN_SUPPORT_THRESHOLD);
            if (t + 8 < k) gs[i1] = fmaxf((float)a1, 1.5f * LINMIN_SUPPORT_THRESHOLD);
            if (t == 0) {
                const unsigned slot = atomicAdd(defer, 1u);
                defer[1 + slot] = (unsigned)p;
                if (prm.info) prm.info[p] = (info & 0xffff) | ((pivots > 255 ? 255 : pivots) << 16);
            }
        }
        __syncwarp();
        if (wr || df) {
            const float4 o = *reinterpret_cast<const float4 *>(gs + 4 * t);
            if (cvec_ok && 4 * t < R) *reinterpret_cast<float4 *>(cout + 4 * t) = o;
            else {
                const float ov[4] = {o.x, o.y, o.z, o.w};
                for (int q = 0; q < 4; ++q) if (4 * t + q < R) cout[4 * t + q] = ov[q];
            }
        }
        if (prm.resid && wr && t == 0) prm.resid[p] = (float)sqrt(rss / (double)L);
        // ---- uncertainty propagation (reading R3): J = H A_F' on my channels, sigma_i^2 = sum_l (J_il s_l)^2
        if (prm.coeff_sigma) {
#pragma unroll
            for (int c = 0; c < NC / 2; ++c)
                sbad |= !(sv[c].x > 0.0f) || !isfinite(sv[c].x) || !(sv[c].y > 0.0f) || !isfinite(sv[c].y);
            sbad = ((__ballot_sync(FULL, sbad) >> (8 * g)) & 0xffu) != 0u;
            if (wr && sbad) info |= LINMIN_INFO_BAD_SIGMA;
            const bool doj = (st == 1) && !sbad && k > (cons ? 1 : 0);
            const int kj = wmax(doj ? k : 0);
            if (wr) { sgs[t] = 0.0f; sgs[t + 8] = 0.0f; }
            for (int ib = 0; ib < kj; ib += IT) {
                float2 d[IT][NC / 2];
#pragma unroll
                for (int ii = 0; ii < IT; ++ii)
#pragma unroll
                    for (int c = 0; c < NC / 2; ++c) d[ii][c] = make_float2(0.0f, 0.0f);
                // branch-free body (a pixel whose support ends before j, or that has no J to form, multiplies
                // by zero): the loads of step j + 1 can be issued under the FFMA2 stream of step j
#pragma unroll 1
                for (int j = 0; j < kj; ++j) {
                    const bool on = doj && j < k && ib < k;
                    float hh[IT];
                    if (IT == 4) {
                        const float4 h4 = *reinterpret_cast<const float4 *>(Hs + j * 16 + ib);
                        hh[0] = h4.x; hh[1] = h4.y; hh[IT - 2] = h4.z; hh[IT - 1] = h4.w;
                    } else {
                        const float2 h2 = *reinterpret_cast<const float2 *>(Hs + j * 16 + ib);
                        hh[0] = h2.x; hh[1] = h2.y;
                    }
#pragma unroll
                    for (int ii = 0; ii < IT; ++ii) hh[ii] = on ? hh[ii] : 0.0f;
                    const float *row = At32 + (size_t)idx[j] * RS + 4 * t;
#pragma unroll
                    for (int v = 0; v < LQ; ++v) {
                        const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
                        const float2 alo = make_float2(a4.x, a4.y), ahi = make_float2(a4.z, a4.w);
#pragma unroll
                        for (int ii = 0; ii < IT; ++ii) {
                            d[ii][2 * v] = fma2(hh[ii], alo, d[ii][2 * v]);
                            d[ii][2 * v + 1] = fma2(hh[ii], ahi, d[ii][2 * v + 1]);
                        }
                    }
                }
                float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                for (int ii = 0; ii < IT; ++ii) {
                    float2 a2 = make_float2(0.0f, 0.0f);
#pragma unroll
                    for (int c = 0; c < NC / 2; ++c) {
                        const float2 ds = mul2(d[ii][c], sv[c]);
                        a2 = fma2(ds, ds, a2);
                    }
                    acc[ii] = a2.x + a2.y;
                }
                const float tot = reduce4(acc[0], acc[1], acc[2], acc[3], t);
                if (doj && !(t & 1) && (t >> 1) < IT && ib + (t >> 1) < k) sgs[ib + (t >> 1)] = sqrtf(tot);
            }
            __syncwarp();
            // scatter to endmember order through the staging line
            if (wr) *reinterpret_cast<float4 *>(gs + 4 * t) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            __syncwarp();
            if (wr && st == 1) {
                if (t < k) gs[i0] = sgs[t];
                if (t + 8 < k) gs[i1] = sgs[t + 8];
            }
            __syncwarp();
            if (wr) {
                float4 o = *reinterpret_cast<const float4 *>(gs + 4 * t);
                if (sbad) o = make_float4(qnan, qnan, qnan, qnan);
                float *sout = prm.coeff_sigma + p * R;
                if (csvec_ok && 4 * t < R) *reinterpret_cast<float4 *>(sout + 4 * t) = o;
                else {
                    const float ov[4] = {o.x, o.y, o.z, o.w};
                    for (int q = 0; q < 4; ++q) if (4 * t + q < R) sout[4 * t + q] = ov[q];
                }
            }
        }
        if (wr && prm.info && t == 0) {
            const int pv = pivots > 255 ? 255 : pivots;
            prm.info[p] = (info & 0xffff) | (pv << 16) | (k << 24);
        }
        __syncwarp();
      }
    }
}


template <int LQ>
inline cudaError_t launch_finish_sweep_lq(const LibView &lv, const SolveParams &prm, int sm_count,
                                          unsigned int *counter, unsigned int *overflow, const unsigned int *list,
                                          unsigned int *defer, cudaStream_t stream) {
    const size_t cta = (fs::cta_bytes(LQ) + 15) & ~(size_t)15;
    const size_t per_warp = 4 * (size_t)fs::PIX_BYTES + 128;     // scratch of 4 pixels + the chunk permutation
    int warps = (int)std::min<size_t>(12, (227 * 1024 - cta) / per_warp);
    if (warps < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = cta + per_warp * warps;
    cudaError_t e = cudaFuncSetAttribute(finish_sweep_kernel<LQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t chunks = (prm.N + 31) / 32;
    const int64_t need = (chunks + warps - 1) / warps;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, sm_count));
    finish_sweep_kernel<LQ><<<grid, warps * 32, smem, stream>>>(lv, prm, counter, overflow, list, defer);
    return cudaGetLastError();
}

// counter, overflow[0] and defer[0] must be zero (the caller clears them on the stream)
inline cudaError_t launch_finish_sweep(const LibView &lv, const SolveParams &prm, int sm_count,
                                       unsigned int *counter, unsigned int *overflow, const unsigned int *list,
                                       unsigned int *defer, cudaStream_t stream) {
    if (lv.L <= 128) return launch_finish_sweep_lq<4>(lv, prm, sm_count, counter, overflow, list, defer, stream);
    return launch_finish_sweep_lq<8>(lv, prm, sm_count, counter, overflow, list, defer, stream);
}

}  // namespace linmin
