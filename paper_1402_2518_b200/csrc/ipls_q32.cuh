// ipls_q32.cuh -- K1 of the R = 32 path: the IPLS Newton iteration, round 2.
//
// Same iteration as ipls_generic.cuh (Mehrotra predictor-corrector on the centred normal equations; reading R1),
// started from the records of start_r32.cuh.  What changed against the round-1 kernel (8 lanes per pixel, 4 pixels
// per warp, prologue fused) is the mapping, chosen from its ncu profile (shared-memory pipe 74 % busy, FMA pipe
// 35 %: every lane of a pixel must receive every entry of every column of the factor, and data can only reach
// registers at 128 B per cycle and SM):
//   * FOUR lanes per pixel, EIGHT pixels per warp.  Lane t owns rows t + 4 s (s = 0..7, cyclic) of the 32 x 32
//     Newton matrix M = G + diag(lambda/a), row t + 4 s up to column 4 s + 3, as 72 packed pairs (144 registers);
//     the rank-one updates are FFMA2 with the row's multiplier broadcast.  The column broadcast of the
//     right-looking LDL' factorisation (one padded shared-memory line per pixel, LDS.128) costs the same number
//     of wavefronts per warp as before but serves twice the pixels: 16 instead of 8 FMAs per delivered float.
//   * No prologue in this kernel (projection and start point are K0's), so a pixel group that has converged takes
//     the next record from a small prefetch queue at once instead of riding along until the slowest of the warp
//     is done: the warp executes the MEAN iteration count of its pixels, not the maximum.
//   * Triangular solves by shuffles inside the 4-lane group.  The predictor's forward substitution (right-hand
//     sides 1 and -w) rides along the factorisation; the corrector's is a 31-step column sweep; the backward
//     substitutions go block by block (4 x 4 diagonal blocks): partial sums of the later rows, one all-reduce over
//     the four lanes, then the lane's column of the inverse diagonal block (3 registers per block, formed during the
//     factorisation from the broadcast column).
//   * G a - b is carried through the Newton identity G da = (r1 - dnu 1) - d o da (no mat-vec per iteration).
//
// Algorithmic work per pixel-iteration: R^3/3 + 8 R^2 + 30 R flops.
#pragma once
#include "common.cuh"
#include "start_r32.cuh"

namespace linmin {
namespace q32 {

constexpr int R = 32;
constexpr int S = 8;            // rows per lane
constexpr int WARPS = 8;        // warps per CTA, one CTA per SM (255 registers)
constexpr int GST = 36;         // padded row stride of G in shared memory (conflict-free LDS.128 over the 4 lanes)
constexpr int XST = 36;         // one exchange line: 32 column entries + pad
constexpr int PRK = 72;         // offset of the park area: a, lambda, G a - b wait here during the factorisation ([3][4 lanes][8])
constexpr int PIXF = 196;       // floats per pixel: two exchange lines + park area; 196 = 4 mod 32 spreads the 8 pixels of a warp
constexpr int QD = 8;           // prefetch queue depth (records) per warp
constexpr int REC = s32::REC;
constexpr int BLK = 256;        // pixels a warp reserves per ticket
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ float gsum(float v) { return group_sum<4>(v); }   // over the 4 lanes of a pixel
__device__ __forceinline__ float gmin(float v) { return group_min<4>(v); }
__device__ __forceinline__ float gmax(float v) { return group_max<4>(v); }

__host__ __device__ inline size_t smem_floats() {
    return (size_t)R * GST + (size_t)WARPS * (8 * PIXF + QD * REC + QD);
}

// column j of the register-resident matrix (static j)
#define QCOL(s, j) (((j) & 1) ? m2[s][(j) >> 1].y : m2[s][(j) >> 1].x)

// L' x = y in place.  m2 holds -L (strictly lower), ct[s][0..2] the lane's column of the inverse of diagonal block s
// (coefficients of the block's totals 1..3; the coefficient of total 0 is [t == 0]).
__device__ __forceinline__ void backward_subst(const float2 (&m2)[S][2 * S], const float (&ct)[S][3], float (&y)[S], int t,
                                               const float2 e2a, const float2 e2b) {
#pragma unroll
    for (int s = S - 1; s >= 0; --s) {
        // my own right-hand side enters at my position of the block (one-hot pairs), then the later rows' shares
        float2 pa = make_float2(y[s] * e2a.x, y[s] * e2a.y), pb = make_float2(y[s] * e2b.x, y[s] * e2b.y);
        float2 qa = make_float2(0.0f, 0.0f), qb = make_float2(0.0f, 0.0f);
#pragma unroll
        for (int sp = s + 1; sp < S; ++sp) {
            if ((sp - s) & 1) { pa = fma2(y[sp], m2[sp][2 * s], pa); pb = fma2(y[sp], m2[sp][2 * s + 1], pb); }
            else { qa = fma2(y[sp], m2[sp][2 * s], qa); qb = fma2(y[sp], m2[sp][2 * s + 1], qb); }
        }
        float v0 = pa.x + qa.x, v1 = pa.y + qa.y, v2 = pb.x + qb.x, v3 = pb.y + qb.y;
        v0 += __shfl_xor_sync(FULL, v0, 1); v1 += __shfl_xor_sync(FULL, v1, 1);
        v2 += __shfl_xor_sync(FULL, v2, 1); v3 += __shfl_xor_sync(FULL, v3, 1);
        v0 += __shfl_xor_sync(FULL, v0, 2); v1 += __shfl_xor_sync(FULL, v1, 2);
        v2 += __shfl_xor_sync(FULL, v2, 2); v3 += __shfl_xor_sync(FULL, v3, 2);
        float x = e2a.x * v0;
        x = fmaf(ct[s][0], v1, x);
        x = fmaf(ct[s][1], v2, x);
        x = fmaf(ct[s][2], v3, x);
        y[s] = x;
    }
}

}  // namespace q32

// counter: device word, zero (the caller clears it on the stream before the launch); rec: records of K0 for the
// pixels [p_begin, p_end).
// CONS false: positivity only (no equality constraint: r_p == 0, dnu == 0, nu stays 0).  A template parameter, not a flag:
// the flag cost the sto path 1.6 % (one more multiply on the chain through dnu).
template <bool CONS>
__global__ void __launch_bounds__(q32::WARPS * 32, 1)
ipls_q32_kernel(LibView lib, SolveParams prm, int64_t p_begin, int64_t p_end, const float *__restrict__ rec,
                unsigned int *__restrict__ counter) {
    using namespace q32;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0]) return;      // non-finite library: the caller is told (status or poisoned outputs)
    float *Gp = smem;                                             // [32][GST]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    float *wbase = Gp + R * GST + (size_t)warp * (8 * PIXF + QD * REC + QD);
    float *xb0 = wbase + g * PIXF;                                // exchange line, buffer 0
    float *xb1 = xb0 + XST;                                       // buffer 1
    float *queue = wbase + 8 * PIXF;                              // [QD][REC] prefetched records
    int *qpix = reinterpret_cast<int *>(queue + QD * REC);        // [QD] pixel (relative to p_begin) of each slot, -1 = none

    for (int e = threadIdx.x; e < R * R; e += blockDim.x) Gp[(e >> 5) * GST + (e & 31)] = lib.Gc[e];
    __syncthreads();

    const float gdmax = lib.scal[0];
    const float tau = 0.995f;
    const float pivot_floor = 1e-12f * gdmax;
    const int64_t npix = p_end - p_begin;
    // one-hot pairs of my position inside a diagonal block: adds lambda/a to the diagonal with FFMA2
    const float2 e2a = make_float2((t == 0) ? 1.0f : 0.0f, (t == 1) ? 1.0f : 0.0f);
    const float2 e2b = make_float2((t == 2) ? 1.0f : 0.0f, (t == 3) ? 1.0f : 0.0f);

    // ---- work tickets: blocks of BLK consecutive pixels; the atomic for the next block is issued when a block is
    //      begun, so its latency is hidden behind BLK pixels of work
    int64_t tk = 0, tk_end = 0, tk_nextblk = 0;
    {
        unsigned int b0 = 0, b1 = 0;
        if (lane == 0) { b0 = atomicAdd(counter, 1u); b1 = atomicAdd(counter, 1u); }
        b0 = __shfl_sync(FULL, b0, 0); b1 = __shfl_sync(FULL, b1, 0);
        tk = (int64_t)b0 * BLK; tk_end = tk + BLK; tk_nextblk = (int64_t)b1 * BLK;
    }
    // issues the prefetch of the next pixel's record into queue slot `slot` (whole warp; 25 lanes x 16 B)
    auto prefetch_next = [&](int slot) {
        if (tk == tk_end) {
            tk = tk_nextblk; tk_end = tk + BLK;
            unsigned int b = 0;
            if (lane == 0) b = atomicAdd(counter, 1u);
            tk_nextblk = (int64_t)__shfl_sync(FULL, b, 0) * BLK;
        }
        const bool ok = tk < npix;
        if (lane == 0) qpix[slot] = ok ? (int)tk : -1;
        if (ok && lane < REC / 4) {
            const unsigned sa = (unsigned)__cvta_generic_to_shared(queue + slot * REC + 4 * lane);
            asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(rec + tk * REC + 4 * lane) : "memory");
        }
        if (ok) ++tk;
    };
#pragma unroll 1
    for (int i = 0; i < QD; ++i) prefetch_next(i);
    asm volatile("cp.async.commit_group;" ::: "memory");
    int head = 0;

    // ---- per-lane state of my pixel: rows t + 4 s
    float a[S], lam[S], gmb[S];          // gmb = G a - b
    float nu = 0.0f, sc = 1.0f, lam0 = 1.0f;
    int flags = 0, iters = 0, pix = -1;
    bool done = true;                    // "needs a pixel"
    bool idle = false;                   // no pixel left for this group
#pragma unroll
    for (int s = 0; s < S; ++s) { a[s] = 1.0f / 32.0f; lam[s] = 1.0f; gmb[s] = 0.0f; }

#pragma unroll 1
    while (true) {
        // ---- residuals and stopping rule (per pixel group)
        float mu, rp;
        {
            float rdm = 0.0f, sa = 0.0f, gp = 0.0f;
#pragma unroll
            for (int s = 0; s < S; ++s) {
                rdm = fmaxf(rdm, fabsf(gmb[s] + nu - lam[s]));
                sa += a[s];
                gp = fmaf(a[s], lam[s], gp);
            }
            rdm = gmax(rdm); sa = gsum(sa); gp = gsum(gp);
            rp = CONS ? sa - 1.0f : 0.0f;
            mu = gp * (1.0f / 32.0f);
            if (!done && !idle) {
                if (flags & LINMIN_INFO_NONFINITE_INPUT) {
                    done = true;
                } else if (gp <= prm.gap_tol * sc && rdm <= prm.feas_tol * sc && fabsf(rp) <= prm.feas_tol) {
                    done = true; flags |= LINMIN_INFO_CONVERGED;
                } else if (iters >= prm.max_iter) {
                    done = true; flags |= LINMIN_INFO_MAX_ITER;
                }
            }
        }
        // ---- groups that are done store their iterate and take the next record from the queue
        const unsigned dmask = __ballot_sync(FULL, done && !idle && t == 0);
        if (dmask) {
            if (done && !idle && pix >= 0) {
                // the iterate, with a_i = 0 where the primal-dual indicator says "inactive" (coalesced: 4 lanes x 32 B)
                __syncwarp(0xfu << (4 * g));
#pragma unroll
                for (int s = 0; s < S; ++s) xb0[t + 4 * s] = (a[s] * sc > LINMIN_TAPIA_KAPPA * lam[s]) ? a[s] : 0.0f;
                __syncwarp(0xfu << (4 * g));
                const int64_t p = p_begin + pix;
                const float4 o0 = *reinterpret_cast<const float4 *>(xb0 + 8 * t);
                const float4 o1 = *reinterpret_cast<const float4 *>(xb0 + 8 * t + 4);
                *reinterpret_cast<float4 *>(prm.coeffs + p * R + 8 * t) = o0;
                *reinterpret_cast<float4 *>(prm.coeffs + p * R + 8 * t + 4) = o1;
                if (prm.info && t == 0) prm.info[p] = flags | (iters << 8);
            }
            asm volatile("cp.async.wait_all;" ::: "memory");
            __syncwarp();
            const int m = __popc(dmask);
            if (done && !idle) {
                const int rank = __popc(dmask & ((1u << (lane & ~3)) - 1u));
                const int slot = (head + rank) & (QD - 1);
                const int np = qpix[slot];
                if (np >= 0) {
                    const float *q = queue + slot * REC;
                    const float4 a0 = *reinterpret_cast<const float4 *>(q + 8 * t), a1 = *reinterpret_cast<const float4 *>(q + 8 * t + 4);
                    const float4 l0 = *reinterpret_cast<const float4 *>(q + 32 + 8 * t), l1 = *reinterpret_cast<const float4 *>(q + 32 + 8 * t + 4);
                    const float4 g0 = *reinterpret_cast<const float4 *>(q + 64 + 8 * t), g1 = *reinterpret_cast<const float4 *>(q + 64 + 8 * t + 4);
                    const float4 sv = *reinterpret_cast<const float4 *>(q + 96);
                    const float2 mr = *reinterpret_cast<const float2 *>(q + 100);
                    a[0] = a0.x; a[1] = a0.y; a[2] = a0.z; a[3] = a0.w; a[4] = a1.x; a[5] = a1.y; a[6] = a1.z; a[7] = a1.w;
                    lam[0] = l0.x; lam[1] = l0.y; lam[2] = l0.z; lam[3] = l0.w; lam[4] = l1.x; lam[5] = l1.y; lam[6] = l1.z; lam[7] = l1.w;
                    gmb[0] = g0.x; gmb[1] = g0.y; gmb[2] = g0.z; gmb[3] = g0.w; gmb[4] = g1.x; gmb[5] = g1.y; gmb[6] = g1.z; gmb[7] = g1.w;
                    nu = sv.x; sc = sv.y; lam0 = sv.z; flags = __float_as_int(sv.w);
                    mu = mr.x; rp = mr.y;          // of the start point (K0): no second pass over the residuals
                    iters = 0; pix = np; done = false;
                } else {
                    idle = true; pix = -1;
                }
            }
            __syncwarp();                 // the slots have been read: they may be refilled
#pragma unroll 1
            for (int i = 0; i < m; ++i) prefetch_next((head + i) & (QD - 1));
            asm volatile("cp.async.commit_group;" ::: "memory");
            head = (head + m) & (QD - 1);
            if (__all_sync(FULL, idle)) break;
            // a fresh pixel goes straight into its first Newton step (the stopping rule sees it next time round)
        }
        if (!idle) ++iters;

        // ---- rows of M (lower part) from G, M = G + diag(lambda / a)
        float2 m2[S][2 * S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
#pragma unroll
            for (int c = 0; c <= s; ++c) {
                const float4 g4 = *reinterpret_cast<const float4 *>(Gp + (t + 4 * s) * GST + 4 * c);
                m2[s][2 * c] = make_float2(g4.x, g4.y);
                m2[s][2 * c + 1] = make_float2(g4.z, g4.w);
            }
        }
        float dinv[S];
        float2 rr[S];          // (row of L^-1 1, row of L^-1 (-w)): the predictor's forward substitution rides along
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const float d = lam[s] * rcp_approx(a[s]);
            dinv[s] = 0.0f;
            m2[s][2 * s] = fma2(d, e2a, m2[s][2 * s]);
            m2[s][2 * s + 1] = fma2(d, e2b, m2[s][2 * s + 1]);
            rr[s] = make_float2(1.0f, -(gmb[s] + nu));
        }
        // the pixel's vectors wait in shared memory while the factorisation needs every register
        {
            float *pk = xb0 + PRK + 8 * t;
            *reinterpret_cast<float4 *>(pk) = make_float4(a[0], a[1], a[2], a[3]);
            *reinterpret_cast<float4 *>(pk + 4) = make_float4(a[4], a[5], a[6], a[7]);
            *reinterpret_cast<float4 *>(pk + 32) = make_float4(lam[0], lam[1], lam[2], lam[3]);
            *reinterpret_cast<float4 *>(pk + 36) = make_float4(lam[4], lam[5], lam[6], lam[7]);
            *reinterpret_cast<float4 *>(pk + 64) = make_float4(gmb[0], gmb[1], gmb[2], gmb[3]);
            *reinterpret_cast<float4 *>(pk + 68) = make_float4(gmb[4], gmb[5], gmb[6], gmb[7]);
        }
        // ---- M = L D L' (right-looking).  m2 ends as -L (strictly lower; zeros on and above the diagonal inside the
        //      diagonal blocks), dinv = 1 / d, ct = my column of the inverse of each diagonal block of L.
        float ct[S][3];
        bool clamped = false;
        float4 l4[S];           // column k (raw), as read back from the exchange line
        float2 zk;              // right-hand sides of row k
        {
#pragma unroll
            for (int s = 0; s < S; ++s) xb0[t + 4 * s] = QCOL(s, 0);
            __syncwarp();
            zk = make_float2(__shfl_sync(FULL, rr[0].x, 0, 4), __shfl_sync(FULL, rr[0].y, 0, 4));
#pragma unroll
            for (int c = 0; c < S; ++c) l4[c] = *reinterpret_cast<const float4 *>(xb0 + 4 * c);
        }
        float l10 = 0.0f, l20 = 0.0f, l30 = 0.0f, l21 = 0.0f, l31 = 0.0f;
#define L4C(j) ((((j) & 3) == 0) ? l4[(j) >> 2].x : ((((j) & 3) == 1) ? l4[(j) >> 2].y : ((((j) & 3) == 2) ? l4[(j) >> 2].z : l4[(j) >> 2].w)))
#pragma unroll
        for (int k = 0; k < R - 1; ++k) {
            const int s0 = k >> 2, t0 = k & 3;
            const int k1 = k + 1, s1 = k1 >> 2;
            float piv = L4C(k);
            if (!(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
            const float rinv = rcp_approx(piv);
            const float nrinv = -rinv;
            float nl[S];
#pragma unroll
            for (int s = s0; s < S; ++s) {
                float v = QCOL(s, k) * nrinv;
                if (s == s0) v = (t > t0) ? v : 0.0f;      // rows at or above k: no update, store 0
                nl[s] = v;
                if (k & 1) m2[s][k >> 1].y = v; else m2[s][k >> 1].x = v;
                rr[s] = fma2(v, zk, rr[s]);
            }
            dinv[s0] = (t == t0) ? rinv : dinv[s0];
            // ---- the diagonal block's entries of this column (every lane has them: the column was broadcast);
            //      after the block's third column, my column of the inverse of the block
            if (t0 == 0) { l10 = l4[s0].y * rinv; l20 = l4[s0].z * rinv; l30 = l4[s0].w * rinv; }
            if (t0 == 1) { l21 = l4[s0].z * rinv; l31 = l4[s0].w * rinv; }
            if (t0 == 2) {
                const float l32 = l4[s0].w * rinv;
                const float i20 = fmaf(l21, l10, -l20);
                const float i31 = fmaf(l32, l21, -l31);
                const float i30 = fmaf(-l32, i20, fmaf(l31, l10, -l30));
                // lane t takes column t of the inverse: blended with the one-hot values of t (no divergent branch)
                ct[s0][0] = fmaf(e2a.x, -l10, e2a.y);
                ct[s0][1] = fmaf(e2a.x, i20, fmaf(e2a.y, -l21, e2b.x));
                ct[s0][2] = fmaf(e2a.x, i30, fmaf(e2a.y, i31, fmaf(e2b.x, -l32, e2b.y)));
            }
            // ---- look-ahead: column k + 1 first, then its exchange
            {
                const float ck1 = L4C(k1);
#pragma unroll
                for (int s = s1; s < S; ++s) {
                    if (k1 & 1) m2[s][k1 >> 1].y = fmaf(nl[s], ck1, m2[s][k1 >> 1].y);
                    else m2[s][k1 >> 1].x = fmaf(nl[s], ck1, m2[s][k1 >> 1].x);
                }
            }
            const float *cb = (k1 & 1) ? xb1 : xb0;
            if (k1 < R - 1) {
                float *cw = (k1 & 1) ? xb1 : xb0;
#pragma unroll
                for (int s = s1; s < S; ++s) cw[t + 4 * s] = QCOL(s, k1);
                __syncwarp();
                zk = make_float2(__shfl_sync(FULL, rr[s1].x, k1 & 3, 4), __shfl_sync(FULL, rr[s1].y, k1 & 3, 4));
            }
            // ---- rest of the rank-one update of step k (columns k + 2 ..), chunk by chunk; a chunk of column k is
            //      replaced by the same chunk of column k + 1 as soon as it has been used
#pragma unroll
            for (int c = k1 >> 2; c < S; ++c) {
                if (c >= ((k + 2) >> 2)) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int jp = 2 * c + h, j0 = 2 * jp;
                        const float2 cp = h ? make_float2(l4[c].z, l4[c].w) : make_float2(l4[c].x, l4[c].y);
                        if (j0 >= k + 2) {
#pragma unroll
                            for (int s = (s0 > c ? s0 : c); s < S; ++s) m2[s][jp] = fma2(nl[s], cp, m2[s][jp]);
                        } else if (j0 + 1 == k + 2) {
#pragma unroll
                            for (int s = (s0 > c ? s0 : c); s < S; ++s) m2[s][jp].y = fmaf(nl[s], cp.y, m2[s][jp].y);
                        }
                    }
                }
                if (k1 < R - 1) l4[c] = *reinterpret_cast<const float4 *>(cb + 4 * c);
            }
        }
#undef L4C
        {   // k = 31: only the last pivot (its owner has it); the last block's inverse column is complete
            float piv = m2[S - 1][2 * S - 1].y;
            if (t == 3 && !(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
            dinv[S - 1] = (t == 3) ? rcp_approx(piv) : dinv[S - 1];
        }
        if (__any_sync(0xfu << (4 * g), clamped)) flags |= LINMIN_INFO_CHOL_REGULARISED;
        {
            const float *pk = xb0 + PRK + 8 * t;
            const float4 a0 = *reinterpret_cast<const float4 *>(pk), a1 = *reinterpret_cast<const float4 *>(pk + 4);
            const float4 l0 = *reinterpret_cast<const float4 *>(pk + 32), l1 = *reinterpret_cast<const float4 *>(pk + 36);
            const float4 g0 = *reinterpret_cast<const float4 *>(pk + 64), g1 = *reinterpret_cast<const float4 *>(pk + 68);
            a[0] = a0.x; a[1] = a0.y; a[2] = a0.z; a[3] = a0.w; a[4] = a1.x; a[5] = a1.y; a[6] = a1.z; a[7] = a1.w;
            lam[0] = l0.x; lam[1] = l0.y; lam[2] = l0.z; lam[3] = l0.w; lam[4] = l1.x; lam[5] = l1.y; lam[6] = l1.z; lam[7] = l1.w;
            gmb[0] = g0.x; gmb[1] = g0.y; gmb[2] = g0.z; gmb[3] = g0.w; gmb[4] = g1.x; gmb[5] = g1.y; gmb[6] = g1.z; gmb[7] = g1.w;
        }

        // ---- predictor: M^-1 = L^-T D^-1 L^-1; nu eliminated through L^-1 1
        float sww = 0.0f, swz = 0.0f;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const float zd = rr[s].x * dinv[s];
            sww = fmaf(zd, rr[s].x, sww);
            swz = fmaf(zd, rr[s].y, swz);
        }
        sww = gsum(sww); swz = gsum(swz);
        const float rsww = CONS ? rcp_approx(sww) : 0.0f;
        float dnu = (swz + rp) * rsww;
        float da[S];
#pragma unroll
        for (int s = 0; s < S; ++s) da[s] = fmaf(-rr[s].x, dnu, rr[s].y) * dinv[s];
        backward_subst(m2, ct, da, t, e2a, e2b);
        float ainv[S];
        float mp = 0.0f, md = 0.0f;     // max of -da/a and -dl/lambda
#pragma unroll
        for (int s = 0; s < S; ++s) {
            ainv[s] = rcp_approx(a[s]);
            mp = fmaxf(mp, -da[s] * ainv[s]);
            md = fmaxf(md, 1.0f + ainv[s] * da[s]);       // -dl/lambda = 1 + da/a
        }
        mp = gmax(mp); md = gmax(md);
        float ap = (mp > 1.0f) ? rcp_approx(mp) : 1.0f;
        float ad = (md > 1.0f) ? rcp_approx(md) : 1.0f;
        float mua = 0.0f;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const float dl = -lam[s] - lam[s] * ainv[s] * da[s];
            mua = fmaf(fmaf(ap, da[s], a[s]), fmaf(ad, dl, lam[s]), mua);
        }
        mua = gsum(mua) * (1.0f / 32.0f);
        float sg = mua * rcp_approx(mu);
        sg = fminf(1.0f, fmaxf(0.0f, sg * sg * sg));
        // ---- corrector
        float cc[S], r1[S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const float dl = -lam[s] - lam[s] * ainv[s] * da[s];
            cc[s] = fmaf(sg, mu, -da[s] * dl);
            r1[s] = fmaf(cc[s], ainv[s], -(gmb[s] + nu));
        }
        // forward substitution L z = r1: column sweep, z_k travels by shuffle inside the group
#pragma unroll
        for (int k = 0; k < R - 1; ++k) {
            const float z = __shfl_sync(FULL, r1[k >> 2], k & 3, 4);
#pragma unroll
            for (int s = k >> 2; s < S; ++s) r1[s] = fmaf(QCOL(s, k), z, r1[s]);
        }
        swz = 0.0f;
#pragma unroll
        for (int s = 0; s < S; ++s) swz = fmaf(rr[s].x * dinv[s], r1[s], swz);
        swz = gsum(swz);
        dnu = (swz + rp) * rsww;
#pragma unroll
        for (int s = 0; s < S; ++s) da[s] = fmaf(-rr[s].x, dnu, r1[s]) * dinv[s];
        backward_subst(m2, ct, da, t, e2a, e2b);
        mp = 0.0f; md = 0.0f;
        float dl[S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
            dl[s] = fmaf(cc[s], ainv[s], -lam[s]) - lam[s] * ainv[s] * da[s];
            mp = fmaxf(mp, -da[s] * ainv[s]);
            md = fmaxf(md, -dl[s] * rcp_approx(lam[s]));
        }
        mp = gmax(mp); md = gmax(md);
        ap = (tau < mp) ? tau * rcp_approx(mp) : 1.0f;     // min(1, tau / mp)
        ad = (tau < md) ? tau * rcp_approx(md) : 1.0f;
        if (idle) { ap = 0.0f; ad = 0.0f; }                // groups without a pixel ride along unchanged
#pragma unroll
        for (int s = 0; s < S; ++s) {
            gmb[s] = fmaf(ap, fmaf(cc[s], ainv[s], -(gmb[s] + nu)) - dnu - lam[s] * ainv[s] * da[s], gmb[s]);
            a[s] = fmaxf(fmaf(ap, da[s], a[s]), 1e-18f);
            lam[s] = fmaxf(fmaf(ad, dl[s], lam[s]), 1e-18f * lam0);
        }
        nu = fmaf(ad, dnu, nu);
    }
}
#undef QCOL

inline cudaError_t launch_ipls_q32(const LibView &lv, const SolveParams &prm, int64_t p_begin, int64_t p_end,
                                   const float *rec, int sm_count, unsigned int *counter, cudaStream_t stream) {
    const size_t smem = q32::smem_floats() * sizeof(float);
    cudaError_t e = lv.cons ? cudaFuncSetAttribute(ipls_q32_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                            : cudaFuncSetAttribute(ipls_q32_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t n = p_end - p_begin;
    const int64_t need = (n + 8 * q32::WARPS - 1) / (8 * q32::WARPS);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, (int64_t)sm_count));
    if (lv.cons) ipls_q32_kernel<true><<<grid, q32::WARPS * 32, smem, stream>>>(lv, prm, p_begin, p_end, rec, counter);
    else ipls_q32_kernel<false><<<grid, q32::WARPS * 32, smem, stream>>>(lv, prm, p_begin, p_end, rec, counter);
    return cudaGetLastError();
}

}  // namespace linmin
