// finish8.cuh -- exact finish + uncertainty + residual for R <= 32, L <= 256 (sm_100a): the
// throughput path of SURVEY.md 8(a) a3-a6.
//
// Same mathematics as finish.cuh (read its header: PAPER.md:54-68 optimality conditions,
// PAPER.md:88 uncertainty reading R3, PAPER.md:143 RMS reading R8).  Mapping:
//   * 8 lanes cooperate on one pixel, 4 pixels per warp (the layout of ipls_r32.cuh).  Lane t owns
//     channels {4 (t + 8 v) + q}: the spectrum, its fp64 residual and the noise std stay in registers;
//     every pass over the L channels is a stream of LDS.128 from the library staged once per CTA in
//     shared memory (fp64 copy for the residual / A_F'r passes, fp32 copy for A'r and J = H A_F'),
//     and the four pixels of a warp share the broadcast when they read the same library row.
//   * everything k-sized (k = support size <= KM = 16) lives in a 2.3 KB per-pixel scratch area in
//     shared memory and is worked on by the pixel's 8 lanes in compact loops with runtime bounds:
//     packed fp64 Cholesky factor of G_FF (left-looking), triangular solves with the right-hand sides
//     in registers (lane j & 7 owns member j) and shuffle broadcasts, in-place inverse W = L^-1,
//     H = W'W - q q'/(1'q).  Small code: the instruction cache, not the ALUs, limited finish_fast.
//   * pixels whose support would exceed KM are appended to an overflow list and finished by
//     finish_fast_kernel (list mode) in a second launch; on the synthetic cubes this list is empty.
#pragma once
#include "common.cuh"
#include "finish.cuh"

namespace linmin {
namespace f8 {

constexpr unsigned FULL = 0xffffffffu;
constexpr int KM = 16;   // support cap of this kernel
constexpr int RP = 32;   // endmember rows staged (rows >= R are zero)

// per-pixel scratch (bytes; every block 16 B aligned)
constexpr int OFF_LF = 0;                       // double[136] packed row-major lower; later W; later Hs float[16][16]
constexpr int OFF_AF = OFF_LF + 136 * 8;        // double[16] coefficients on the support
constexpr int OFF_QV = OFF_AF + 16 * 8;         // double[16] K 1
constexpr int OFF_ROWB = OFF_QV + 16 * 8;       // double[16] row buffer
constexpr int OFF_HP = OFF_ROWB + 16 * 8;       // float[136] packed H
constexpr int OFF_G = OFF_HP + 136 * 4;         // float[32] gradient / staging of outputs
constexpr int OFF_SG = OFF_G + 32 * 4;          // float[16] coeff_sigma per member
constexpr int OFF_IDX = OFF_SG + 16 * 4;        // int[16]
constexpr int OFF_STATE = OFF_IDX + 16 * 4;     // uchar[32]: 0 free, 1 in F, 2 blocked
constexpr int PIX_BYTES = OFF_STATE + 32;       // 2304
static_assert(PIX_BYTES % 16 == 0, "scratch alignment");

__host__ __device__ inline size_t cta_bytes(int R, int LQ) {
    return (((size_t)R * R * 8 + 15) & ~(size_t)15) + (size_t)RP * 32 * LQ * 8 + (size_t)RP * 32 * LQ * 4;
}

__device__ __forceinline__ double gsum(double v) {
    v += __shfl_xor_sync(FULL, v, 1);
    v += __shfl_xor_sync(FULL, v, 2);
    v += __shfl_xor_sync(FULL, v, 4);
    return v;
}
__device__ __forceinline__ float gsum(float v) {
    v += __shfl_xor_sync(FULL, v, 1);
    v += __shfl_xor_sync(FULL, v, 2);
    v += __shfl_xor_sync(FULL, v, 4);
    return v;
}
__device__ __forceinline__ double gmin(double v) {
    v = fmin(v, __shfl_xor_sync(FULL, v, 1));
    v = fmin(v, __shfl_xor_sync(FULL, v, 2));
    v = fmin(v, __shfl_xor_sync(FULL, v, 4));
    return v;
}
__device__ __forceinline__ float gminf(float v) {
    v = fminf(v, __shfl_xor_sync(FULL, v, 1));
    v = fminf(v, __shfl_xor_sync(FULL, v, 2));
    v = fminf(v, __shfl_xor_sync(FULL, v, 4));
    return v;
}
__device__ __forceinline__ float gmaxf(float v) {
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 1));
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 2));
    v = fmaxf(v, __shfl_xor_sync(FULL, v, 4));
    return v;
}
__device__ __forceinline__ unsigned gor(unsigned v) {
    v |= __shfl_xor_sync(FULL, v, 1);
    v |= __shfl_xor_sync(FULL, v, 2);
    v |= __shfl_xor_sync(FULL, v, 4);
    return v;
}
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
__device__ __forceinline__ double rsqrt_d(double x) {   // fp32 MUFU seed + two Newton steps
    double y = (double)rsqrtf((float)x);
    double hx = 0.5 * x;
    y = y * (1.5 - hx * y * y);
    y = y * (1.5 - hx * y * y);
    return y;
}
__device__ __forceinline__ int tri(int i) { return (i * (i + 1)) >> 1; }

}  // namespace f8

// LQ = float4 chunks of the spectrum per lane: L <= 32 LQ
template <int LQ>
__global__ void __launch_bounds__(512, 1)
finish8_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter,
               unsigned int *__restrict__ overflow /* [0] = count, [1 + i] = pixel */) {
    using namespace f8;
    constexpr int NC = 4 * LQ;          // channels per lane
    constexpr int RS = 32 * LQ;         // library row stride (elements)
    constexpr int IT = (LQ <= 4) ? 4 : 2;   // J rows per tile
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = lib.L, R = lib.R;
    double *G64s = (double *)smem_raw;
    double *At64 = (double *)(smem_raw + (((size_t)R * R * 8 + 15) & ~(size_t)15));   // [RP][2][8 LQ][2]
    float *At32 = (float *)(At64 + (size_t)RP * RS);                                    // [RP][32 LQ]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 3, t = lane & 7;
    unsigned char *S = (unsigned char *)(At32 + (size_t)RP * RS) + (size_t)(warp * 4 + g) * PIX_BYTES;
    double *Lf = (double *)(S + OFF_LF);
    float *Hs = (float *)(S + OFF_LF);
    double *aFs = (double *)(S + OFF_AF);
    double *qv = (double *)(S + OFF_QV);
    double *rowb = (double *)(S + OFF_ROWB);
    float *Hp = (float *)(S + OFF_HP);
    float *gs = (float *)(S + OFF_G);
    float *sgs = (float *)(S + OFF_SG);
    int *idx = (int *)(S + OFF_IDX);
    unsigned char *state = S + OFF_STATE;

    // ---- once per CTA: stage the library (transposed; fp64 copy split in two planes per float4)
    for (int e = threadIdx.x; e < R * R; e += blockDim.x) G64s[e] = lib.G64[e];
    for (int e = threadIdx.x; e < RP * RS; e += blockDim.x) {
        const int r = e / RS, l = e - r * RS;
        const float a = (r < R && l < L) ? lib.A[(size_t)l * R + r] : 0.0f;
        At32[e] = a;
        const int c = l >> 2, q = l & 3;
        At64[(size_t)r * RS + (q >> 1) * (RS / 2) + c * 2 + (q & 1)] = (double)a;
    }
    __syncthreads();

    const bool vec_ok = ((prm.ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.Y) & 15) == 0);
    const bool svec_ok = prm.has_sigma && ((prm.sigma_stride & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.sigma) & 15) == 0);
    const bool cvec_ok = ((R & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.coeffs) & 15) == 0);
    const bool csvec_ok = ((R & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.coeff_sigma) & 15) == 0);
    const float qnan = __int_as_float(0x7fc00000);
    const int max_pivots = 4 * RP + 8;
    const int o0 = tri(t), o1 = tri(t + 8);   // packed starts of my two rows

    while (true) {
        unsigned int grp = 0;
        if (lane == 0) grp = atomicAdd(counter, 1u);
        grp = __shfl_sync(FULL, grp, 0);
        const int64_t p0 = (int64_t)grp * 4;
        if (p0 >= prm.N) break;
        const bool valid = (p0 + g) < prm.N;
        const int64_t p = valid ? (p0 + g) : (prm.N - 1);
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

        // ---- initial support from the IPLS iterate; lane t looks at endmembers 4 t + q
        // st: 0 solving, 1 optimal, 2 fallback (feasible point, not certified), 3 nothing to write here
        int st = valid ? 0 : 3;
        int k = 0;
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
            if (mask == 0u) {   // can not happen for a point of the simplex; be safe: the largest entry
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
        // lane j & 7 owns members j = t (slot 0) and t + 8 (slot 1): coefficient, right-hand sides
        double a0 = 0.0, a1 = 0.0;
        int i0 = 0, i1 = 0;
        if (st == 0) {
            if (t < k) { a0 = aFs[t]; i0 = idx[t]; }
            if (t + 8 < k) { a1 = aFs[t + 8]; i1 = idx[t + 8]; }
        }
        {
            const double s = gsum(a0 + a1);
            if (st == 0) {
                a0 /= s; a1 /= s;
                if (t < k) aFs[t] = a0;
                if (t + 8 < k) aFs[t + 8] = a1;
            }
        }
        __syncwarp();

        int pivots = 0, last_added = -1;
        double r[NC];
        double q0 = 0.0, q1 = 0.0, sq = 1.0;
#pragma unroll
        for (int c = 0; c < NC; ++c) r[c] = 0.0;

        while (__any_sync(FULL, st == 0)) {
            const bool act = (st == 0);
            const int kw = wmax(act ? k : 0);
            // ---- gather G_FF (packed rows) and factor it (fp64, left-looking by columns)
            if (act) {
                for (int i = 0; i < k; ++i) {
                    const int gi = idx[i] * R;
                    for (int j = t; j <= i; j += 8) Lf[tri(i) + j] = G64s[gi + idx[j]];
                }
            }
            __syncwarp();
            int rej = -1;
            for (int j = 0; j < kw; ++j) {
                // rows i = j + t and j + t + 8 of column j
                const int ia = j + t, ib = j + t + 8;
                double sa = 0.0, sb2 = 0.0, gjj = 1.0;
                const bool on = act && rej < 0 && j < k;
                if (on) {
                    gjj = Lf[tri(j) + j];
                    const double *rj = Lf + tri(j);
                    if (ia < k) {
                        const double *ri = Lf + tri(ia);
                        sa = ri[j];
                        for (int m = 0; m < j; ++m) sa -= ri[m] * rj[m];
                    }
                    if (ib < k) {
                        const double *ri = Lf + tri(ib);
                        sb2 = ri[j];
                        for (int m = 0; m < j; ++m) sb2 -= ri[m] * rj[m];
                    }
                }
                const double sj = __shfl_sync(FULL, sa, 0, 8);    // diagonal: lane t = 0 has row j
                __syncwarp();                                       // reads of column j inputs done
                if (on) {
                    if (!(sj > 1e-13 * gjj)) {
                        rej = j;
                    } else {
                        const double dj = rsqrt_d(sj);
                        if (t == 0) Lf[tri(j) + j] = dj;            // the diagonal stores 1 / L_jj
                        else if (ia < k) Lf[tri(ia) + j] = sa * dj;
                        if (ib < k) Lf[tri(ib) + j] = sb2 * dj;
                    }
                }
                __syncwarp();
            }
            bool skip = !act;
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
            {
                const double s = gsum(a0 + a1);
                if (act && rej >= 0) {
                    if (k == 0 || pivots > max_pivots) {
                        st = 2;
                    } else {
                        a0 /= s; a1 /= s;
                        if (t < k) aFs[t] = a0;
                        if (t + 8 < k) aFs[t + 8] = a1;
                    }
                }
            }
            __syncwarp();

            // ---- residual at the current point (fp64, registers) and g_F = A_F' r
#pragma unroll
            for (int c = 0; c < NC; ++c) if (!skip) r[c] = (double)yv[c];
            for (int j = 0; j < kw; ++j) {
                if (!skip && j < k) {
                    const double aj = aFs[j];
                    const double *row = At64 + (size_t)idx[j] * RS + 2 * t;
#pragma unroll
                    for (int v = 0; v < LQ; ++v) {
                        const double2 lo = *reinterpret_cast<const double2 *>(row + 16 * v);
                        const double2 hi = *reinterpret_cast<const double2 *>(row + RS / 2 + 16 * v);
                        r[4 * v + 0] -= lo.x * aj; r[4 * v + 1] -= lo.y * aj;
                        r[4 * v + 2] -= hi.x * aj; r[4 * v + 3] -= hi.y * aj;
                    }
                }
            }
            double p0v = 0.0, p1v = 0.0;     // g_F of my members, then K g_F
            for (int j = 0; j < kw; ++j) {
                double s = 0.0;
                if (!skip && j < k) {
                    const double *row = At64 + (size_t)idx[j] * RS + 2 * t;
#pragma unroll
                    for (int v = 0; v < LQ; ++v) {
                        const double2 lo = *reinterpret_cast<const double2 *>(row + 16 * v);
                        const double2 hi = *reinterpret_cast<const double2 *>(row + RS / 2 + 16 * v);
                        s += lo.x * r[4 * v + 0]; s += lo.y * r[4 * v + 1];
                        s += hi.x * r[4 * v + 2]; s += hi.y * r[4 * v + 3];
                    }
                }
                s = gsum(s);
                if (t == (j & 7)) { if (j < 8) p0v = s; else p1v = s; }
            }
            // ---- two solves in one sweep: q = K 1, pv = K g_F (right-hand sides in registers)
            q0 = (t < k) ? 1.0 : 0.0; q1 = (t + 8 < k) ? 1.0 : 0.0;
            for (int j = 0; j < kw; ++j) {          // forward: L z = rhs
                const bool on = !skip && j < k;
                const double dj = on ? Lf[tri(j) + j] : 0.0;
                const double zq = __shfl_sync(FULL, ((j < 8) ? q0 : q1) * dj, j & 7, 8);
                const double zp = __shfl_sync(FULL, ((j < 8) ? p0v : p1v) * dj, j & 7, 8);
                if (on) {
                    if (t == (j & 7)) { if (j < 8) { q0 = zq; p0v = zp; } else { q1 = zq; p1v = zp; } }
                    if (t > j && t < k) { const double l = Lf[o0 + j]; q0 -= l * zq; p0v -= l * zp; }
                    if (t + 8 > j && t + 8 < k) { const double l = Lf[o1 + j]; q1 -= l * zq; p1v -= l * zp; }
                }
            }
            for (int j = kw - 1; j >= 0; --j) {     // backward: L' x = z
                const bool on = !skip && j < k;
                const double dj = on ? Lf[tri(j) + j] : 0.0;
                const double zq = __shfl_sync(FULL, ((j < 8) ? q0 : q1) * dj, j & 7, 8);
                const double zp = __shfl_sync(FULL, ((j < 8) ? p0v : p1v) * dj, j & 7, 8);
                if (on) {
                    if (t == (j & 7)) { if (j < 8) { q0 = zq; p0v = zp; } else { q1 = zq; p1v = zp; } }
                    if (t < j) { const double l = Lf[tri(j) + t]; q0 -= l * zq; p0v -= l * zp; }
                    if (t + 8 < j) { const double l = Lf[tri(j) + t + 8]; q1 -= l * zq; p1v -= l * zp; }
                }
            }
            const double sqn = gsum(q0 + q1);
            const double sp = gsum(p0v + p1v);
            const double suma = gsum(a0 + a1);
            bool accepted = false;
            {
                const double mu = (sp - (1.0 - suma)) / sqn;
                const double t0v = a0 + p0v - mu * q0, t1v = a1 + p1v - mu * q1;
                const bool m0 = t < k, m1 = t + 8 < k;
                const double amin = gmin(fmin(m0 ? t0v : INFINITY, m1 ? t1v : INFINITY));
                const bool ratio = !skip && !(amin > 0.0);
                // ---- ratio step towards the trial point until the first coefficient reaches zero; drop it
                double tt = INFINITY;
                if (m0 && !(t0v > 0.0)) { const double den = a0 - t0v; tt = fmin(tt, den > 0.0 ? a0 / den : 0.0); }
                if (m1 && !(t1v > 0.0)) { const double den = a1 - t1v; tt = fmin(tt, den > 0.0 ? a1 / den : 0.0); }
                double alpha = fmin(1.0, gmin(tt));
                if (alpha < 0.0) alpha = 0.0;
                const double n0v = a0 + alpha * (t0v - a0), n1v = a1 + alpha * (t1v - a1);
                bool b0 = false, b1 = false;
                if (m0 && !(t0v > 0.0)) { const double den = a0 - t0v; b0 = (den > 0.0 ? a0 / den : 0.0) <= alpha; }
                if (m1 && !(t1v > 0.0)) { const double den = a1 - t1v; b1 = (den > 0.0 ? a1 / den : 0.0) <= alpha; }
                const bool keep0 = m0 && !b0 && (n0v > 0.0), keep1 = m1 && !b1 && (n1v > 0.0);
                // ranks of the kept members: ballots over the group, slot 0 members come first
                const unsigned bk0 = (__ballot_sync(FULL, keep0) >> (8 * g)) & 0xffu;
                const unsigned bk1 = (__ballot_sync(FULL, keep1) >> (8 * g)) & 0xffu;
                const double ssum = gsum((keep0 ? n0v : 0.0) + (keep1 ? n1v : 0.0));
                __syncwarp();       // every read of idx / aFs of this round precedes the writes below
                if (ratio) {
                    if (m0 && !keep0) state[i0] = (i0 == last_added && alpha == 0.0) ? 2 : 0;
                    if (m1 && !keep1) state[i1] = (i1 == last_added && alpha == 0.0) ? 2 : 0;
                    const int r0 = __popc(bk0 & ((1u << t) - 1u));
                    const int r1 = __popc(bk0) + __popc(bk1 & ((1u << t) - 1u));
                    if (keep0) { idx[r0] = i0; aFs[r0] = n0v / ssum; }
                    if (keep1) { idx[r1] = i1; aFs[r1] = n1v / ssum; }
                    k = __popc(bk0) + __popc(bk1);
                    last_added = -1;
                    ++pivots;
                    if (k == 0 || pivots > max_pivots) st = 2;
                } else if (!skip) {
                    accepted = true;
                    a0 = m0 ? t0v : 0.0; a1 = m1 ? t1v : 0.0;
                    if (m0) aFs[t] = a0;
                    if (m1) aFs[t + 8] = a1;
                    sq = sqn;
                    if (m0) qv[t] = q0;
                    if (m1) qv[t + 8] = q1;
                }
                __syncwarp();
                if (ratio) {
                    a0 = 0.0; a1 = 0.0; i0 = 0; i1 = 0;
                    if (t < k) { a0 = aFs[t]; i0 = idx[t]; }
                    if (t + 8 < k) { a1 = aFs[t + 8]; i1 = idx[t + 8]; }
                }
            }
            // ---- accepted: residual, nu and multipliers at the new point
            const int kw2 = wmax(accepted ? k : 0);
            if (kw2 > 0) {
#pragma unroll
                for (int c = 0; c < NC; ++c) if (accepted) r[c] = (double)yv[c];
                for (int j = 0; j < kw2; ++j) {
                    if (accepted && j < k) {
                        const double aj = aFs[j];
                        const double *row = At64 + (size_t)idx[j] * RS + 2 * t;
#pragma unroll
                        for (int v = 0; v < LQ; ++v) {
                            const double2 lo = *reinterpret_cast<const double2 *>(row + 16 * v);
                            const double2 hi = *reinterpret_cast<const double2 *>(row + RS / 2 + 16 * v);
                            r[4 * v + 0] -= lo.x * aj; r[4 * v + 1] -= lo.y * aj;
                            r[4 * v + 2] -= hi.x * aj; r[4 * v + 3] -= hi.y * aj;
                        }
                    }
                }
                float rf[NC];
#pragma unroll
                for (int c = 0; c < NC; ++c) rf[c] = (float)r[c];
                // g_i = A_i' r for every endmember, 4 at a time (fp32 dot products of the fp64 residual)
                for (int c4 = 0; c4 < RP / 4; ++c4) {
                    float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float *row = At32 + (size_t)(4 * c4 + e) * RS + 4 * t;
#pragma unroll
                        for (int v = 0; v < LQ; ++v) {
                            const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
                            acc[e] = fmaf(a4.x, rf[4 * v + 0], acc[e]); acc[e] = fmaf(a4.y, rf[4 * v + 1], acc[e]);
                            acc[e] = fmaf(a4.z, rf[4 * v + 2], acc[e]); acc[e] = fmaf(a4.w, rf[4 * v + 3], acc[e]);
                        }
                    }
                    const float tot = reduce4(acc[0], acc[1], acc[2], acc[3], t);
                    if (accepted && !(t & 1)) gs[4 * c4 + (t >> 1)] = tot;
                }
                __syncwarp();
                float nu = 0.0f;
                if (accepted) {
                    if (t < k) nu += gs[i0] * (float)a0;
                    if (t + 8 < k) nu += gs[i1] * (float)a1;
                }
                nu = gsum(nu);
                const float4 g4 = *reinterpret_cast<const float4 *>(gs + 4 * t);
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
        }

        const bool wr = (st == 1 || st == 2);
        // ---- coefficients (exact zeros off the support), staged in endmember order
        if (wr) *reinterpret_cast<float4 *>(gs + 4 * t) = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        __syncwarp();
        if (wr) {
            if (t < k) gs[i0] = (float)a0;
            if (t + 8 < k) gs[i1] = (float)a1;
        }
        __syncwarp();
        if (wr) {
            const float4 o = *reinterpret_cast<const float4 *>(gs + 4 * t);
            if (cvec_ok && 4 * t < R) *reinterpret_cast<float4 *>(cout + 4 * t) = o;
            else {
                const float ov[4] = {o.x, o.y, o.z, o.w};
                for (int q = 0; q < 4; ++q) if (4 * t + q < R) cout[4 * t + q] = ov[q];
            }
        }
        // ---- residual (fallback: the loop left r at another point)
        if (__any_sync(FULL, st == 2)) {
            const bool fb = (st == 2);
            const int kf = wmax(fb ? k : 0);
#pragma unroll
            for (int c = 0; c < NC; ++c) if (fb) r[c] = (double)yv[c];
            for (int j = 0; j < kf; ++j) {
                if (fb && j < k) {
                    const double aj = aFs[j];
                    const double *row = At64 + (size_t)idx[j] * RS + 2 * t;
#pragma unroll
                    for (int v = 0; v < LQ; ++v) {
                        const double2 lo = *reinterpret_cast<const double2 *>(row + 16 * v);
                        const double2 hi = *reinterpret_cast<const double2 *>(row + RS / 2 + 16 * v);
                        r[4 * v + 0] -= lo.x * aj; r[4 * v + 1] -= lo.y * aj;
                        r[4 * v + 2] -= hi.x * aj; r[4 * v + 3] -= hi.y * aj;
                    }
                }
            }
            if (fb) info |= LINMIN_INFO_FINISH_FALLBACK;
        }
        if (prm.resid) {
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < NC; ++c) s += r[c] * r[c];
            s = gsum(s);
            if (wr && t == 0) prm.resid[p] = (float)sqrt(s / (double)L);
        }
        // ---- uncertainty propagation (reading R3)
        if (prm.coeff_sigma) {
            float sv[NC];
            bool sbad = false;
            if (prm.has_sigma) {
                const float *sp = prm.sigma + p * prm.sigma_stride;
#pragma unroll
                for (int v = 0; v < LQ; ++v) {
                    const int l = 4 * (t + 8 * v);
                    if (svec_ok && l + 3 < L) {
                        float4 t4 = *reinterpret_cast<const float4 *>(sp + l);
                        sv[4 * v + 0] = t4.x; sv[4 * v + 1] = t4.y; sv[4 * v + 2] = t4.z; sv[4 * v + 3] = t4.w;
                    } else {
#pragma unroll
                        for (int qq = 0; qq < 4; ++qq) sv[4 * v + qq] = (l + qq < L) ? sp[l + qq] : 1.0f;
                    }
#pragma unroll
                    for (int qq = 0; qq < 4; ++qq) sbad |= !(sv[4 * v + qq] > 0.0f) || !isfinite(sv[4 * v + qq]);
                }
            } else {
#pragma unroll
                for (int c = 0; c < NC; ++c) sv[c] = 1.0f;
            }
            sbad = ((__ballot_sync(FULL, sbad) >> (8 * g)) & 0xffu) != 0u;
            if (wr && sbad) info |= LINMIN_INFO_BAD_SIGMA;
            const bool doj = (st == 1) && !sbad && k > 1;
            const int kj = wmax(doj ? k : 0);
            if (wr) { sgs[t] = 0.0f; sgs[t + 8] = 0.0f; }
            if (kj > 0) {
                // W = L^-1 in place, row by row (row i of L is copied out first: its entries are
                // overwritten by W_ij while other lanes still need L_im)
                for (int i = 1; i < kj; ++i) {
                    const bool on = doj && i < k;
                    if (on) {
                        if (t < i) rowb[t] = Lf[tri(i) + t];
                        if (t + 8 < i) rowb[t + 8] = Lf[tri(i) + t + 8];
                    }
                    __syncwarp();
                    if (on) {
                        const double di = Lf[tri(i) + i];
                        for (int j = t; j < i; j += 8) {
                            double s = rowb[j] * Lf[tri(j) + j];
                            for (int m = j + 1; m < i; ++m) s += rowb[m] * Lf[tri(m) + j];
                            Lf[tri(i) + j] = -di * s;
                        }
                    }
                    __syncwarp();
                }
                // H = W'W - q q'/(1'q), packed lower, fp32
                if (doj) {
                    const double rs = 1.0 / sq;
                    for (int i = 0; i < k; ++i) {
                        const double qi = qv[i];
                        for (int j = t; j <= i; j += 8) {
                            double s = 0.0;
                            for (int m = i; m < k; ++m) s += Lf[tri(m) + i] * Lf[tri(m) + j];
                            Hp[tri(i) + j] = (float)(s - qi * qv[j] * rs);
                        }
                    }
                }
                __syncwarp();
                // expand to a zero-padded square (overlays the factor, which is dead now)
                if (doj) {
                    for (int e = t; e < KM * KM; e += 8) {
                        const int i = e >> 4, j = e & 15;
                        const int hi = max(i, j), lo = min(i, j);
                        Hs[e] = (hi < k) ? Hp[tri(hi) + lo] : 0.0f;
                    }
                }
                __syncwarp();
                // J = H A_F' on my channels, IT support members at a time; sigma_i^2 = sum_l (J_il s_l)^2
                for (int ib = 0; ib < kj; ib += IT) {
                    float d[IT][NC];
#pragma unroll
                    for (int ii = 0; ii < IT; ++ii)
#pragma unroll
                        for (int c = 0; c < NC; ++c) d[ii][c] = 0.0f;
                    for (int j = 0; j < kj; ++j) {
                        if (doj && j < k && ib < k) {
                            float hh[IT];
                            if (IT == 4) {
                                const float4 h4 = *reinterpret_cast<const float4 *>(Hs + j * KM + ib);
                                hh[0] = h4.x; hh[1] = h4.y; hh[IT - 2] = h4.z; hh[IT - 1] = h4.w;
                            } else {
                                const float2 h2 = *reinterpret_cast<const float2 *>(Hs + j * KM + ib);
                                hh[0] = h2.x; hh[1] = h2.y;
                            }
                            const float *row = At32 + (size_t)idx[j] * RS + 4 * t;
#pragma unroll
                            for (int v = 0; v < LQ; ++v) {
                                const float4 a4 = *reinterpret_cast<const float4 *>(row + 32 * v);
#pragma unroll
                                for (int ii = 0; ii < IT; ++ii) {
                                    d[ii][4 * v + 0] = fmaf(hh[ii], a4.x, d[ii][4 * v + 0]);
                                    d[ii][4 * v + 1] = fmaf(hh[ii], a4.y, d[ii][4 * v + 1]);
                                    d[ii][4 * v + 2] = fmaf(hh[ii], a4.z, d[ii][4 * v + 2]);
                                    d[ii][4 * v + 3] = fmaf(hh[ii], a4.w, d[ii][4 * v + 3]);
                                }
                            }
                        }
                    }
                    float acc[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
                    for (int ii = 0; ii < IT; ++ii)
#pragma unroll
                        for (int c = 0; c < NC; ++c) {
                            const float ds = d[ii][c] * sv[c];
                            acc[ii] = fmaf(ds, ds, acc[ii]);
                        }
                    const float tot = reduce4(acc[0], acc[1], acc[2], acc[3], t);
                    if (doj && !(t & 1) && (t >> 1) < IT && ib + (t >> 1) < k) sgs[ib + (t >> 1)] = sqrtf(tot);
                }
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

inline bool finish8_supported(int L, int R) { return R <= 32 && L <= 256; }

template <int LQ>
inline cudaError_t launch_finish8_lq(const LibView &lv, const SolveParams &prm, int sm_count,
                                     unsigned int *counter, unsigned int *overflow, cudaStream_t stream) {
    const size_t cta = (f8::cta_bytes(lv.R, LQ) + 15) & ~(size_t)15;
    const size_t per_warp = 4 * (size_t)f8::PIX_BYTES;
    int warps = (int)std::min<size_t>(16, (226 * 1024 - cta) / per_warp);
    if (warps < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = cta + per_warp * warps;
    cudaError_t e = cudaFuncSetAttribute(finish8_kernel<LQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t groups = (prm.N + 3) / 4;
    const int64_t need = (groups + warps - 1) / warps;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, sm_count));
    finish8_kernel<LQ><<<grid, warps * 32, smem, stream>>>(lv, prm, counter, overflow);
    return cudaGetLastError();
}

// counter and overflow[0] must be zero (the caller clears them on the stream)
inline cudaError_t launch_finish8(const LibView &lv, const SolveParams &prm, int sm_count,
                                  unsigned int *counter, unsigned int *overflow, cudaStream_t stream) {
    if (lv.L <= 128) return launch_finish8_lq<4>(lv, prm, sm_count, counter, overflow, stream);
    return launch_finish8_lq<8>(lv, prm, sm_count, counter, overflow, stream);
}

}  // namespace linmin
