// finish_fast.cuh -- exact finish + uncertainty + residual for R <= 64 (supports up to 32 members), L <= 512 (sm_100a).
//
// Same mathematics as finish.cuh (read its header: PAPER.md:54-68 optimality conditions,
// PAPER.md:88 uncertainty reading R3, PAPER.md:143 RMS reading R8), re-mapped for speed:
//   * one warp per pixel; lane q owns channels {4 q + 128 v} (y and the fp64 residual stay in
//     registers), lane j < k owns support member j (its coefficient, its row of the k x k factor
//     for the substitutions), lane i < R owns endmember i when multipliers are evaluated;
//   * the library is staged once per CTA in shared memory, TRANSPOSED and padded
//     (At[r][128 LV + 4]) so that the three L-sized passes -- residual, A_F'r, A'r, J = H A_F' --
//     are LDS.128 streams without bank conflicts; the fp64 Gram matrix sits beside it;
//   * triangular solves keep the right-hand sides in registers and broadcast one value per step by
//     shuffle (no shared-memory round trip, no barrier); 1/sqrt in fp64 is an fp32 MUFU seed plus
//     two Newton steps;
//   * warps fetch pixels from a global counter (the number of support changes varies per pixel).
#pragma once
#include "common.cuh"
#include "finish.cuh"

namespace linmin {
namespace ff {

constexpr unsigned FULL = 0xffffffffu;
constexpr int KM = 32;

__host__ __device__ inline int ast(int LV) { return 128 * LV + 4; }
__host__ __device__ inline size_t g64_bytes(int R) { return ((size_t)R * R * 8 + 15) & ~(size_t)15; }
__host__ __device__ inline size_t cta_bytes(int R, int LV) { return g64_bytes(R) + (size_t)R * ast(LV) * 4; }
__host__ __device__ inline size_t warp_bytes(int LV) {
    return (size_t)(KM * (KM + 1) / 2) * 8   // Lf
           + (size_t)KM * 8 + 64 * 8         // aFs, tmp (by endmember: up to 64)
           + (size_t)KM * KM * 4             // Hs
           + (size_t)128 * LV * 4            // rbuf
           + (size_t)KM * 4 + 64;            // idx, state (by endmember)
}

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(FULL, v, src); }
__device__ __forceinline__ double warp_min_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmin(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
// 1/sqrt(x) in fp64 from the fp32 MUFU seed (x must be representable in fp32 range)
__device__ __forceinline__ double rsqrt_d(double x) {
    double y = (double)rsqrtf((float)x);
    double hx = 0.5 * x;
    y = y * (1.5 - hx * y * y);
    y = y * (1.5 - hx * y * y);
    return y;
}
// sums of 4 values over the warp with 6 shuffles; lanes with (lane >> 3) == i end with the total of v_i
__device__ __forceinline__ float reduce4(float v0, float v1, float v2, float v3, int lane) {
    const bool hi = lane & 16;
    float s0 = hi ? v0 : v2, s1 = hi ? v1 : v3;       // what goes to the partner
    float k0 = hi ? v2 : v0, k1 = hi ? v3 : v1;       // what stays
    k0 += __shfl_xor_sync(FULL, s0, 16);
    k1 += __shfl_xor_sync(FULL, s1, 16);
    const bool h2 = lane & 8;
    float s = h2 ? k0 : k1, k = h2 ? k1 : k0;
    k += __shfl_xor_sync(FULL, s, 8);
    k += __shfl_xor_sync(FULL, k, 4);
    k += __shfl_xor_sync(FULL, k, 2);
    k += __shfl_xor_sync(FULL, k, 1);
    return k;
}

}  // namespace ff

// RH = 1: R <= 32, lane i owns endmember i; RH = 2: R <= 64, lane i owns endmembers i and i + 32.  The support is capped
// at KM = 32 members either way; with RH = 2 a pixel that needs more goes to `overflow` ([0] = count, [1 + i] = pixel)
// untouched and is finished by the any-size kernel.
template <int LV, int RH>
__global__ void __launch_bounds__(512, 1)
finish_fast_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter,
                   const unsigned int *__restrict__ list /* NULL: all pixels; else [0] = count, [1 + i] = pixel */,
                   unsigned int *__restrict__ overflow) {
    using namespace ff;
    if ((list && list[0] == 0u) || lib.flags[0]) return;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int L = lib.L, R = lib.R;
    const bool cons = lib.cons != 0;      // false: positivity only (no normalisation, mu == nu == 0, H = K, empty support allowed)
    const int AST = ast(LV);
    double *G64s = (double *)smem_raw;                    // [R][R]
    float *At = (float *)(smem_raw + g64_bytes(R));        // [R][AST], zero padded beyond L (16 B aligned)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char *wb = smem_raw + ((cta_bytes(R, LV) + 15) & ~(size_t)15) + (size_t)warp * ((warp_bytes(LV) + 15) & ~(size_t)15);
    double *Lf = (double *)wb;                             // packed lower, column-major, runtime k
    double *aFs = Lf + KM * (KM + 1) / 2;                  // [KM] coefficients on the support
    double *tmp = aFs + KM;                                // [KM]
    float *Hs = (float *)(tmp + 64);                       // [KM][KM] symmetric   (tmp: [64], by endmember)
    float *rbuf = Hs + KM * KM;                            // [128 LV] fp32 residual
    int *idx = (int *)(rbuf + 128 * LV);                   // [KM]
    unsigned char *state = (unsigned char *)(idx + KM);    // [64] by endmember: 0 free, 1 in F, 2 blocked

    for (int e = threadIdx.x; e < R * R; e += blockDim.x) G64s[e] = lib.G64[e];
    for (int e = threadIdx.x; e < R * AST; e += blockDim.x) {
        int r = e / AST, l = e - r * AST;
        At[e] = (l < L) ? lib.A[(size_t)l * R + r] : 0.0f;
    }
    __syncthreads();

    const bool vec_ok = ((prm.ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.Y) & 15) == 0);
    const bool svec_ok = prm.has_sigma && ((prm.sigma_stride & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.sigma) & 15) == 0);
    const float qnan = __int_as_float(0x7fc00000);
    const int max_pivots = 4 * KM + 8;
    const unsigned lt_mask = (1u << lane) - 1u;

    while (true) {
        unsigned int pu = 0;
        if (lane == 0) pu = atomicAdd(counter, 1u);
        pu = __shfl_sync(FULL, pu, 0);
        int64_t p = (int64_t)pu;
        if (list) {
            if (pu >= list[0]) break;
            p = (int64_t)list[1 + pu];
        }
        if (p >= prm.N) break;
        float *cout = prm.coeffs + p * R;
        int info = prm.info ? prm.info[p] : 0;

        // ---- spectrum -> registers
        float yv[4 * LV];
        const float *yp = prm.Y + p * prm.ldY;
        bool bad = false;
#pragma unroll
        for (int v = 0; v < LV; ++v) {
            const int l = 4 * lane + 128 * v;
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
        if (__any_sync(FULL, bad)) {
#pragma unroll
            for (int h = 0; h < RH; ++h) {
                const int e = lane + 32 * h;
                if (e < R) {
                    cout[e] = qnan;
                    if (prm.coeff_sigma) prm.coeff_sigma[p * R + e] = qnan;
                }
            }
            if (lane == 0) {
                if (prm.resid) prm.resid[p] = qnan;
                if (prm.info) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            }
            continue;
        }
        // ---- initial support from the IPLS iterate; lane j < k owns support member j
        int k;
        int myidx = 0;
        double aF = 0.0;
        {
            float ai[RH];
            bool in[RH];
            unsigned m[2] = {0u, 0u};
#pragma unroll
            for (int h = 0; h < RH; ++h) {
                ai[h] = (lane + 32 * h < R) ? cout[lane + 32 * h] : -1.0f;
                in[h] = ai[h] > LINMIN_SUPPORT_THRESHOLD;
                m[h] = __ballot_sync(FULL, in[h]);
            }
            if ((m[0] | m[1]) == 0u && cons) {   // can not happen for a point of the simplex; be safe: largest entry
                float best = warp_max(RH > 1 ? fmaxf(ai[0], ai[RH - 1]) : ai[0]);
                m[0] = __ballot_sync(FULL, ai[0] == best);
                m[0] = m[0] & (0u - m[0]);
                if (RH > 1) { m[1] = m[0] ? 0u : __ballot_sync(FULL, ai[RH - 1] == best); m[1] = m[1] & (0u - m[1]); }
#pragma unroll
                for (int h = 0; h < RH; ++h) { in[h] = (m[h] >> lane) & 1u; ai[h] = 1.0f; }
            }
            k = __popc(m[0]) + __popc(m[1]);
            if (RH > 1 && k > KM) {          // wider than this kernel's cap: the any-size kernel takes the pixel as it is
                if (lane == 0 && overflow) { const unsigned slot = atomicAdd(overflow, 1u); overflow[1 + slot] = (unsigned)p; }
                continue;
            }
#pragma unroll
            for (int h = 0; h < RH; ++h) {
                const int rank = (h ? __popc(m[0]) : 0) + __popc(m[h] & lt_mask);
                if (lane + 32 * h < R) state[lane + 32 * h] = in[h] ? 1 : 0;
                if (in[h]) { idx[rank] = lane + 32 * h; aFs[rank] = (double)ai[h]; }
            }
            __syncwarp();
            if (lane < k) { myidx = idx[lane]; aF = aFs[lane]; }
            double s = warp_sum(aF);
            if (cons) aF /= s;
            if (lane < k) aFs[lane] = aF;
            __syncwarp();
        }

        int pivots = 0, last_added = -1;
        bool fallback = false;
        double r[4 * LV];
        double dinv = 0.0, q = 0.0;     // lane j: 1/L_jj and (K 1)_j of the current factor
        double sq = 1.0;
        while (true) {
            // ---- gather G_FF; lane i builds row i
            {
                int off = 0;
                for (int j = 0; j < k; ++j) {
                    if (lane >= j && lane < k) Lf[off + lane - j] = G64s[myidx * R + idx[j]];
                    off += k - j;
                }
            }
            __syncwarp();
            // ---- Cholesky (fp64), left-looking; lane i owns row i
            int rej = -1;
            {
                int offj = 0;
                for (int j = 0; j < k; ++j) {
                    double s = 0.0, gjj = Lf[offj];
                    if (lane >= j && lane < k) {
                        s = Lf[offj + lane - j];
                        int offk = 0;
                        for (int kk = 0; kk < j; ++kk) {
                            s -= Lf[offk + lane - kk] * Lf[offk + j - kk];
                            offk += k - kk;
                        }
                    }
                    double sj = shfl_d(s, j);
                    if (!(sj > 1e-13 * gjj)) { rej = j; break; }
                    double dj = rsqrt_d(sj);
                    if (lane > j && lane < k) Lf[offj + lane - j] = s * dj;
                    if (lane == j) dinv = dj;
                    __syncwarp();
                    offj += k - j;
                }
            }
            if (rej >= 0) {
                // A_F lost rank at member `rej` (R9): drop it, block it, stay at the same point
                bool keep = (lane < k) && (lane != rej);
                if (lane == rej) state[myidx] = 2;
                unsigned km = __ballot_sync(FULL, keep);
                int rank = __popc(km & lt_mask);
                __syncwarp();
                if (keep) { idx[rank] = myidx; aFs[rank] = aF; }
                k = __popc(km);
                __syncwarp();
                last_added = -1;
                if (k == 0 && cons) { fallback = true; break; }
                myidx = 0; aF = 0.0;
                if (lane < k) { myidx = idx[lane]; aF = aFs[lane]; }
                double s = warp_sum(aF);
                if (cons) aF /= s;
                if (lane < k) aFs[lane] = aF;
                __syncwarp();
                if (++pivots > max_pivots) { fallback = true; break; }
                continue;
            }
            // ---- residual at the current point (fp64, registers) and g_F = A_F' r
#pragma unroll
            for (int c = 0; c < 4 * LV; ++c) r[c] = (double)yv[c];
            for (int j = 0; j < k; ++j) {
                const double aj = aFs[j];
                const float *row = At + idx[j] * AST + 4 * lane;
#pragma unroll
                for (int v = 0; v < LV; ++v) {
                    float4 a4 = *reinterpret_cast<const float4 *>(row + 128 * v);
                    r[4 * v + 0] -= (double)a4.x * aj; r[4 * v + 1] -= (double)a4.y * aj;
                    r[4 * v + 2] -= (double)a4.z * aj; r[4 * v + 3] -= (double)a4.w * aj;
                }
            }
            double gF = 0.0;
            for (int j = 0; j < k; ++j) {
                const float *row = At + idx[j] * AST + 4 * lane;
                double s = 0.0;
#pragma unroll
                for (int v = 0; v < LV; ++v) {
                    float4 a4 = *reinterpret_cast<const float4 *>(row + 128 * v);
                    s += (double)a4.x * r[4 * v + 0]; s += (double)a4.y * r[4 * v + 1];
                    s += (double)a4.z * r[4 * v + 2]; s += (double)a4.w * r[4 * v + 3];
                }
                s = warp_sum(s);
                if (lane == j) gF = s;
            }
            // ---- two solves in one sweep: q = K 1, pv = K g_F (right-hand sides in registers)
            double x0 = (lane < k) ? 1.0 : 0.0, x1 = gF;
            {
                int offj = 0;
                for (int j = 0; j < k; ++j) {          // forward
                    double z0 = shfl_d(x0 * dinv, j), z1 = shfl_d(x1 * dinv, j);
                    if (lane == j) { x0 = z0; x1 = z1; }
                    if (lane > j && lane < k) {
                        double l = Lf[offj + lane - j];
                        x0 -= l * z0; x1 -= l * z1;
                    }
                    offj += k - j;
                }
                const int offme = lane * k - (lane * (lane - 1)) / 2;   // start of column `lane`
                for (int j = k - 1; j >= 0; --j) {     // backward: L' x = z
                    double z0 = shfl_d(x0 * dinv, j), z1 = shfl_d(x1 * dinv, j);
                    if (lane == j) { x0 = z0; x1 = z1; }
                    if (lane < j) {
                        double l = Lf[offme + j - lane];
                        x0 -= l * z0; x1 -= l * z1;
                    }
                }
            }
            q = x0;
            sq = warp_sum(q);
            const double sp = warp_sum(x1);
            const double suma = warp_sum(aF);
            const double mu = cons ? (sp - (1.0 - suma)) / sq : 0.0;
            const double atry = aF + x1 - mu * q;
            double amin = warp_min_d((lane < k) ? atry : INFINITY);
            if (!(amin > 0.0)) {
                // ---- ratio step towards atry until the first coefficient reaches zero; drop it
                double tt = INFINITY;
                if (lane < k && !(atry > 0.0)) {
                    double den = aF - atry;
                    tt = den > 0.0 ? aF / den : 0.0;
                }
                double alpha = fmin(1.0, warp_min_d(tt));
                if (alpha < 0.0) alpha = 0.0;
                double an = aF + alpha * (atry - aF);
                bool blocking = (lane < k) && !(atry > 0.0) && (tt <= alpha);
                bool keep = (lane < k) && !blocking && (an > 0.0);
                if (lane < k && !keep) state[myidx] = (myidx == last_added && alpha == 0.0) ? 2 : 0;
                unsigned km = __ballot_sync(FULL, keep);
                int rank = __popc(km & lt_mask);
                double s = warp_sum(keep ? an : 0.0);
                __syncwarp();
                if (keep) { idx[rank] = myidx; aFs[rank] = cons ? an / s : an; }
                k = __popc(km);
                __syncwarp();
                last_added = -1;
                myidx = 0; aF = 0.0;
                if (lane < k) { myidx = idx[lane]; aF = aFs[lane]; }
                if ((k == 0 && cons) || ++pivots > max_pivots) { fallback = true; break; }
                continue;
            }
            // ---- accept; residual, nu and multipliers at the new point
            aF = (lane < k) ? atry : 0.0;
            if (lane < k) aFs[lane] = aF;
            __syncwarp();
#pragma unroll
            for (int c = 0; c < 4 * LV; ++c) r[c] = (double)yv[c];
            for (int j = 0; j < k; ++j) {
                const double aj = aFs[j];
                const float *row = At + idx[j] * AST + 4 * lane;
#pragma unroll
                for (int v = 0; v < LV; ++v) {
                    float4 a4 = *reinterpret_cast<const float4 *>(row + 128 * v);
                    r[4 * v + 0] -= (double)a4.x * aj; r[4 * v + 1] -= (double)a4.y * aj;
                    r[4 * v + 2] -= (double)a4.z * aj; r[4 * v + 3] -= (double)a4.w * aj;
                }
            }
#pragma unroll
            for (int v = 0; v < LV; ++v)
                *reinterpret_cast<float4 *>(rbuf + 4 * lane + 128 * v) =
                    make_float4((float)r[4 * v + 0], (float)r[4 * v + 1], (float)r[4 * v + 2], (float)r[4 * v + 3]);
            __syncwarp();
            // g_i = A_i' r for every endmember (fp32 dot products of the fp64 residual); lane i
            float gi[RH];
#pragma unroll
            for (int h = 0; h < RH; ++h) {
                const float *row = At + (lane + 32 * h < R ? lane + 32 * h : 0) * AST;
                float g = 0.0f;
#pragma unroll 8
                for (int c = 0; c < 32 * LV; ++c) {
                    float4 a4 = *reinterpret_cast<const float4 *>(row + 4 * c);
                    float4 r4 = *reinterpret_cast<const float4 *>(rbuf + 4 * c);
                    g = fmaf(a4.x, r4.x, g); g = fmaf(a4.y, r4.y, g);
                    g = fmaf(a4.z, r4.z, g); g = fmaf(a4.w, r4.w, g);
                }
                gi[h] = g;
            }
            // nu = sum_{j in F} g_j a_j : bring a_F to endmember lanes through state/aFs
            int st[RH];
            float nus = 0.0f, gab = 0.0f;
            {
                // lane j < k holds (myidx, aF); scatter a_F to endmember order via shared memory
#pragma unroll
                for (int h = 0; h < RH; ++h) if (lane + 32 * h < R) tmp[lane + 32 * h] = 0.0;
                __syncwarp();
                if (lane < k) tmp[myidx] = aF;
                __syncwarp();
#pragma unroll
                for (int h = 0; h < RH; ++h) {
                    const bool live = lane + 32 * h < R;
                    st[h] = live ? state[lane + 32 * h] : 2;
                    nus = fmaf(gi[h], live ? (float)tmp[lane + 32 * h] : 0.0f, nus);
                    gab = fmaxf(gab, live ? fabsf(gi[h]) : 0.0f);
                }
            }
            const float nu = cons ? warp_sum(nus) : 0.0f;
            float li[RH], lmin = INFINITY;
#pragma unroll
            for (int h = 0; h < RH; ++h) { li[h] = (st[h] == 0) ? (nu - gi[h]) : INFINITY; lmin = fminf(lmin, li[h]); }
            const float gmaxv = warp_max(gab);
            const float lbest = warp_min(lmin);
            unsigned mm[2] = {0u, 0u};
#pragma unroll
            for (int h = 0; h < RH; ++h) mm[h] = __ballot_sync(FULL, li[h] == lbest && st[h] == 0);
            if (!(lbest < -1e-6f * gmaxv) || (mm[0] | mm[1]) == 0u) break;          // optimal
            if (k >= KM || pivots >= max_pivots) { fallback = true; break; }
            const int jadd = mm[0] ? (__ffs(mm[0]) - 1) : (32 + __ffs(mm[1]) - 1);
            if (lane == (jadd & 31)) state[jadd] = 1;
            if (lane == k) { myidx = jadd; aF = 0.0; idx[k] = jadd; aFs[k] = 0.0; }
            ++k; ++pivots; last_added = jadd;
            __syncwarp();
        }

        // ---- outputs: coefficients (exact zeros off the support)
        if (RH > 1 && fallback && k >= KM && overflow) {    // the support wants to outgrow the cap: any-size kernel
            if (lane == 0) { const unsigned slot = atomicAdd(overflow, 1u); overflow[1 + slot] = (unsigned)p; }
            __syncwarp();
            continue;
        }
        {
#pragma unroll
            for (int h = 0; h < RH; ++h) if (lane + 32 * h < R) tmp[lane + 32 * h] = 0.0;
            __syncwarp();
            if (lane < k) tmp[myidx] = aF;
            __syncwarp();
#pragma unroll
            for (int h = 0; h < RH; ++h) if (lane + 32 * h < R) cout[lane + 32 * h] = (float)tmp[lane + 32 * h];
        }
        if (fallback) {
#pragma unroll
            for (int c = 0; c < 4 * LV; ++c) r[c] = (double)yv[c];
            for (int j = 0; j < k; ++j) {
                const double aj = aFs[j];
                const float *row = At + idx[j] * AST + 4 * lane;
#pragma unroll
                for (int v = 0; v < LV; ++v) {
                    float4 a4 = *reinterpret_cast<const float4 *>(row + 128 * v);
                    r[4 * v + 0] -= (double)a4.x * aj; r[4 * v + 1] -= (double)a4.y * aj;
                    r[4 * v + 2] -= (double)a4.z * aj; r[4 * v + 3] -= (double)a4.w * aj;
                }
            }
            info |= LINMIN_INFO_FINISH_FALLBACK;
        }
        if (prm.resid) {
            double s = 0.0;
#pragma unroll
            for (int c = 0; c < 4 * LV; ++c) s += r[c] * r[c];
            s = warp_sum(s);
            if (lane == 0) prm.resid[p] = (float)sqrt(s / (double)L);
        }
        // ---- uncertainty propagation (reading R3)
        if (prm.coeff_sigma) {
            float *sout = prm.coeff_sigma + p * R;
            float sv[4 * LV];
            bool sbad = false;
            if (prm.has_sigma) {
                const float *sp = prm.sigma + p * prm.sigma_stride;
#pragma unroll
                for (int v = 0; v < LV; ++v) {
                    const int l = 4 * lane + 128 * v;
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
                for (int c = 0; c < 4 * LV; ++c) sv[c] = 1.0f;
            }
            sbad = __any_sync(FULL, sbad);
            float myout = 0.0f;                           // lane j < k: sigma of support member j
            if (sbad) {
                info |= LINMIN_INFO_BAD_SIGMA;
            } else if (k > (cons ? 1 : 0) && !fallback) {
                // W = L^-1 in place, columns from the last to the first (lane i owns row i)
                for (int j = k - 1; j >= 0; --j) {
                    const int offj = j * k - (j * (j - 1)) / 2;
                    if (lane > j && lane < k) tmp[lane] = Lf[offj + lane - j];
                    __syncwarp();
                    const double wjj = shfl_d(dinv, j);
                    if (lane > j && lane < k) {
                        double s = dinv * tmp[lane];
                        int offm = offj + (k - j);            // column j + 1
                        for (int m = j + 1; m < lane; ++m) {
                            s += Lf[offm + lane - m] * tmp[m];
                            offm += k - m;
                        }
                        Lf[offj + lane - j] = -s * wjj;
                    }
                    __syncwarp();
                }
                // H = W'W - q q'/(1'q), symmetric, fp32; lane i fills row i (j <= i) and its mirror
                {
                    const double rs = cons ? 1.0 / sq : 0.0;        // pos: H = K, no projection
                    int offj = 0;
                    for (int j = 0; j < k; ++j) {
                        const double qj = shfl_d(q, j), dj = shfl_d(dinv, j);
                        if (lane >= j && lane < k) {
                            // sum_{m >= lane} W(m, lane) W(m, j)
                            double s = dinv * ((lane == j) ? dj : Lf[offj + lane - j]);
                            int offl = lane * k - (lane * (lane - 1)) / 2;
                            for (int m = lane + 1; m < k; ++m) s += Lf[offl + m - lane] * Lf[offj + m - j];
                            float h = (float)(s - q * qj * rs);
                            Hs[j * KM + lane] = h;
                            Hs[lane * KM + j] = h;
                        }
                        offj += k - j;
                    }
                }
                __syncwarp();
                // J = H A_F' on my channels, 4 support members at a time; sigma_i^2 = sum_l (J_il s_l)^2
                for (int i0 = 0; i0 < k; i0 += 4) {
                    float d[4][4 * LV];
#pragma unroll
                    for (int ii = 0; ii < 4; ++ii)
#pragma unroll
                        for (int c = 0; c < 4 * LV; ++c) d[ii][c] = 0.0f;
                    for (int j = 0; j < k; ++j) {
                        const float4 h4 = *reinterpret_cast<const float4 *>(Hs + j * KM + i0);
                        const float hh[4] = {h4.x, h4.y, h4.z, h4.w};
                        const float *row = At + idx[j] * AST + 4 * lane;
#pragma unroll
                        for (int v = 0; v < LV; ++v) {
                            float4 a4 = *reinterpret_cast<const float4 *>(row + 128 * v);
#pragma unroll
                            for (int ii = 0; ii < 4; ++ii) {
                                d[ii][4 * v + 0] = fmaf(hh[ii], a4.x, d[ii][4 * v + 0]);
                                d[ii][4 * v + 1] = fmaf(hh[ii], a4.y, d[ii][4 * v + 1]);
                                d[ii][4 * v + 2] = fmaf(hh[ii], a4.z, d[ii][4 * v + 2]);
                                d[ii][4 * v + 3] = fmaf(hh[ii], a4.w, d[ii][4 * v + 3]);
                            }
                        }
                    }
                    float acc[4];
#pragma unroll
                    for (int ii = 0; ii < 4; ++ii) {
                        acc[ii] = 0.0f;
#pragma unroll
                        for (int c = 0; c < 4 * LV; ++c) {
                            float ds = d[ii][c] * sv[c];
                            acc[ii] = fmaf(ds, ds, acc[ii]);
                        }
                    }
                    float tot = ff::reduce4(acc[0], acc[1], acc[2], acc[3], lane);   // lanes 8 i..8 i+7: total of acc[i]
                    // member i0 + ii lives in lane i0 + ii: fetch from lane 8 ii
#pragma unroll
                    for (int ii = 0; ii < 4; ++ii) {
                        float v = __shfl_sync(FULL, tot, 8 * ii);
                        if (lane == i0 + ii) myout = sqrtf(v);
                    }
                }
            }
            // scatter to endmember order
#pragma unroll
            for (int h = 0; h < RH; ++h) if (lane + 32 * h < R) rbuf[lane + 32 * h] = 0.0f;
            __syncwarp();
            if (lane < k) rbuf[myidx] = myout;
            __syncwarp();
#pragma unroll
            for (int h = 0; h < RH; ++h) if (lane + 32 * h < R) sout[lane + 32 * h] = sbad ? qnan : rbuf[lane + 32 * h];
        }
        if (prm.info && lane == 0) {
            int pv = pivots > 255 ? 255 : pivots;
            prm.info[p] = (info & 0xffff) | (pv << 16) | (k << 24);
        }
        __syncwarp();
    }
}

inline bool finish_fast_supported(int L, int R) { return R <= 64 && L <= 512; }

inline int finish_fast_lv(int L) { return L <= 128 ? 1 : (L <= 256 ? 2 : 4); }

template <int LV, int RH>
inline cudaError_t launch_finish_fast_lv(const LibView &lv, const SolveParams &prm, int sm_count, unsigned int *counter,
                                         const unsigned int *list, unsigned int *overflow, cudaStream_t stream) {
    const size_t cta = (ff::cta_bytes(lv.R, LV) + 15) & ~(size_t)15;
    const size_t per_warp = (ff::warp_bytes(LV) + 15) & ~(size_t)15;
    if (cta + per_warp > 220 * 1024) return cudaErrorInvalidConfiguration;
    int warps = (int)std::min<size_t>(16, (220 * 1024 - cta) / per_warp);
    const size_t smem = cta + per_warp * warps;
    cudaError_t e = cudaFuncSetAttribute(finish_fast_kernel<LV, RH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int64_t need = (prm.N + warps - 1) / warps;
    int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, sm_count));
    finish_fast_kernel<LV, RH><<<grid, warps * 32, smem, stream>>>(lv, prm, counter, list, overflow);
    return cudaGetLastError();
}

// counter (and overflow[0], when given) must be zero (the caller clears them on the stream); list, overflow: see the kernel
inline cudaError_t launch_finish_fast(const LibView &lv, const SolveParams &prm, int sm_count, unsigned int *counter,
                                      const unsigned int *list, unsigned int *overflow, cudaStream_t stream) {
    if (lv.R <= 32) {
        switch (finish_fast_lv(lv.L)) {
            case 1: return launch_finish_fast_lv<1, 1>(lv, prm, sm_count, counter, list, overflow, stream);
            case 2: return launch_finish_fast_lv<2, 1>(lv, prm, sm_count, counter, list, overflow, stream);
            default: return launch_finish_fast_lv<4, 1>(lv, prm, sm_count, counter, list, overflow, stream);
        }
    }
    switch (finish_fast_lv(lv.L)) {
        case 1: return launch_finish_fast_lv<1, 2>(lv, prm, sm_count, counter, list, overflow, stream);
        case 2: return launch_finish_fast_lv<2, 2>(lv, prm, sm_count, counter, list, overflow, stream);
        default: return launch_finish_fast_lv<4, 2>(lv, prm, sm_count, counter, list, overflow, stream);
    }
}
// fits in shared memory with at least four warps?
inline bool finish_fast_fits(int L, int R) {
    const int LV = finish_fast_lv(L);
    const size_t cta = (ff::cta_bytes(R, LV) + 15) & ~(size_t)15, per_warp = (ff::warp_bytes(LV) + 15) & ~(size_t)15;
    return finish_fast_supported(L, R) && cta + 4 * per_warp <= 220 * 1024;
}

}  // namespace linmin
