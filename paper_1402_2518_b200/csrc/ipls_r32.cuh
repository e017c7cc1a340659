// ipls_r32.cuh -- register-blocked projection + IPLS kernel for R = 32 endmembers (sm_100a), v4.
//
// Same iteration as ipls_generic.cuh (Mehrotra predictor-corrector on the centred normal equations;
// PAPER.md:71-73 names IPLS and prints no steps -- DESIGN.md reading R1), mapped to the hardware:
//
//   * 8 lanes cooperate on one pixel, 4 pixels per warp, 8 warps per SM (255 registers, no spill traffic
//     on the dependent chains).  Lane t of a group owns rows i = t + 8 s (s = 0..3, cyclic) of the
//     32 x 32 Newton matrix M = G + diag(lambda/a): row i is kept in REGISTERS up to column 8 s + 7, as
//     40 packed pairs (80 registers), so that the rank-one updates are FFMA2 (fma.rn.f32x2).
//   * Start point (Mehrotra's heuristic for this QP): the sum-constrained LS point of the regularised
//     problem, x = Gi b - q (1'Gi b - 1)/(1'q) with Gi = (G + 1e-4 max G_ii I)^-1 precomputed per library,
//     and its reduced gradient as multipliers, both shifted into the interior.  5.8 iterations on the
//     OMEGA-like cubes instead of 10.1 from the barycentre.
//   * Square-root-free Cholesky M = L D L', right-looking, fully unrolled (static register indices).
//     Step k: every lane puts its raw entries of column k on a double-buffered, bank-padded shared
//     line, one __syncwarp, every lane reads the column back with LDS.128 (16 FMAs per load) and forms
//     1/d_k itself.  Column k + 1 is updated and exchanged BEFORE the rest of the rank-one update of
//     step k (look-ahead), so the shared-memory round trip overlaps the FFMA2 stream.
//   * The forward substitution of the predictor (right-hand sides 1 and -w) is fused into the
//     factorisation: the two right-hand sides ride along as a packed pair per row.
//   * Blocked substitutions: every lane forms its row of the inverse of the four 8 x 8 diagonal blocks
//     of L (under the FFMA2 stream of the factorisation, as soon as a block is final); a substitution is then 7 exchanges through shared memory (all-gather in the forward,
//     reduce-scatter in the backward direction) instead of a 31-step shuffle chain.
//   * G, Gi (padded rows), the centred library (re-laid out so that a lane's four rows are one LDS.128)
//     and the channel means live in shared memory, loaded once per CTA; warps run independently on
//     groups of 4 pixels taken from a global atomic counter; the spectrum of the NEXT group is fetched
//     with cp.async while the current one iterates.
//
// Algorithmic work per pixel: 2 L R + it (R^3/3 + 8 R^2 + 30 R) flops.
#pragma once
#include "common.cuh"

namespace linmin {

namespace r32 {

constexpr int R = 32;
constexpr int GST = 36;        // padded row stride of G in shared memory (bank-conflict-free LDS.128)
constexpr int XST = 56;        // one exchange line: 32 column entries + 8 x 2 right-hand sides + pad
constexpr int TBO = 2 * XST;   // diagonal blocks of -L: [4][8][8] floats
constexpr int RSO = TBO + 256; // reduce-scatter buffers: 2 x [8][12] floats
constexpr int AGO = RSO + 192; // all-gather buffers: 2 x 8 floats
constexpr int PIXF = 584;      // fixed floats per pixel (576 used; 584 = 8 mod 32 spreads the pixels),
                               // followed by two spectrum buffers of lpad(L) floats (this pixel, the next one)
constexpr int WARPS = 8;      // warps per CTA, one CTA per SM
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ float gsum(float v) { return group_sum<8>(v); }   // over the 8 lanes of a pixel
__device__ __forceinline__ float gmin(float v) { return group_min<8>(v); }
__device__ __forceinline__ float gmax(float v) { return group_max<8>(v); }

// shared-memory footprint in floats
__host__ __device__ inline int lpad(int L) { return (L + 3) & ~3; }
__host__ __device__ inline size_t smem_floats(int L) {
    return (size_t)2 * R * GST + 3 * R         // Gp, Gip, row sums of Gi (and their total), row sums of G
           + (size_t)lpad(L) * R + lpad(L)      // Acp, c
           + (size_t)WARPS * 4 * (PIXF + 2 * lpad(L));
}

// column j of the register-resident matrix (static j)
#define LM_COL(s, j) (((j) & 1) ? m2[s][(j) >> 1].y : m2[s][(j) >> 1].x)

// ---- exchanges inside a pixel group (8 lanes) through shared memory; consecutive calls alternate buffers
// all-gather: every lane contributes one value and receives all eight
__device__ __forceinline__ void allgather8(float *buf, int t, float v, float4 &lo, float4 &hi) {
    buf[t] = v;
    __syncwarp();
    lo = *reinterpret_cast<const float4 *>(buf);
    hi = *reinterpret_cast<const float4 *>(buf + 4);
}
// reduce-scatter: every lane contributes eight values, lane t receives the sum of the lanes' value t
__device__ __forceinline__ float reduce_scatter8(float *buf, int t, const float2 (&c)[4]) {
    *reinterpret_cast<float4 *>(buf + t * 12) = make_float4(c[0].x, c[0].y, c[1].x, c[1].y);
    *reinterpret_cast<float4 *>(buf + t * 12 + 4) = make_float4(c[2].x, c[2].y, c[3].x, c[3].y);
    __syncwarp();
    const float s0 = buf[0 * 12 + t] + buf[1 * 12 + t], s1 = buf[2 * 12 + t] + buf[3 * 12 + t];
    const float s2 = buf[4 * 12 + t] + buf[5 * 12 + t], s3 = buf[6 * 12 + t] + buf[7 * 12 + t];
    return (s0 + s1) + (s2 + s3);
}
__device__ __forceinline__ float2 dot8(const float2 &p0, const float2 &p1, const float2 &p2, const float2 &p3,
                                       const float4 &lo, const float4 &hi) {
    float2 a = fma2(p0, make_float2(lo.x, lo.y), make_float2(0.0f, 0.0f));
    float2 b = fma2(p2, make_float2(hi.x, hi.y), make_float2(0.0f, 0.0f));
    a = fma2(p1, make_float2(lo.z, lo.w), a);
    b = fma2(p3, make_float2(hi.z, hi.w), b);
    return make_float2(a.x + b.x, a.y + b.y);
}

// Blocked substitutions.  L is unit lower, m2 holds -L (zeros on and above the diagonal of the 8 x 8
// diagonal blocks T_s), ti[s] is row t of T_s^-1 (the lane's own row).  The dependent chain is 7
// shared-memory exchanges instead of 31 shuffle steps.
// L z = r:  z_s = T_s^-1 (r_s - sum_{s' < s} L_{s s'} z_{s'})
__device__ __forceinline__ void forward_subst_blk(const float2 (&m2)[4][16], const float2 (&ti)[4][4],
                                                  float (&r)[4], float *ag, int t) {
    float4 zl[3], zh[3];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
        float rp = r[s];
#pragma unroll
        for (int sp = 0; sp < s; ++sp) {
            const float2 d = dot8(m2[s][4 * sp], m2[s][4 * sp + 1], m2[s][4 * sp + 2], m2[s][4 * sp + 3], zl[sp], zh[sp]);
            rp += d.x + d.y;
        }
        float4 gl, gh;
        allgather8(ag, t, rp, gl, gh);
        const float2 d = dot8(ti[s][0], ti[s][1], ti[s][2], ti[s][3], gl, gh);
        r[s] = d.x + d.y;
        if (s < 3) allgather8(ag + 8, t, r[s], zl[s], zh[s]);
    }
}
// L' x = y:  x_s = T_s^-T (y_s - sum_{s' > s} L_{s' s}' x_{s'}); every lane adds its row's share, the
// shares are summed by reduce-scatter
__device__ __forceinline__ void backward_subst_blk(const float2 (&m2)[4][16], const float2 (&ti)[4][4],
                                                   float (&y)[4], float *rs, int t) {
    float2 acc[3][4];
#pragma unroll
    for (int s = 0; s < 3; ++s)
#pragma unroll
        for (int jp = 0; jp < 4; ++jp) acc[s][jp] = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int s = 3; s >= 0; --s) {
        if (s < 3) y[s] += reduce_scatter8(rs, t, acc[s]);
        float2 c[4];
#pragma unroll
        for (int jp = 0; jp < 4; ++jp) c[jp] = make_float2(ti[s][jp].x * y[s], ti[s][jp].y * y[s]);
        y[s] = reduce_scatter8(rs + 96, t, c);
#pragma unroll
        for (int sp = 0; sp < s; ++sp)
#pragma unroll
            for (int jp = 0; jp < 4; ++jp) acc[sp][jp] = fma2(y[s], m2[s][4 * sp + jp], acc[sp][jp]);
    }
}

}  // namespace r32

__global__ void __launch_bounds__(r32::WARPS * 32, 1)
ipls_r32_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter) {
    using namespace r32;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0] & 1) return;      // non-finite library: the caller is told (status or poisoned outputs)
    const int L = lib.L;
    const int Lp = lpad(L);
    float *Gp = smem;                        // [32][GST]
    float *Gip = Gp + R * GST;               // [32][GST] inverse of the regularised G (start point)
    float *Giq = Gip + R * GST;              // [32] row sums of Gi, [32] their total
    float *Grs = Giq + 2 * R;                // [32] row sums of G
    float *Acp = Grs + R;                    // [Lp][32]: Acp[l][t*4+s] = Ac[l][t+8s]
    float *cv = Acp + (size_t)Lp * R;        // [Lp]
    const int lane = threadIdx.x & 31, g = lane >> 3, t = lane & 7;
    float *pix = cv + Lp + (size_t)((threadIdx.x >> 5) * 4 + g) * (PIXF + 2 * Lp);
    float *xb0 = pix;                        // exchange line, buffer 0
    float *xb1 = pix + XST;                  // buffer 1
    float *Tb = pix + TBO;                   // diagonal blocks of -L
    float *rsb = pix + RSO;                  // reduce-scatter buffers
    float *agb = pix + AGO;                  // all-gather buffers
    float *yb0 = pix + PIXF;                 // spectrum buffers: the current pixel and the prefetched next one
    float *yb1 = yb0 + Lp;

    // ---- once per CTA: stage the library data
    for (int e = threadIdx.x; e < R * R; e += blockDim.x) {
        Gp[(e >> 5) * GST + (e & 31)] = lib.Gc[e];
        Gip[(e >> 5) * GST + (e & 31)] = lib.Gi[e];
    }
    for (int e = threadIdx.x; e < Lp * R; e += blockDim.x) {
        int l = e >> 5, c = e & 31, tt = c >> 2, s = c & 3;
        Acp[e] = (l < L) ? lib.Ac[(size_t)l * R + tt + 8 * s] : 0.0f;
    }
    for (int l = threadIdx.x; l < Lp; l += blockDim.x) cv[l] = (l < L) ? lib.c[l] : 0.0f;
    __syncthreads();
    if (threadIdx.x < R) Giq[threadIdx.x] = lib.Giq[threadIdx.x];
    __syncthreads();
    if (threadIdx.x == 0) {
        float s = 0.0f;
        for (int j = 0; j < R; ++j) s += Giq[j];
        Giq[R] = s;
    }
    if (threadIdx.x >= 32 && threadIdx.x < 32 + R) {
        float s = 0.0f;
        for (int j = 0; j < R; ++j) s += Gp[(threadIdx.x - 32) * GST + j];
        Grs[threadIdx.x - 32] = s;
    }
    __syncthreads();

    const float gdmax = lib.scal[0];
    const float tau = 0.995f;
    const float pivot_floor = 1e-12f * gdmax;
    // one-hot pairs of my position inside a diagonal block: adds lambda/a to the diagonal with FFMA2
    float2 e2[4];
#pragma unroll
    for (int jp = 0; jp < 4; ++jp) e2[jp] = make_float2((t == 2 * jp) ? 1.0f : 0.0f, (t == 2 * jp + 1) ? 1.0f : 0.0f);

    // spectra arrive by cp.async (16 B per lane and step) one task ahead of their use
    const bool vec_ok = ((L & 3) == 0) && ((prm.ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.Y) & 15) == 0);
    // work counter: the atomic for task i + 2 is issued at the start of task i and read at its end
    auto take_ticket = [&]() -> unsigned int { return (lane == 0) ? atomicAdd(counter, 1u) : 0u; };
    auto prefetch = [&](unsigned int grp_, float *dst) {
        const int64_t q0 = (int64_t)grp_ * 4;
        if (q0 >= prm.N) return;
        const int64_t q = (q0 + g < prm.N) ? (q0 + g) : (prm.N - 1);
        const float *src = prm.Y + q * prm.ldY;
        if (vec_ok) {
            for (int l = 4 * t; l < Lp; l += 32) {
                const unsigned sa = (unsigned)__cvta_generic_to_shared(dst + l);
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sa), "l"(src + l) : "memory");
            }
        } else {
            for (int l = t; l < Lp; l += 8) dst[l] = (l < L) ? src[l] : 0.0f;
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    unsigned int grp = __shfl_sync(FULL, take_ticket(), 0);
    unsigned int grp_next = __shfl_sync(FULL, take_ticket(), 0);
    prefetch(grp, yb0);
    int par = 0;
    while (true) {
        const int64_t p0 = (int64_t)grp * 4;
        if (p0 >= prm.N) break;
        const bool valid = (p0 + g) < prm.N;
        const int64_t p = valid ? (p0 + g) : (prm.N - 1);
        float *ybuf = par ? yb1 : yb0;
        const unsigned int ticket = take_ticket();
        prefetch(grp_next, par ? yb0 : yb1);
        if ((int64_t)grp_next * 4 < prm.N) asm volatile("cp.async.wait_group 1;" ::: "memory");
        else asm volatile("cp.async.wait_group 0;" ::: "memory");
        __syncwarp();

        // ---- centre my chunks of the spectrum in place, flag non-finite values
        bool bad = false;
        for (int l = 4 * t; l < Lp; l += 32) {
            float4 y4 = *reinterpret_cast<const float4 *>(ybuf + l);
            const float4 c4 = *reinterpret_cast<const float4 *>(cv + l);
            bad |= !isfinite(y4.x) || !isfinite(y4.y) || !isfinite(y4.z) || !isfinite(y4.w);
            y4.x -= c4.x; y4.y -= c4.y; y4.z -= c4.z; y4.w -= c4.w;
            *reinterpret_cast<float4 *>(ybuf + l) = y4;
        }
        bad = __any_sync(0xffu << (8 * g), bad);
        __syncwarp();
        if (bad) for (int l = t; l < Lp; l += 8) ybuf[l] = 0.0f;
        __syncwarp();

        // ---- projection b = Ac'(y - c)
        float2 b01 = make_float2(0.0f, 0.0f), b23 = make_float2(0.0f, 0.0f);
        {
            float2 c01 = make_float2(0.0f, 0.0f), c23 = make_float2(0.0f, 0.0f);
#pragma unroll 4
            for (int l4 = 0; l4 < Lp; l4 += 4) {
                const float4 y4 = *reinterpret_cast<const float4 *>(ybuf + l4);
                const float4 a0 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 0) * R + t * 4);
                const float4 a1 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 1) * R + t * 4);
                const float4 a2 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 2) * R + t * 4);
                const float4 a3 = *reinterpret_cast<const float4 *>(Acp + (size_t)(l4 + 3) * R + t * 4);
                b01 = fma2(y4.x, make_float2(a0.x, a0.y), b01); b23 = fma2(y4.x, make_float2(a0.z, a0.w), b23);
                c01 = fma2(y4.y, make_float2(a1.x, a1.y), c01); c23 = fma2(y4.y, make_float2(a1.z, a1.w), c23);
                b01 = fma2(y4.z, make_float2(a2.x, a2.y), b01); b23 = fma2(y4.z, make_float2(a2.z, a2.w), b23);
                c01 = fma2(y4.w, make_float2(a3.x, a3.y), c01); c23 = fma2(y4.w, make_float2(a3.z, a3.w), c23);
            }
            b01.x += c01.x; b01.y += c01.y; b23.x += c23.x; b23.y += c23.y;
        }
        const float b[4] = {b01.x, b01.y, b23.x, b23.y};
        float bmax = gmax(fmaxf(fmaxf(fabsf(b[0]), fabsf(b[1])), fmaxf(fabsf(b[2]), fabsf(b[3]))));
        const float sc = fmaxf(bmax, 1e-3f * gdmax);

        // ---- start (Mehrotra's heuristic on this QP): x = the sum-constrained LS point of the regularised
        //      problem, lambda = its reduced gradient, both shifted into the interior
        float a[4], lam[4], w[4], Ga[4];
        float nu, lam0;
        {
            __syncwarp();
#pragma unroll
            for (int s = 0; s < 4; ++s) xb1[t + 8 * s] = b[s];
            __syncwarp();
            float2 x2[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) x2[s] = make_float2(0.0f, 0.0f);
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float4 b4 = *reinterpret_cast<const float4 *>(xb1 + 4 * c);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const float4 g4 = *reinterpret_cast<const float4 *>(Gip + (t + 8 * s) * GST + 4 * c);
                    x2[s] = fma2(make_float2(g4.x, g4.y), make_float2(b4.x, b4.y), x2[s]);
                    x2[s] = fma2(make_float2(g4.z, g4.w), make_float2(b4.z, b4.w), x2[s]);
                }
            }
            float x[4], q[4], sx = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) { x[s] = x2[s].x + x2[s].y; q[s] = Giq[t + 8 * s]; sx += x[s]; }
            sx = gsum(sx);
            const float mu0 = (sx - 1.0f) * rcp_approx(Giq[R]);
#pragma unroll
            for (int s = 0; s < 4; ++s) { x[s] = fmaf(-mu0, q[s], x[s]); xb0[t + 8 * s] = x[s]; }
            __syncwarp();
#pragma unroll
            for (int s = 0; s < 4; ++s) x2[s] = make_float2(0.0f, 0.0f);
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float4 b4 = *reinterpret_cast<const float4 *>(xb0 + 4 * c);
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const float4 g4 = *reinterpret_cast<const float4 *>(Gp + (t + 8 * s) * GST + 4 * c);
                    x2[s] = fma2(make_float2(g4.x, g4.y), make_float2(b4.x, b4.y), x2[s]);
                    x2[s] = fma2(make_float2(g4.z, g4.w), make_float2(b4.z, b4.w), x2[s]);
                }
            }
            float gx = 0.0f, mnx = INFINITY, mng = INFINITY;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                Ga[s] = x2[s].x + x2[s].y;                  // G x
                lam[s] = Ga[s] - b[s];                      // gradient at x
                gx = fmaf(lam[s], x[s], gx);
                mnx = fminf(mnx, x[s]); mng = fminf(mng, lam[s]);
            }
            gx = gsum(gx); mnx = gmin(mnx); mng = gmin(mng);
            nu = -gx;
            const float dp = fmaxf(-mnx, 0.0f), dd = fmaxf(-(mng + nu), 0.0f);
            float xl = 0.0f, sl = 0.0f, sxx = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                x[s] += dp; lam[s] += nu + dd;
                xl = fmaf(x[s], lam[s], xl); sl += lam[s]; sxx += x[s];
            }
            xl = gsum(xl); sl = gsum(sl); sxx = gsum(sxx);
            const float dp2 = 0.05f * xl * rcp_approx(fmaxf(sl, 1e-30f)), dd2 = 0.05f * xl * rcp_approx(fmaxf(sxx, 1e-30f));
            float sa = 0.0f, lm = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                a[s] = x[s] + dp2 + 1e-3f;
                lam[s] = lam[s] + dd2 + 1e-4f * sc;
                sa += a[s]; lm = fmaxf(lm, lam[s]);
            }
            sa = gsum(sa); lam0 = gmax(lm);
            const float rsa = 1.0f / sa;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                a[s] *= rsa;
                Ga[s] = fmaf(dp + dp2 + 1e-3f, Grs[t + 8 * s], Ga[s]) * rsa;     // G a of the shifted, normalised point
            }
            if (!(lam0 > 0.0f) || !isfinite(lam0) || !isfinite(sa)) {     // degenerate data: fall back to the flat start
                lam0 = fmaxf(bmax, 1e-3f * gdmax);
#pragma unroll
                for (int s = 0; s < 4; ++s) { a[s] = 1.0f / 32.0f; lam[s] = lam0; Ga[s] = Grs[t + 8 * s] * (1.0f / 32.0f); }
                nu = 0.0f;
            }
        }
        int iters = 0, flags = bad ? LINMIN_INFO_NONFINITE_INPUT : 0;
        bool done = false;
        for (int it = 0;; ++it) {
            // ---- rows of M (lower part) from G.  G a is not recomputed: the Newton system gives
            //      G da = (r1 - dnu 1) - d o da row by row, so G a is carried along with a (no exchange of a,
            //      no loads of the upper part of G: 80 wavefronts less on the shared-memory pipe per iteration)
            float2 m2[4][16];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
#pragma unroll
                for (int c = 0; c < 2 * s + 2; ++c) {
                    const float4 g4 = *reinterpret_cast<const float4 *>(Gp + (t + 8 * s) * GST + 4 * c);
                    m2[s][2 * c] = make_float2(g4.x, g4.y);
                    m2[s][2 * c + 1] = make_float2(g4.z, g4.w);
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
            // ---- M = G + diag(lambda / a)
            float ainv[4], d[4], dinv[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                ainv[s] = rcp_approx(a[s]);
                d[s] = lam[s] * ainv[s];
                dinv[s] = 0.0f;
#pragma unroll
                for (int jp = 0; jp < 4; ++jp) m2[s][4 * s + jp] = fma2(d[s], e2[jp], m2[s][4 * s + jp]);
            }
            // ---- M = L D L' (right-looking), with the predictor's forward substitution riding along:
            //      rr[s] = (row of L^-1 1, row of L^-1 (-w)).  m2 ends as -L (strictly lower; zeros on and
            //      above the diagonal inside the diagonal blocks), dinv = 1 / d.
            float2 rr[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) rr[s] = make_float2(1.0f, -w[s]);
            // Diagonal blocks of -L go to shared memory as soon as they are final, and every lane forms its row
            // of T_s^-1 (x_j = [j == t] + sum_{i > j} x_i (-L)_{i j}) two steps later, under the FFMA2 stream of
            // the factorisation instead of in a latency-bound phase of its own.
            float2 ti[4][4];
#define TINV_STORE(s_)                                                                                          \
    {                                                                                                           \
        *reinterpret_cast<float4 *>(Tb + (s_) * 64 + t * 8) =                                                   \
            make_float4(m2[s_][4 * (s_)].x, m2[s_][4 * (s_)].y, m2[s_][4 * (s_) + 1].x, m2[s_][4 * (s_) + 1].y); \
        *reinterpret_cast<float4 *>(Tb + (s_) * 64 + t * 8 + 4) = make_float4(                                  \
            m2[s_][4 * (s_) + 2].x, m2[s_][4 * (s_) + 2].y, m2[s_][4 * (s_) + 3].x, m2[s_][4 * (s_) + 3].y);    \
    }
#define TINV_ROWS(s_)                                                                            \
    {                                                                                            \
        float T[8][8];                                                                           \
        _Pragma("unroll") for (int i = 1; i < 8; ++i) {                                          \
            const float4 u = *reinterpret_cast<const float4 *>(Tb + (s_) * 64 + i * 8);          \
            T[i][0] = u.x; T[i][1] = u.y; T[i][2] = u.z; T[i][3] = u.w;                          \
            if (i > 4) {                                                                         \
                const float4 v = *reinterpret_cast<const float4 *>(Tb + (s_) * 64 + i * 8 + 4);  \
                T[i][4] = v.x; T[i][5] = v.y; T[i][6] = v.z; T[i][7] = v.w;                      \
            }                                                                                    \
        }                                                                                        \
        float x[8];                                                                              \
        _Pragma("unroll") for (int j = 7; j >= 0; --j) {                                         \
            float v = (t == j) ? 1.0f : 0.0f;                                                    \
            _Pragma("unroll") for (int i = j + 1; i < 8; ++i) v = fmaf(x[i], T[i][j], v);        \
            x[j] = v;                                                                            \
        }                                                                                        \
        _Pragma("unroll") for (int jp = 0; jp < 4; ++jp) ti[s_][jp] = make_float2(x[2 * jp], x[2 * jp + 1]); \
    }
            bool clamped = false;
            // Look-ahead schedule: column k + 1 is updated and put on the exchange line BEFORE the rest of
            // the rank-one update of step k, so that the shared-memory round trip of step k + 1 overlaps
            // the FFMA2 stream of step k.  l4[c] / zk hold column k (raw) and the row-k right-hand sides.
            float4 l4[8];
            float2 zk;
            {
#pragma unroll
                for (int s = 0; s < 4; ++s) xb0[t + 8 * s] = LM_COL(s, 0);
                __syncwarp();
                zk = make_float2(__shfl_sync(FULL, rr[0].x, 0, 8), __shfl_sync(FULL, rr[0].y, 0, 8));
#pragma unroll
                for (int c = 0; c < 8; ++c) l4[c] = *reinterpret_cast<const float4 *>(xb0 + 4 * c);
            }
#define L4C(j) ((((j) & 3) == 0) ? l4[(j) >> 2].x : ((((j) & 3) == 1) ? l4[(j) >> 2].y : ((((j) & 3) == 2) ? l4[(j) >> 2].z : l4[(j) >> 2].w)))
#pragma unroll
            for (int k = 0; k < 31; ++k) {
                const int s0 = k >> 3, t0 = k & 7;
                const int k1 = k + 1, s1 = k1 >> 3;
                if (k == 7) TINV_STORE(0)
                if (k == 15) TINV_STORE(1)
                if (k == 23) TINV_STORE(2)
                if (k == 9) TINV_ROWS(0)
                if (k == 17) TINV_ROWS(1)
                if (k == 25) TINV_ROWS(2)
                float piv = L4C(k);
                if (!(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
                const float rinv = rcp_approx(piv);
                const float nrinv = -rinv;
                float nl[4];
#pragma unroll
                for (int s = s0; s < 4; ++s) {
                    float v = LM_COL(s, k) * nrinv;
                    if (s == s0) v = (t > t0) ? v : 0.0f;      // rows at or above k: no update, store 0
                    nl[s] = v;
                    if (k & 1) m2[s][k >> 1].y = v; else m2[s][k >> 1].x = v;
                    rr[s] = fma2(v, zk, rr[s]);
                }
                dinv[s0] = (t == t0) ? rinv : dinv[s0];
                // ---- look-ahead: column k + 1 first, then its exchange
                {
                    const float ck1 = L4C(k1);
#pragma unroll
                    for (int s = s1; s < 4; ++s) {
                        if (k1 & 1) m2[s][k1 >> 1].y = fmaf(nl[s], ck1, m2[s][k1 >> 1].y);
                        else m2[s][k1 >> 1].x = fmaf(nl[s], ck1, m2[s][k1 >> 1].x);
                    }
                }
                const float *cb = (k1 & 1) ? xb1 : xb0;
                if (k1 < 31) {
                    float *cw = (k1 & 1) ? xb1 : xb0;
#pragma unroll
                    for (int s = s1; s < 4; ++s) cw[t + 8 * s] = LM_COL(s, k1);
                    __syncwarp();
                    // right-hand sides of row k + 1: two shuffles (off the pivot chain) instead of a store and
                    // a load on the shared-memory pipe, which is the busiest unit of this kernel
                    zk = make_float2(__shfl_sync(FULL, rr[s1].x, k1 & 7, 8), __shfl_sync(FULL, rr[s1].y, k1 & 7, 8));
                }
                // ---- rest of the rank-one update of step k (columns k + 2 ..), chunk by chunk; a chunk of
                //      column k is replaced by the same chunk of column k + 1 as soon as it has been used
                //      (one column buffer in registers; the pivot chunk is reloaded first)
#pragma unroll
                for (int c = k1 >> 2; c < 8; ++c) {
                    if (c >= ((k + 2) >> 2)) {
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
                            const int jp = 2 * c + h, j0 = 2 * jp;
                            const float2 cp = h ? make_float2(l4[c].z, l4[c].w) : make_float2(l4[c].x, l4[c].y);
                            if (j0 >= k + 2) {
#pragma unroll
                                for (int s = s0; s < 4; ++s)
                                    if (j0 < 8 * s + 8) m2[s][jp] = fma2(nl[s], cp, m2[s][jp]);
                            } else if (j0 + 1 == k + 2) {
#pragma unroll
                                for (int s = s0; s < 4; ++s)
                                    if (j0 < 8 * s + 8) m2[s][jp].y = fmaf(nl[s], cp.y, m2[s][jp].y);
                            }
                        }
                    }
                    if (k1 < 31) l4[c] = *reinterpret_cast<const float4 *>(cb + 4 * c);
                }
            }
#undef L4C
            {   // k = 31: only the last pivot (its owner has it) -- nothing left to update
                float piv = m2[3][15].y;
                if (t == 7 && !(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
                dinv[3] = (t == 7) ? rcp_approx(piv) : dinv[3];
                m2[3][15].y = 0.0f;
            }
            if (__any_sync(0xffu << (8 * g), clamped)) flags |= LINMIN_INFO_CHOL_REGULARISED;
            // ---- last diagonal block (blocks 0..2 were inverted under the factorisation)
            TINV_STORE(3)
            __syncwarp();
            TINV_ROWS(3)
#undef TINV_STORE
#undef TINV_ROWS
            // ---- predictor: M^-1 = L^-T D^-1 L^-1; nu eliminated through L^-1 1
            float sww = 0.0f, swz = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const float zd = rr[s].x * dinv[s];
                sww = fmaf(zd, rr[s].x, sww);
                swz = fmaf(zd, rr[s].y, swz);
            }
            sww = gsum(sww); swz = gsum(swz);
            const float rsww = 1.0f / sww;
            float dnu = (swz + rp) * rsww;
            float da[4], dl[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) da[s] = fmaf(-rr[s].x, dnu, rr[s].y) * dinv[s];
            backward_subst_blk(m2, ti, da, rsb, t);
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
            float cc[4], r1[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                cc[s] = fmaf(sg, mu, -da[s] * dl[s]);
                r1[s] = fmaf(cc[s], ainv[s], -w[s]);
            }
            forward_subst_blk(m2, ti, r1, agb, t);
            swz = 0.0f;
#pragma unroll
            for (int s = 0; s < 4; ++s) swz = fmaf(rr[s].x * dinv[s], r1[s], swz);
            swz = gsum(swz);
            dnu = (swz + rp) * rsww;
#pragma unroll
            for (int s = 0; s < 4; ++s) da[s] = fmaf(-rr[s].x, dnu, r1[s]) * dinv[s];
            backward_subst_blk(m2, ti, da, rsb, t);
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
                Ga[s] = fmaf(ap, fmaf(cc[s], ainv[s], -w[s]) - dnu - d[s] * da[s], Ga[s]);
                a[s] = fmaxf(fmaf(ap, da[s], a[s]), 1e-18f);
                lam[s] = fmaxf(fmaf(ad, dl[s], lam[s]), 1e-18f * lam0);
            }
            nu = fmaf(ad, dnu, nu);
        }

        // ---- store the iterate (coalesced: 8 lanes x float4 = one 128 B row) and the info word
        __syncwarp();
#pragma unroll
        for (int s = 0; s < 4; ++s) xb0[t + 8 * s] = (a[s] * sc > LINMIN_TAPIA_KAPPA * lam[s]) ? a[s] : 0.0f;
        __syncwarp();
        if (valid) {
            float4 o = *reinterpret_cast<const float4 *>(xb0 + 4 * t);
            *reinterpret_cast<float4 *>(prm.coeffs + p * R + 4 * t) = o;
            if (prm.info && t == 0) prm.info[p] = flags | (iters << 8);
        }
        __syncwarp();
        grp = grp_next;
        grp_next = __shfl_sync(FULL, ticket, 0);
        par ^= 1;
    }
}
#undef LM_COL

inline bool ipls_r32_supported(int L) {
    return r32::smem_floats(L) * sizeof(float) <= 226 * 1024;
}

// counter: device word, zero (the caller clears it on the stream before the launch)
inline cudaError_t launch_ipls_r32(const LibView &lv, const SolveParams &prm, int sm_count,
                                   unsigned int *counter, cudaStream_t stream) {
    size_t smem = r32::smem_floats(lv.L) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(ipls_r32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int64_t groups = (prm.N + 3) / 4;
    int64_t need = (groups + r32::WARPS - 1) / r32::WARPS;
    int grid = (int)std::max<int64_t>(1, std::min<int64_t>(need, (int64_t)sm_count));
    ipls_r32_kernel<<<grid, r32::WARPS * 32, smem, stream>>>(lv, prm, counter);
    return cudaGetLastError();
}

}  // namespace linmin
