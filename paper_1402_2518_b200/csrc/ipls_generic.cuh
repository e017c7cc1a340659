// ipls_generic.cuh -- projection + IPLS (primal-dual interior-point least squares), any R <= 256.
//
// PAPER.md:71-73 (sec. 2.2) names IPLS (Chouzenoux et al.) and states only that convexity of F
// gives convergence; it prints no steps (reading R1).  The iteration below is a standard
// Mehrotra predictor-corrector primal-dual method on the per-pixel QP
//      min 1/2 a'G a - b'a   s.t.  a >= 0 (multipliers lambda),  1'a = 1 (multiplier nu)
// with G = Ac'Ac, b = Ac'(y - c) (centred library, precompute.cuh).  Perturbed KKT system:
//      G a - b - lambda + nu 1 = 0,   1'a = 1,   a_i lambda_i = mu.
// One Newton step:  M = G + diag(lambda/a);  v = M^-1 1;  u = M^-1( -(G a - b + nu 1) + c/a );
//      dnu = (1'u + r_p)/(1'v);  da = u - v dnu;  dlambda = -lambda + c/a - (lambda/a) da;
// c = 0 (predictor), then c = sigma mu 1 - da_aff * dlambda_aff with sigma = (mu_aff/mu)^3
// (corrector); fraction-to-boundary 0.995, separate primal and dual step lengths.
//
// This generic kernel keeps everything of a pixel in shared memory and lets a TEAM of threads
// (a warp, or the whole CTA for R > 64) cooperate on the Cholesky factorisation and the triangular
// solves.  It is the any-size path; R = 32 has a register-blocked kernel of its own.  Like that kernel it
// starts from Mehrotra's heuristic point and carries G a along with a (no mat-vec per iteration).
#pragma once
#include "common.cuh"

namespace linmin {

template <int TEAM>
struct TeamOps;

template <>
struct TeamOps<32> {
    static __device__ __forceinline__ int tid() { return threadIdx.x & 31; }
    static __device__ __forceinline__ void sync() { __syncwarp(); }
    static __device__ __forceinline__ float sum(float v, float *) { return warp_sum(v); }
    static __device__ __forceinline__ float max(float v, float *) { return warp_max(v); }
    static __device__ __forceinline__ float min(float v, float *) { return warp_min(v); }
};

// the whole CTA is one team; `red` is a 2 x 32-float scratch area in shared memory
template <int TEAM>
struct TeamOps {
    static __device__ __forceinline__ int tid() { return threadIdx.x; }
    static __device__ __forceinline__ void sync() { __syncthreads(); }
    template <typename Op>
    static __device__ __forceinline__ float reduce(float v, float *red, Op op, float ident) {
        int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(0xffffffffu, v, o));
        if (lane == 0) red[w] = v;
        __syncthreads();
        float r = (lane < TEAM / 32) ? red[lane] : ident;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) r = op(r, __shfl_xor_sync(0xffffffffu, r, o));
        __syncthreads();
        return r;
    }
    static __device__ __forceinline__ float sum(float v, float *red) {
        return reduce(v, red, [](float a, float b) { return a + b; }, 0.0f);
    }
    static __device__ __forceinline__ float max(float v, float *red) {
        return reduce(v, red, [](float a, float b) { return fmaxf(a, b); }, -INFINITY);
    }
    static __device__ __forceinline__ float min(float v, float *red) {
        return reduce(v, red, [](float a, float b) { return fminf(a, b); }, INFINITY);
    }
};

// In-place left-looking Cholesky of the packed (column-major lower) n x n matrix Mp.
// dinv[j] = 1/L_jj.  The diagonal slot of row i carries the running pivot M_ii - sum_{k<j} L_ik^2: the
// thread that finishes L_ij subtracts its square at once, so the pivot of column j is ONE load for every
// thread instead of a j-term recomputation (that loop was half of the kernel's work).
// A pivot below `floorv` is clamped (returns true if that happened).
template <int TEAM, typename T>
__device__ __forceinline__ bool team_cholesky(T *Mp, T *dinv, int n, T floorv) {
    using Ops = TeamOps<TEAM>;
    const int t = Ops::tid();
    bool clamped = false;
    for (int j = 0; j < n; ++j) {
        T sj = Mp[cm(n, j, j)];
        if (!(sj > floorv)) { sj = floorv; clamped = true; }
        const T dj = (T)1 / sqrt(sj);
        if (t == 0) dinv[j] = dj;
        // Rows j+1 .. n-1 of column j: L_ij = (M_ij - sum_{k<j} L_ik L_jk) / L_jj.  When fewer rows than
        // threads remain, g = 2, 4, .. 32 lanes (of one warp) share a row: each takes every g-th term of the
        // sum and the parts are added by shuffles, so the late columns (long sums, few rows) keep the whole
        // team busy instead of leaving most of it at the barrier.
        const int nr = n - 1 - j;
        int g = 1;
        while (g < 32 && nr * (g * 2) <= TEAM) g <<= 1;
        const int rows_per_pass = TEAM / g;
        const int part = t & (g - 1), rl = t / g;
        for (int r0 = 0; r0 < nr; r0 += rows_per_pass) {
            const int i = j + 1 + r0 + rl;
            const bool active = i < n;
            const int ii = active ? i : j;                      // a valid row for the loads of idle lanes
            // element (r, k) of the packed matrix sits at cb(k) + r with cb(k) = k (n - 1) - k (k - 1)/2
            // my terms k = part, part + g, ..: cb advances by d, d shrinks by g^2 (no multiply in the loop);
            // four partial sums keep four load pairs in flight
            T s0 = 0, s1 = 0, s2 = 0, s3 = 0;
            int k = part;
            int c = k * (n - 1) - ((k * (k - 1)) >> 1);
            int d = g * (n - 1) - ((g * (g - 1)) >> 1) - g * k;
            const int g2 = g * g;
            for (; k + 3 * g < j; k += 4 * g) {
                const int c0 = c, c1 = c0 + d, c2 = c1 + d - g2, c3 = c2 + d - 2 * g2;
                s0 += Mp[c0 + ii] * Mp[c0 + j];
                s1 += Mp[c1 + ii] * Mp[c1 + j];
                s2 += Mp[c2 + ii] * Mp[c2 + j];
                s3 += Mp[c3 + ii] * Mp[c3 + j];
                c = c3 + d - 3 * g2;
                d -= 4 * g2;
            }
            for (; k < j; k += g) { s0 += Mp[c + ii] * Mp[c + j]; c += d; d -= g2; }
            T s = (s0 + s1) + (s2 + s3);
            for (int o = g >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (active && part == 0) {
                s = (Mp[cm(n, i, j)] - s) * dj;
                Mp[cm(n, i, j)] = s;
                Mp[cm(n, i, i)] -= s * s;
            }
        }
        Ops::sync();
    }
    return clamped;
}

// Solve (L L') x = rhs in place for NRHS right-hand sides stored at x[0], x[1] (each n long).
template <int TEAM, int NRHS, typename T>
__device__ __forceinline__ void team_solve(const T *Mp, const T *dinv, int n, T *x0, T *x1) {
    using Ops = TeamOps<TEAM>;
    const int t = Ops::tid();
    if constexpr (TEAM == 32) {
        // one warp, n <= 64: the right-hand sides live in registers (rows t and t + 32) and x_j travels by
        // shuffle; a step is shuffle + FMA instead of store / barrier / load through shared memory
        const int r1 = t + 32;
        const bool h0 = t < n, h1 = r1 < n;
        T a0 = h0 ? x0[t] : (T)0, b0 = h1 ? x0[r1] : (T)0;
        T a1 = (NRHS > 1 && h0) ? x1[t] : (T)0, b1 = (NRHS > 1 && h1) ? x1[r1] : (T)0;
        const T d0 = h0 ? dinv[t] : (T)0, d1 = h1 ? dinv[r1] : (T)0;
        for (int j = 0; j < n; ++j) {      // forward: L z = rhs
            const T dj = dinv[j];
            const T z0 = __shfl_sync(0xffffffffu, (j < 32) ? a0 : b0, j & 31) * dj;
            const T z1 = NRHS > 1 ? __shfl_sync(0xffffffffu, (j < 32) ? a1 : b1, j & 31) * dj : (T)0;
            if (h0 && t > j) { const T l = Mp[cm(n, t, j)]; a0 -= l * z0; if (NRHS > 1) a1 -= l * z1; }
            if (h1 && r1 > j) { const T l = Mp[cm(n, r1, j)]; b0 -= l * z0; if (NRHS > 1) b1 -= l * z1; }
        }
        a0 *= d0; b0 *= d1; a1 *= d0; b1 *= d1;
        for (int j = n - 1; j >= 0; --j) { // backward: L' x = z
            const T dj = dinv[j];
            const T z0 = __shfl_sync(0xffffffffu, (j < 32) ? a0 : b0, j & 31) * dj;
            const T z1 = NRHS > 1 ? __shfl_sync(0xffffffffu, (j < 32) ? a1 : b1, j & 31) * dj : (T)0;
            if (t < j) { const T l = Mp[cm(n, j, t)]; a0 -= l * z0; if (NRHS > 1) a1 -= l * z1; }
            if (r1 < j) { const T l = Mp[cm(n, j, r1)]; b0 -= l * z0; if (NRHS > 1) b1 -= l * z1; }
        }
        if (h0) { x0[t] = a0 * d0; if (NRHS > 1) x1[t] = a1 * d0; }
        if (h1) { x0[r1] = b0 * d1; if (NRHS > 1) x1[r1] = b1 * d1; }
        Ops::sync();
    } else {
    for (int j = 0; j < n; ++j) {          // forward: L z = rhs
        T z0 = x0[j] * dinv[j];
        T z1 = NRHS > 1 ? x1[j] * dinv[j] : (T)0;
        for (int i = j + 1 + t; i < n; i += TEAM) {
            T l = Mp[cm(n, i, j)];
            x0[i] -= l * z0;
            if (NRHS > 1) x1[i] -= l * z1;
        }
        Ops::sync();
    }
    for (int i = t; i < n; i += TEAM) {
        x0[i] *= dinv[i];
        if (NRHS > 1) x1[i] *= dinv[i];
    }
    Ops::sync();
    for (int j = n - 1; j >= 0; --j) {     // backward: L' x = z
        T z0 = x0[j] * dinv[j];
        T z1 = NRHS > 1 ? x1[j] * dinv[j] : (T)0;
        for (int i = t; i < j; i += TEAM) {
            T l = Mp[cm(n, j, i)];
            x0[i] -= l * z0;
            if (NRHS > 1) x1[i] -= l * z1;
        }
        Ops::sync();
    }
    for (int i = t; i < n; i += TEAM) {
        x0[i] *= dinv[i];
        if (NRHS > 1) x1[i] *= dinv[i];
    }
    Ops::sync();
    }
}

// ---- warp-per-pixel path (R <= 64): the lower triangle of the Newton matrix is kept ROW-major, row i padded
// to a multiple of 4 floats (16 B aligned rows; the footprint of the packed layout), so the sums of the
// left-looking factorisation run over contiguous k: two LDS.128 feed four FMAs with no index arithmetic
// (the packed column-major layout cost 30 instructions per four terms).
// start of row i: rows 4b .. 4b+3 hold 4(b+1) floats each
__host__ __device__ __forceinline__ int ipls_rowoff(int i) { const int b = i >> 2, r = i & 3; return 8 * b * (b + 1) + 4 * r * (b + 1); }
__host__ __device__ inline int ipls_tri_floats(int n) { return n > 0 ? ipls_rowoff(n - 1) + 4 * (((n - 1) >> 2) + 1) : 0; }

__device__ __forceinline__ bool warp_cholesky_rm(float *M, float *dinv, int n, float floorv) {
    const int t = threadIdx.x & 31;
    bool clamped = false;
    for (int j = 0; j < n; ++j) {
        float sj = M[ipls_rowoff(j) + j];               // running pivot (see team_cholesky)
        if (!(sj > floorv)) { sj = floorv; clamped = true; }
        const float dj = 1.0f / sqrtf(sj);
        if (t == 0) dinv[j] = dj;
        const int nr = n - 1 - j;
        int g = 1;
        while (g < 32 && nr * (g * 2) <= 32) g <<= 1;   // g lanes share one row when few rows remain
        const int rows_per_pass = 32 / g;
        const int part = t & (g - 1), rl = t / g;
        const float *rowj = M + ipls_rowoff(j);
        const int jv = j >> 2;                           // whole float4 chunks below column j
        for (int r0 = 0; r0 < nr; r0 += rows_per_pass) {
            const int i = j + 1 + r0 + rl;
            const bool active = i < n;
            float *rowi = M + ipls_rowoff(active ? i : j);
            float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;
            for (int q = part; q < jv; q += g) {
                const float4 a = *reinterpret_cast<const float4 *>(rowi + 4 * q);
                const float4 b = *reinterpret_cast<const float4 *>(rowj + 4 * q);
                s0 = fmaf(a.x, b.x, s0); s1 = fmaf(a.y, b.y, s1); s2 = fmaf(a.z, b.z, s2); s3 = fmaf(a.w, b.w, s3);
            }
            if (part == 0)
                for (int k = 4 * jv; k < j; ++k) s0 = fmaf(rowi[k], rowj[k], s0);
            float s = (s0 + s1) + (s2 + s3);
            for (int o = g >> 1; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (active && part == 0) {
                s = (rowi[j] - s) * dj;
                rowi[j] = s;
                rowi[i] -= s * s;
            }
        }
        __syncwarp();
    }
    return clamped;
}

// (L L') x = rhs for the row-major factor: right-hand sides in registers (rows t, t + 32), x_j by shuffle
template <int NRHS>
__device__ __forceinline__ void warp_solve_rm(const float *M, const float *dinv, int n, float *x0, float *x1) {
    const int t = threadIdx.x & 31, r1 = t + 32;
    const bool h0 = t < n, h1 = r1 < n;
    float a0 = h0 ? x0[t] : 0.0f, b0 = h1 ? x0[r1] : 0.0f;
    float a1 = (NRHS > 1 && h0) ? x1[t] : 0.0f, b1 = (NRHS > 1 && h1) ? x1[r1] : 0.0f;
    const float d0 = h0 ? dinv[t] : 0.0f, d1 = h1 ? dinv[r1] : 0.0f;
    const float *row0 = M + ipls_rowoff(h0 ? t : 0), *row1 = M + ipls_rowoff(h1 ? r1 : 0);
    for (int j = 0; j < n; ++j) {      // forward: L z = rhs
        const float dj = dinv[j];
        const float z0 = __shfl_sync(0xffffffffu, (j < 32) ? a0 : b0, j & 31) * dj;
        const float z1 = NRHS > 1 ? __shfl_sync(0xffffffffu, (j < 32) ? a1 : b1, j & 31) * dj : 0.0f;
        if (h0 && t > j) { const float l = row0[j]; a0 -= l * z0; if (NRHS > 1) a1 -= l * z1; }
        if (h1 && r1 > j) { const float l = row1[j]; b0 -= l * z0; if (NRHS > 1) b1 -= l * z1; }
    }
    a0 *= d0; b0 *= d1; a1 *= d0; b1 *= d1;
    for (int j = n - 1; j >= 0; --j) { // backward: L' x = z
        const float dj = dinv[j];
        const float z0 = __shfl_sync(0xffffffffu, (j < 32) ? a0 : b0, j & 31) * dj;
        const float z1 = NRHS > 1 ? __shfl_sync(0xffffffffu, (j < 32) ? a1 : b1, j & 31) * dj : 0.0f;
        const float *rowj = M + ipls_rowoff(j);
        if (t < j) { const float l = rowj[t]; a0 -= l * z0; if (NRHS > 1) a1 -= l * z1; }
        if (r1 < j) { const float l = rowj[r1]; b0 -= l * z0; if (NRHS > 1) b1 -= l * z1; }
    }
    if (h0) { x0[t] = a0 * d0; if (NRHS > 1) x1[t] = a1 * d0; }
    if (h1) { x0[r1] = b0 * d1; if (NRHS > 1) x1[r1] = b1 * d1; }
    __syncwarp();
}

// floats of one team: TEAM == 32 keeps the row-major padded matrix, the CTA team the packed one
__host__ __device__ inline size_t ipls_generic_vec_floats(int L, int R) { return ((size_t)10 * R + L + 64 + 3) & ~(size_t)3; }
__host__ __device__ inline size_t ipls_warp_team_floats(int L, int R) {
    return ipls_generic_vec_floats(L, R) + (size_t)ipls_tri_floats(R);
}
__host__ __device__ inline size_t ipls_generic_team_floats(int L, int R) {
    return (size_t)10 * R + L + (size_t)R * (R + 1) / 2 + 64;
}

// grid-stride over pixels; TEAM == 32: one warp per pixel, blockDim.x/32 pixels per CTA pass;
// TEAM == blockDim.x: one pixel per CTA pass.
template <int TEAM>
__global__ void __launch_bounds__(256) ipls_generic_kernel(LibView lib, SolveParams prm) {
    using Ops = TeamOps<TEAM>;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0]) return;      // non-finite library: the caller is told (status or poisoned outputs)
    const float gdmax = lib.scal[0];
    const int L = lib.L, R = lib.R;
    const int teams_per_cta = blockDim.x / TEAM;
    const int team = threadIdx.x / TEAM;
    const int t = Ops::tid();
    float *base = smem + (size_t)team * (TEAM == 32 ? ipls_warp_team_floats(L, R) : ipls_generic_team_floats(L, R));
    float *a = base, *lam = a + R, *b = lam + R, *w = b + R, *u = w + R, *v = u + R, *da = v + R,
          *dl = da + R, *dinv = dl + R, *Ga = dinv + R, *yc = Ga + R, *red = yc + L,
          *Mp = (TEAM == 32) ? base + ipls_generic_vec_floats(L, R) : red + 64;
    const float fR = (float)R;
    const float tau = 0.995f;
    const bool cons = lib.cons != 0;      // false: positivity only -- no nu, no primal equality residual

    for (int64_t p = (int64_t)blockIdx.x * teams_per_cta + team; p < prm.N;
         p += (int64_t)gridDim.x * teams_per_cta) {
        // ---- load spectrum, centre it, detect non-finite input
        const float *y = prm.Y + p * prm.ldY;
        float badf = 0.0f;
        for (int l = t; l < L; l += TEAM) {
            float yv = y[l];
            if (!isfinite(yv)) badf = 1.0f;
            yc[l] = yv - lib.c[l];
        }
        Ops::sync();
        badf = Ops::max(badf, red);
        if (badf > 0.0f) {
            for (int i = t; i < R; i += TEAM) prm.coeffs[p * R + i] = 1.0f / fR;
            if (prm.info && t == 0) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            Ops::sync();
            continue;
        }
        // ---- projection b = Ac'(y - c)   ("X.S^T")
        float bmax = 0.0f;
        for (int i = t; i < R; i += TEAM) {
            float s = 0.0f;
            for (int l = 0; l < L; ++l) s = fmaf(lib.Ac[(size_t)l * R + i], yc[l], s);
            b[i] = s;
            bmax = fmaxf(bmax, fabsf(s));
        }
        bmax = Ops::max(bmax, red);
        const float sc = fmaxf(bmax, 1e-3f * gdmax);
        // ---- start (Mehrotra's heuristic, as in ipls_r32.cuh): the sum-constrained LS point of the regularised
        //      problem, x = Gi b - q (1'Gi b - 1)/(1'q), its reduced gradient as multipliers, both shifted inside
        float nu, lam0;
        {
            Ops::sync();
            float sx = 0.0f, sq = 0.0f;
            for (int i = t; i < R; i += TEAM) {
                float s = 0.0f;
                for (int j = 0; j < R; ++j) s = fmaf(lib.Gi[(size_t)j * R + i], b[j], s);
                u[i] = s; sx += s; sq += lib.Giq[i];
            }
            sx = Ops::sum(sx, red); sq = Ops::sum(sq, red);
            const float mu0 = cons ? (sx - 1.0f) / sq : 0.0f;
            for (int i = t; i < R; i += TEAM) u[i] = fmaf(-mu0, lib.Giq[i], u[i]);       // x
            Ops::sync();
            float gx = 0.0f, mnx = INFINITY, mng = INFINITY;
            for (int i = t; i < R; i += TEAM) {
                float s = 0.0f, rs = 0.0f;
                for (int j = 0; j < R; ++j) { const float gji = lib.Gc[(size_t)j * R + i]; s = fmaf(gji, u[j], s); rs += gji; }
                Ga[i] = s;                    // G x
                v[i] = rs;                    // row sum of G
                const float gi = s - b[i];
                lam[i] = gi;
                gx = fmaf(gi, u[i], gx); mnx = fminf(mnx, u[i]); mng = fminf(mng, gi);
            }
            gx = Ops::sum(gx, red); mnx = Ops::min(mnx, red); mng = Ops::min(mng, red);
            nu = cons ? -gx : 0.0f;
            const float dp = fmaxf(-mnx, 0.0f), dd = fmaxf(-(mng + nu), 0.0f);
            float xl = 0.0f, sl = 0.0f, sxx = 0.0f;
            for (int i = t; i < R; i += TEAM) {
                const float xi = u[i] + dp, li = lam[i] + nu + dd;
                u[i] = xi; lam[i] = li;
                xl = fmaf(xi, li, xl); sl += li; sxx += xi;
            }
            xl = Ops::sum(xl, red); sl = Ops::sum(sl, red); sxx = Ops::sum(sxx, red);
            const float dp2 = 0.05f * xl / fmaxf(sl, 1e-30f), dd2 = 0.05f * xl / fmaxf(sxx, 1e-30f);
            float sa = 0.0f, lm = 0.0f;
            for (int i = t; i < R; i += TEAM) {
                const float ai = u[i] + dp2 + 1e-3f, li = lam[i] + dd2 + 1e-4f * sc;
                a[i] = ai; lam[i] = li;
                sa += ai; lm = fmaxf(lm, li);
            }
            sa = Ops::sum(sa, red); lam0 = Ops::max(lm, red);
            const float rsa = cons ? 1.0f / sa : 1.0f;      // pos: the point is not normalised
            const bool ok = (lam0 > 0.0f) && isfinite(lam0) && isfinite(sa) && isfinite(rsa);
            if (!ok) { lam0 = fmaxf(bmax, 1e-3f * gdmax); nu = 0.0f; }
            for (int i = t; i < R; i += TEAM) {
                if (ok) {
                    a[i] *= rsa;
                    Ga[i] = fmaf(dp + dp2 + 1e-3f, v[i], Ga[i]) * rsa;      // G a of the shifted, normalised point
                } else {                                                     // degenerate data: the barycentre
                    a[i] = 1.0f / fR; lam[i] = lam0; Ga[i] = v[i] / fR;
                }
            }
        }
        int iters = 0, flags = 0;
        Ops::sync();

        for (int it = 0;; ++it) {
            // ---- residuals
            float rdmax = 0.0f, suma = 0.0f, gap = 0.0f;
            for (int i = t; i < R; i += TEAM) {
                float wi = Ga[i] - b[i] + nu;      // G a is carried along with a (Newton identity, see the update)
                w[i] = wi;
                rdmax = fmaxf(rdmax, fabsf(wi - lam[i]));
                suma += a[i];
                gap = fmaf(a[i], lam[i], gap);
            }
            rdmax = Ops::max(rdmax, red);
            suma = Ops::sum(suma, red);
            gap = Ops::sum(gap, red);
            const float rp = cons ? suma - 1.0f : 0.0f;
            if (gap <= prm.gap_tol * sc && rdmax <= prm.feas_tol * sc && fabsf(rp) <= prm.feas_tol) {
                flags |= LINMIN_INFO_CONVERGED;
                break;
            }
            if (it >= prm.max_iter) { flags |= LINMIN_INFO_MAX_ITER; break; }
            ++iters;
            const float mu = gap / fR;
            // ---- Newton matrix M = Gc + diag(lambda / a), packed lower, then Cholesky
            bool regularised;
            if constexpr (TEAM == 32) {
                for (int i = 0; i < R; ++i)                  // row i of the lower triangle, row-major
                    for (int k = t; k <= i; k += 32) {
                        float m = lib.Gc[(size_t)i * R + k];
                        if (k == i) m += lam[i] / a[i];
                        Mp[ipls_rowoff(i) + k] = m;
                    }
                Ops::sync();
                regularised = warp_cholesky_rm(Mp, dinv, R, 1e-12f * gdmax);
            } else {
                for (int j = 0; j < R; ++j)
                    for (int i = j + t; i < R; i += TEAM) {
                        float m = lib.Gc[(size_t)j * R + i];
                        if (i == j) m += lam[i] / a[i];
                        Mp[cm(R, i, j)] = m;
                    }
                Ops::sync();
                regularised = team_cholesky<TEAM, float>(Mp, dinv, R, 1e-12f * gdmax);
            }
            if (regularised) flags |= LINMIN_INFO_CHOL_REGULARISED;
            // ---- predictor
            for (int i = t; i < R; i += TEAM) { u[i] = -w[i]; v[i] = 1.0f; }
            Ops::sync();
            if constexpr (TEAM == 32) warp_solve_rm<2>(Mp, dinv, R, u, v);
            else team_solve<TEAM, 2, float>(Mp, dinv, R, u, v);
            float su = 0.0f, sv = 0.0f;
            for (int i = t; i < R; i += TEAM) { su += u[i]; sv += v[i]; }
            su = Ops::sum(su, red);
            sv = Ops::sum(sv, red);
            float dnu = cons ? (su + rp) / sv : 0.0f;
            float ap = INFINITY, ad = INFINITY;
            for (int i = t; i < R; i += TEAM) {
                float dai = u[i] - v[i] * dnu;
                float dli = -lam[i] - (lam[i] / a[i]) * dai;
                da[i] = dai; dl[i] = dli;
                if (dai < 0.0f) ap = fminf(ap, -a[i] / dai);
                if (dli < 0.0f) ad = fminf(ad, -lam[i] / dli);
            }
            ap = fminf(1.0f, Ops::min(ap, red));
            ad = fminf(1.0f, Ops::min(ad, red));
            float mua = 0.0f;
            for (int i = t; i < R; i += TEAM) mua = fmaf(a[i] + ap * da[i], lam[i] + ad * dl[i], mua);
            mua = Ops::sum(mua, red) / fR;
            float sg = mua / mu;
            sg = fminf(1.0f, fmaxf(0.0f, sg * sg * sg));
            // ---- corrector
            for (int i = t; i < R; i += TEAM) {
                float cc = sg * mu - da[i] * dl[i];
                dl[i] = cc;
                u[i] = -w[i] + cc / a[i];
            }
            Ops::sync();
            if constexpr (TEAM == 32) warp_solve_rm<1>(Mp, dinv, R, u, nullptr);
            else team_solve<TEAM, 1, float>(Mp, dinv, R, u, nullptr);
            su = 0.0f;
            for (int i = t; i < R; i += TEAM) su += u[i];
            su = Ops::sum(su, red);
            dnu = cons ? (su + rp) / sv : 0.0f;
            ap = INFINITY; ad = INFINITY;
            for (int i = t; i < R; i += TEAM) {
                float dai = u[i] - v[i] * dnu;
                float dli = -lam[i] + dl[i] / a[i] - (lam[i] / a[i]) * dai;
                da[i] = dai; dl[i] = dli;
                if (dai < 0.0f) ap = fminf(ap, -a[i] / dai);
                if (dli < 0.0f) ad = fminf(ad, -lam[i] / dli);
            }
            ap = fminf(1.0f, tau * Ops::min(ap, red));
            ad = fminf(1.0f, tau * Ops::min(ad, red));
            // G da = (r1 - dnu 1) - (lambda/a) o da row by row (M da = r1 - dnu 1, M = G + diag(lambda/a)), with
            // r1 = -w + cc/a and cc = dl + lambda + (lambda/a) da recovered from the corrector's dl
            for (int i = t; i < R; i += TEAM) {
                const float di = lam[i] / a[i];
                const float cc_over_a = dl[i] + lam[i] + di * da[i];
                Ga[i] = fmaf(ap, (-w[i] + cc_over_a) - dnu - di * da[i], Ga[i]);
                a[i] = fmaxf(fmaf(ap, da[i], a[i]), 1e-18f);
                lam[i] = fmaxf(fmaf(ad, dl[i], lam[i]), 1e-18f * lam0);
            }
            nu = fmaf(ad, dnu, nu);
            Ops::sync();
        }
        // hand-over: zero where the primal-dual indicator says inactive (LINMIN_TAPIA_KAPPA, common.cuh)
        for (int i = t; i < R; i += TEAM) prm.coeffs[p * R + i] = (a[i] * sc > LINMIN_TAPIA_KAPPA * lam[i]) ? a[i] : 0.0f;
        if (prm.info && t == 0) prm.info[p] = flags | (iters << 8);
        Ops::sync();
    }
}

}  // namespace linmin
