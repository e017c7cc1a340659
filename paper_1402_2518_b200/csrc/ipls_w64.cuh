// ipls_w64.cuh -- projection + IPLS for 33 <= R <= 64 endmembers (sm_100a): one warp per pixel, Newton matrix in registers.
//
// SURVEY.md 8(a) a1 + a2 for the CRISM-like configuration (BASELINE.json configs[2]: L = 240, R = 64), for the paper's
// own library sizes (36 / 44 spectra, 37 with the slack of slo: PAPER.md:175, 250, 333-339) and for R = 32 + slack.
// Same iteration as ipls_generic.cuh / ipls_q32.cuh (Mehrotra predictor-corrector on the centred normal equations;
// reading R1).  The any-size kernel keeps the matrix in shared memory and pays two shared-memory operands per FMA of
// its left-looking factorisation (15 k cycles.SM per pixel-iteration at R = 64, 3 % of the FP32 peak).  Here:
//   * lane t owns rows t and t + 32 of M = G + diag(lambda/a) in REGISTERS (row t up to column 31, row t + 32 up to
//     column 63: 48 packed pairs = 96 registers); rows beyond R are identity rows that never couple.
//   * right-looking LDL': per step the raw column goes through one 64-float line in shared memory (2 STS.32 per
//     lane, LDS.128 read-back chunk by chunk), the rank-one update is FFMA2 with the row's multiplier as the scalar
//     operand; look-ahead of one column.  The predictor's forward substitution (two right-hand sides) rides along.
//   * the corrector's forward substitution is a 63-step column sweep by shuffle; for the two backward substitutions
//     every lane dumps its rows of -L once per iteration into a packed row-major triangle in shared memory and the
//     sweep reads row j coalesced (x_j by shuffle).
//   * every per-row vector is two registers per lane, so the kernel fits 12 warps per SM (3 per scheduler).
// Algorithmic work per pixel: 2 L R + it (R^3/3 + 8 R^2 + 30 R) flops.
#pragma once
#include "common.cuh"

namespace linmin {
namespace w64 {

constexpr int RP = 64;          // padded endmember count
constexpr int WARPS = 12;
constexpr int GST = 68;         // row stride of G / Gi in shared memory: 68 = 4 mod 32, conflict-free LDS.128 by row
constexpr int TRI = 2176;       // packed row-major triangle: rows 4b .. 4b+3 hold 4 (b + 1) floats
constexpr unsigned FULL = 0xffffffffu;

__host__ __device__ __forceinline__ int rowoff(int i) { const int b = i >> 2, r = i & 3; return 8 * b * (b + 1) + 4 * r * (b + 1); }
__host__ __device__ inline int lpad(int L) { return (L + 3) & ~3; }
__host__ __device__ inline size_t cta_floats(int L) { return (size_t)lpad(L) * RP + lpad(L) + 2 * RP * GST + 2 * RP; }
__host__ __device__ inline size_t warp_floats(int L) { return (size_t)lpad(L) + 2 * RP + 2 * RP + TRI; }
__host__ __device__ inline size_t smem_bytes(int L, int warps) { return (cta_floats(L) + (size_t)warps * warp_floats(L)) * sizeof(float); }

#define WA(j) (((j) & 1) ? ma[(j) >> 1].y : ma[(j) >> 1].x)
#define WB(j) (((j) & 1) ? mb[(j) >> 1].y : mb[(j) >> 1].x)

// L' x = y in place (rows t, t + 32); tri holds -L by rows; x_j travels by shuffle
__device__ __forceinline__ void backward_sweep(const float *tri, float &xa, float &xb, int t) {
#pragma unroll 4
    for (int j = RP - 1; j >= 32; --j) {
        const float z = __shfl_sync(FULL, xb, j & 31);
        const float *row = tri + rowoff(j);
        xa = fmaf(row[t], z, xa);
        if (t + 32 < j) xb = fmaf(row[t + 32], z, xb);
    }
#pragma unroll 4
    for (int j = 31; j >= 1; --j) {
        const float z = __shfl_sync(FULL, xa, j);
        if (t < j) xa = fmaf(tri[rowoff(j) + t], z, xa);
    }
}

}  // namespace w64

__global__ void __launch_bounds__(w64::WARPS * 32, 1)
ipls_w64_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter, int warps) {
    using namespace w64;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0]) return;
    const int L = lib.L, R = lib.R, Lp = lpad(L);
    float *Acs = smem;                            // [Lp][64] centred library, zero beyond L and R
    float *cv = Acs + (size_t)Lp * RP;            // [Lp]
    float *Gp = cv + Lp;                          // [64][GST]; rows beyond R: identity
    float *Gip = Gp + RP * GST;                   // [64][GST]; rows beyond R: zero
    float *Giq = Gip + RP * GST;                  // [64]
    float *Grs = Giq + RP;                        // [64] row sums of G
    const int warp = threadIdx.x >> 5, t = threadIdx.x & 31;
    float *wb = Grs + RP + (size_t)warp * warp_floats(L);
    float *ys = wb;                               // [Lp] centred spectrum
    float *xl0 = ys + Lp, *xl1 = xl0 + RP;        // exchange lines
    float *vec = xl1 + RP;                        // [2][64] scratch vectors
    float *tri = vec + 2 * RP;                    // packed -L

    for (int e = threadIdx.x; e < Lp * RP; e += blockDim.x) {
        const int l = e >> 6, r = e & 63;
        Acs[e] = (l < L && r < R) ? lib.Ac[(size_t)l * R + r] : 0.0f;
    }
    for (int l = threadIdx.x; l < Lp; l += blockDim.x) cv[l] = (l < L) ? lib.c[l] : 0.0f;
    for (int e = threadIdx.x; e < RP * RP; e += blockDim.x) {
        const int i = e >> 6, j = e & 63;
        const bool in = i < R && j < R;
        Gp[i * GST + j] = in ? lib.Gc[(size_t)i * R + j] : ((i == j) ? 1.0f : 0.0f);
        Gip[i * GST + j] = in ? lib.Gi[(size_t)i * R + j] : 0.0f;
    }
    if (threadIdx.x < RP) Giq[threadIdx.x] = (threadIdx.x < R) ? lib.Giq[threadIdx.x] : 0.0f;
    __syncthreads();
    if (threadIdx.x < RP) {
        float s = 0.0f;
        if (threadIdx.x < R) for (int j = 0; j < R; ++j) s += Gp[threadIdx.x * GST + j];
        Grs[threadIdx.x] = s;
    }
    __syncthreads();
    if (warp >= warps) return;

    const float gdmax = lib.scal[0];
    const bool cons = lib.cons != 0;      // false: positivity only -- no nu, the start point is not normalised
    const float rGiqTot = cons ? 1.0f / lib.scal[1] : 0.0f;
    const float tau = 0.995f, fR = (float)R;
    const float pivot_floor = 1e-12f * gdmax;
    const bool va = t < R, vb = t + 32 < R;       // my rows exist

    while (true) {
        unsigned int tk = 0;
        if (t == 0) tk = atomicAdd(counter, 1u);
        const int64_t p = (int64_t)__shfl_sync(FULL, tk, 0);
        if (p >= prm.N) break;
        // ---- spectrum, centred; non-finite input
        const float *y = prm.Y + p * prm.ldY;
        bool bad = false;
        for (int l = t; l < Lp; l += 32) {
            const float yv = (l < L) ? y[l] : 0.0f;
            bad |= !isfinite(yv);
            ys[l] = yv - cv[l];
        }
        bad = __any_sync(FULL, bad);
        __syncwarp();
        if (bad) {
            if (va) prm.coeffs[p * R + t] = 1.0f / fR;
            if (vb) prm.coeffs[p * R + t + 32] = 1.0f / fR;
            if (prm.info && t == 0) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            __syncwarp();
            continue;
        }
        // ---- projection b = Ac'(y - c): lane t takes endmembers t and t + 32
        float ba, bb;
        {
            float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f, u0 = 0.0f, u1 = 0.0f, u2 = 0.0f, u3 = 0.0f;
            for (int l = 0; l < Lp; l += 4) {
                const float4 y4 = *reinterpret_cast<const float4 *>(ys + l);
                const float *a = Acs + (size_t)l * RP + t;
                s0 = fmaf(a[0], y4.x, s0); u0 = fmaf(a[32], y4.x, u0);
                s1 = fmaf(a[RP], y4.y, s1); u1 = fmaf(a[RP + 32], y4.y, u1);
                s2 = fmaf(a[2 * RP], y4.z, s2); u2 = fmaf(a[2 * RP + 32], y4.z, u2);
                s3 = fmaf(a[3 * RP], y4.w, s3); u3 = fmaf(a[3 * RP + 32], y4.w, u3);
            }
            ba = (s0 + s1) + (s2 + s3); bb = (u0 + u1) + (u2 + u3);
        }
        const float bmax = warp_max(fmaxf(fabsf(ba), fabsf(bb)));
        const float sc = fmaxf(bmax, 1e-3f * gdmax);
        // mat-vec with a 64 x 64 matrix in shared memory: out rows t, t + 32 of M v (v on line `src`)
        auto matvec = [&](const float *M, const float *src, float &oa, float &ob) {
            float s0 = 0.0f, s1 = 0.0f, u0 = 0.0f, u1 = 0.0f;
#pragma unroll 4
            for (int c = 0; c < RP / 4; ++c) {
                const float4 v = *reinterpret_cast<const float4 *>(src + 4 * c);
                const float4 ra = *reinterpret_cast<const float4 *>(M + t * GST + 4 * c);
                const float4 rb = *reinterpret_cast<const float4 *>(M + (t + 32) * GST + 4 * c);
                s0 = fmaf(ra.x, v.x, s0); s1 = fmaf(ra.y, v.y, s1); s0 = fmaf(ra.z, v.z, s0); s1 = fmaf(ra.w, v.w, s1);
                u0 = fmaf(rb.x, v.x, u0); u1 = fmaf(rb.y, v.y, u1); u0 = fmaf(rb.z, v.z, u0); u1 = fmaf(rb.w, v.w, u1);
            }
            oa = s0 + s1; ob = u0 + u1;
        };
        // ---- start (Mehrotra's heuristic, as in ipls_generic.cuh)
        float aa, ab, la, lb, ga, gb, nu, lam0;        // a, lambda, G a - b by row; nu; floor scale of lambda
        {
            vec[t] = ba; vec[t + 32] = bb;
            __syncwarp();
            float xa, xb;
            matvec(Gip, vec, xa, xb);
            const float sx = warp_sum(xa + xb);
            const float mu0 = (sx - 1.0f) * rGiqTot;
            xa = fmaf(-mu0, Giq[t], xa); xb = fmaf(-mu0, Giq[t + 32], xb);
            vec[RP + t] = xa; vec[RP + t + 32] = xb;
            __syncwarp();
            float Gxa, Gxb;
            matvec(Gp, vec + RP, Gxa, Gxb);
            if (!vb) Gxb = 0.0f;                                   // identity row of the padding
            if (!va) Gxa = 0.0f;
            float gra = Gxa - ba, grb = Gxb - bb;                  // gradient at x
            const float gx = warp_sum(gra * xa + grb * xb);
            const float mnx = warp_min(fminf(va ? xa : INFINITY, vb ? xb : INFINITY));
            const float mng = warp_min(fminf(va ? gra : INFINITY, vb ? grb : INFINITY));
            nu = cons ? -gx : 0.0f;
            const float dp = fmaxf(-mnx, 0.0f), dd = fmaxf(-(mng + nu), 0.0f);
            xa += dp; xb += dp; gra += nu + dd; grb += nu + dd;
            const float xlm = warp_sum((va ? xa * gra : 0.0f) + (vb ? xb * grb : 0.0f));
            const float sl = warp_sum((va ? gra : 0.0f) + (vb ? grb : 0.0f));
            const float sxx = warp_sum((va ? xa : 0.0f) + (vb ? xb : 0.0f));
            const float dp2 = 0.05f * xlm / fmaxf(sl, 1e-30f), dd2 = 0.05f * xlm / fmaxf(sxx, 1e-30f);
            aa = xa + dp2 + 1e-3f; ab = xb + dp2 + 1e-3f;
            la = gra + dd2 + 1e-4f * sc; lb = grb + dd2 + 1e-4f * sc;
            const float sa = warp_sum((va ? aa : 0.0f) + (vb ? ab : 0.0f));
            lam0 = warp_max(fmaxf(va ? la : 0.0f, vb ? lb : 0.0f));
            const float rsa = cons ? 1.0f / sa : 1.0f;
            const bool ok = (lam0 > 0.0f) && isfinite(lam0) && isfinite(sa) && isfinite(rsa);
            if (ok) {
                aa *= rsa; ab *= rsa;
                ga = fmaf(dp + dp2 + 1e-3f, Grs[t], Gxa) * rsa - ba;      // G a of the shifted, normalised point, minus b
                gb = fmaf(dp + dp2 + 1e-3f, Grs[t + 32], Gxb) * rsa - bb;
            } else {                                                       // degenerate data: the barycentre
                lam0 = fmaxf(bmax, 1e-3f * gdmax); nu = 0.0f;
                aa = ab = 1.0f / fR; la = lb = lam0;
                ga = Grs[t] / fR - ba; gb = Grs[t + 32] / fR - bb;
            }
            if (!va) { aa = 1.0f; la = 0.0f; ga = 0.0f; }
            if (!vb) { ab = 1.0f; lb = 0.0f; gb = 0.0f; }
        }
        int iters = 0, flags = 0;

        for (int it = 0;; ++it) {
            // ---- residuals and stopping rule
            const float wa = va ? ga + nu : 0.0f, wbv = vb ? gb + nu : 0.0f;
            const float rdm = warp_max(fmaxf(va ? fabsf(wa - la) : 0.0f, vb ? fabsf(wbv - lb) : 0.0f));
            const float sa = warp_sum((va ? aa : 0.0f) + (vb ? ab : 0.0f));
            const float gp = warp_sum((va ? aa * la : 0.0f) + (vb ? ab * lb : 0.0f));
            const float rp = cons ? sa - 1.0f : 0.0f;
            if (gp <= prm.gap_tol * sc && rdm <= prm.feas_tol * sc && fabsf(rp) <= prm.feas_tol) { flags |= LINMIN_INFO_CONVERGED; break; }
            if (it >= prm.max_iter) { flags |= LINMIN_INFO_MAX_ITER; break; }
            ++iters;
            const float mu = gp / fR;
            // ---- rows of M from G, diagonal added
            float2 ma[16], mb[32];
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float4 g4 = *reinterpret_cast<const float4 *>(Gp + t * GST + 4 * c);
                ma[2 * c] = make_float2(g4.x, g4.y); ma[2 * c + 1] = make_float2(g4.z, g4.w);
            }
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const float4 g4 = *reinterpret_cast<const float4 *>(Gp + (t + 32) * GST + 4 * c);
                mb[2 * c] = make_float2(g4.x, g4.y); mb[2 * c + 1] = make_float2(g4.z, g4.w);
            }
            const float ainva = rcp_approx(aa), ainvb = rcp_approx(ab);
            const float da_ = la * ainva, db_ = lb * ainvb;            // d = lambda / a
            // diagonal entries: column t of row t, column t + 32 of row t + 32 (lane-dependent slot: one-hot adds)
#pragma unroll
            for (int jp = 0; jp < 16; ++jp) {
                const float2 e = make_float2((t == 2 * jp) ? 1.0f : 0.0f, (t == 2 * jp + 1) ? 1.0f : 0.0f);
                ma[jp] = fma2(da_, e, ma[jp]);
                mb[16 + jp] = fma2(db_, e, mb[16 + jp]);
            }
            float2 rra = va ? make_float2(1.0f, -wa) : make_float2(0.0f, 0.0f);
            float2 rrb = vb ? make_float2(1.0f, -wbv) : make_float2(0.0f, 0.0f);
            float dinva = 0.0f, dinvb = 0.0f;
            bool clamped = false;
            // ---- M = L D L' (right-looking), look-ahead of one column
            xl0[t] = WA(0); xl0[t + 32] = WB(0);
            __syncwarp();
            float2 zk = make_float2(__shfl_sync(FULL, rra.x, 0), __shfl_sync(FULL, rra.y, 0));
#pragma unroll
            for (int k = 0; k < RP - 1; ++k) {
                const float *cl = (k & 1) ? xl1 : xl0;           // raw column k
                float *nw = (k & 1) ? xl0 : xl1;                 // where column k + 1 goes
                const int k1 = k + 1;
                float piv = cl[k];
                if (!(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
                const float rinv = rcp_approx(piv), nrinv = -rinv;
                float nla = 0.0f, nlb;
                if (k < 32) {
                    nla = (t > k) ? WA(k) * nrinv : 0.0f;
                    if (k & 1) ma[k >> 1].y = nla; else ma[k >> 1].x = nla;
                    rra = fma2(nla, zk, rra);
                    nlb = WB(k) * nrinv;
                    dinva = (t == k) ? rinv : dinva;
                } else {
                    nlb = (t + 32 > k) ? WB(k) * nrinv : 0.0f;
                    dinvb = (t + 32 == k) ? rinv : dinvb;
                }
                if (k & 1) mb[k >> 1].y = nlb; else mb[k >> 1].x = nlb;
                rrb = fma2(nlb, zk, rrb);
                // look-ahead: column k + 1, then its exchange
                {
                    const float ck1 = cl[k1];
                    if (k1 < 32) { if (k1 & 1) ma[k1 >> 1].y = fmaf(nla, ck1, ma[k1 >> 1].y); else ma[k1 >> 1].x = fmaf(nla, ck1, ma[k1 >> 1].x); }
                    if (k1 & 1) mb[k1 >> 1].y = fmaf(nlb, ck1, mb[k1 >> 1].y); else mb[k1 >> 1].x = fmaf(nlb, ck1, mb[k1 >> 1].x);
                }
                if (k1 < RP - 1) {
                    if (k1 < 32) nw[t] = WA(k1);
                    nw[t + 32] = WB(k1);
                }
                // rest of the rank-one update (columns k + 2 ..), chunk by chunk
#pragma unroll
                for (int c = (k + 2) >> 2; c < RP / 4; ++c) {
                    const float4 v = *reinterpret_cast<const float4 *>(cl + 4 * c);
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const int jp = 2 * c + h, j0 = 2 * jp;
                        const float2 cp = h ? make_float2(v.z, v.w) : make_float2(v.x, v.y);
                        if (j0 >= k + 2) {
                            if (jp < 16 && k < 31) ma[jp] = fma2(nla, cp, ma[jp]);
                            mb[jp] = fma2(nlb, cp, mb[jp]);
                        } else if (j0 + 1 == k + 2) {
                            if (jp < 16 && k < 31) ma[jp].y = fmaf(nla, cp.y, ma[jp].y);
                            mb[jp].y = fmaf(nlb, cp.y, mb[jp].y);
                        }
                    }
                }
                if (k1 < RP - 1) {
                    __syncwarp();
                    zk = (k1 < 32) ? make_float2(__shfl_sync(FULL, rra.x, k1), __shfl_sync(FULL, rra.y, k1))
                                   : make_float2(__shfl_sync(FULL, rrb.x, k1 - 32), __shfl_sync(FULL, rrb.y, k1 - 32));
                }
            }
            {   // last pivot (row 63: lane 31)
                float piv = mb[31].y;
                if (t == 31 && !(piv > pivot_floor)) { piv = pivot_floor; clamped = true; }
                dinvb = (t == 31) ? rcp_approx(piv) : dinvb;
            }
            if (__any_sync(FULL, clamped)) flags |= LINMIN_INFO_CHOL_REGULARISED;
            // ---- -L by rows into shared memory for the backward substitutions
            __syncwarp();
            {
                float *ra = tri + rowoff(t), *rb = tri + rowoff(t + 32);
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    if (c <= (t >> 2)) *reinterpret_cast<float4 *>(ra + 4 * c) = make_float4(ma[2 * c].x, ma[2 * c].y, ma[2 * c + 1].x, ma[2 * c + 1].y);
#pragma unroll
                for (int c = 0; c < 16; ++c)
                    if (c <= 8 + (t >> 2)) *reinterpret_cast<float4 *>(rb + 4 * c) = make_float4(mb[2 * c].x, mb[2 * c].y, mb[2 * c + 1].x, mb[2 * c + 1].y);
            }
            __syncwarp();
            // ---- predictor
            float sww = warp_sum(rra.x * dinva * rra.x + rrb.x * dinvb * rrb.x);
            float swz = warp_sum(rra.x * dinva * rra.y + rrb.x * dinvb * rrb.y);
            const float rsww = cons ? 1.0f / sww : 0.0f;       // pos: dnu == 0 (nu stays 0)
            float dnu = (swz + rp) * rsww;
            float xa = fmaf(-rra.x, dnu, rra.y) * dinva, xb = fmaf(-rrb.x, dnu, rrb.y) * dinvb;
            backward_sweep(tri, xa, xb, t);
            float mp = warp_max(fmaxf(-xa * ainva, -xb * ainvb));
            float md = warp_max(fmaxf(va ? 1.0f + ainva * xa : 0.0f, vb ? 1.0f + ainvb * xb : 0.0f));
            float ap = (mp > 1.0f) ? 1.0f / mp : 1.0f, ad = (md > 1.0f) ? 1.0f / md : 1.0f;
            const float dla = -la - da_ * xa, dlb = -lb - db_ * xb;
            float mua = warp_sum((va ? fmaf(ap, xa, aa) * fmaf(ad, dla, la) : 0.0f) + (vb ? fmaf(ap, xb, ab) * fmaf(ad, dlb, lb) : 0.0f)) / fR;
            float sg = mua / mu;
            sg = fminf(1.0f, fmaxf(0.0f, sg * sg * sg));
            // ---- corrector
            const float cca = fmaf(sg, mu, -xa * dla), ccb = fmaf(sg, mu, -xb * dlb);
            float ra_ = va ? fmaf(cca, ainva, -wa) : 0.0f, rb_ = vb ? fmaf(ccb, ainvb, -wbv) : 0.0f;
            const float r1a = ra_, r1b = rb_;
#pragma unroll
            for (int k = 0; k < RP - 1; ++k) {         // forward substitution: column sweep
                const float z = (k < 32) ? __shfl_sync(FULL, ra_, k) : __shfl_sync(FULL, rb_, k - 32);
                if (k < 32) ra_ = fmaf(WA(k), z, ra_);
                rb_ = fmaf(WB(k), z, rb_);
            }
            swz = warp_sum(rra.x * dinva * ra_ + rrb.x * dinvb * rb_);
            dnu = (swz + rp) * rsww;
            xa = fmaf(-rra.x, dnu, ra_) * dinva; xb = fmaf(-rrb.x, dnu, rb_) * dinvb;
            backward_sweep(tri, xa, xb, t);
            const float dl2a = fmaf(cca, ainva, -la) - da_ * xa, dl2b = fmaf(ccb, ainvb, -lb) - db_ * xb;
            mp = warp_max(fmaxf(-xa * ainva, -xb * ainvb));
            md = warp_max(fmaxf(va ? -dl2a / la : 0.0f, vb ? -dl2b / lb : 0.0f));
            ap = (tau < mp) ? tau / mp : 1.0f;
            ad = (tau < md) ? tau / md : 1.0f;
            if (va) {
                ga = fmaf(ap, r1a - dnu - da_ * xa, ga);
                aa = fmaxf(fmaf(ap, xa, aa), 1e-18f);
                la = fmaxf(fmaf(ad, dl2a, la), 1e-18f * lam0);
            }
            if (vb) {
                gb = fmaf(ap, r1b - dnu - db_ * xb, gb);
                ab = fmaxf(fmaf(ap, xb, ab), 1e-18f);
                lb = fmaxf(fmaf(ad, dl2b, lb), 1e-18f * lam0);
            }
            nu = fmaf(ad, dnu, nu);
        }
        // hand-over: zero where the primal-dual indicator says inactive (LINMIN_TAPIA_KAPPA, common.cuh)
        if (va) prm.coeffs[p * R + t] = (aa * sc > LINMIN_TAPIA_KAPPA * la) ? aa : 0.0f;
        if (vb) prm.coeffs[p * R + t + 32] = (ab * sc > LINMIN_TAPIA_KAPPA * lb) ? ab : 0.0f;
        if (prm.info && t == 0) prm.info[p] = flags | (iters << 8);
        __syncwarp();
    }
}
#undef WA
#undef WB

inline int ipls_w64_warps(int L) {
    int w = w64::WARPS;
    while (w > 1 && w64::smem_bytes(L, w) > 226 * 1024) --w;
    return w64::smem_bytes(L, w) <= 226 * 1024 ? w : 0;
}

// counter: device word, zero
inline cudaError_t launch_ipls_w64(const LibView &lv, const SolveParams &prm, int sm_count, unsigned int *counter,
                                   cudaStream_t stream) {
    const int warps = ipls_w64_warps(lv.L);
    if (warps < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = w64::smem_bytes(lv.L, warps);
    cudaError_t e = cudaFuncSetAttribute(ipls_w64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((prm.N + warps - 1) / warps, sm_count));
    ipls_w64_kernel<<<grid, w64::WARPS * 32, smem, stream>>>(lv, prm, counter, warps);
    return cudaGetLastError();
}

}  // namespace linmin
