// start_r32.cuh -- K0 of the R = 32 path: projection b = Ac'(y - c) and the start point of IPLS, for every pixel.
//
// SURVEY.md 8(a) a1 ("X S^T": the one dense contraction of the path, [N x L] . [L x R]) and the first half
// of a2.  The projection is a GEMM with a tiny right-hand matrix, so it is register-blocked over PIXELS: a lane owns
// 4 pixels x all 32 endmembers (128 accumulators, as 64 packed pairs over pixel pairs), a warp a tile of 128
// pixels.  One library row (32 floats, the same for every lane: a shared-memory broadcast) then feeds 128 FMAs per
// lane, i.e. 16 FMAs per float delivered from shared memory -- the FMA pipe, not the shared-memory pipe, is the
// limit (the round-1 kernel projected with 4 endmembers x 1 pixel per lane: 1 FMA per float, 89 % shared-memory
// pipe).  The spectra arrive through cp.async (16 B, coalesced: 64 contiguous bytes per row and chunk) in chunks
// of 16 channels, double-buffered per warp, into rows padded to 20 floats (conflict-free LDS.128 by pixel).
//
// Start point (Mehrotra's heuristic for this QP): x = the sum-constrained LS point of the regularised
// problem, x = Gi b - q (1'Gi b - 1)/(1'q), its reduced gradient as multipliers, both shifted into the interior.
// The two 32 x 32 mat-vecs run as packed FMAs over a PAIR of pixels with the matrix row broadcast.
//
// Output: one 416-byte record per pixel for the iteration kernel (ipls_q32.cuh): a, lambda, G a - b (each in the
// lane-major order of that kernel: position 8 t + s holds row t + 4 s), nu, the scale sc, lambda0 and the flags.
#pragma once
#include "common.cuh"

namespace linmin {
namespace s32 {

constexpr int R = 32;
constexpr int WARPS = 8;
constexpr int TP = 128;        // pixels per warp tile
constexpr int CH = 16;         // channels per staged chunk
constexpr int YST = 20;        // padded row stride (floats) of a staged chunk: conflict-free LDS.128 by pixel
constexpr int REC = 104;       // floats per record: a[32] lambda[32] (Ga - b)[32] nu sc lambda0 flags mu rp - -
constexpr unsigned FULL = 0xffffffffu;

__host__ __device__ inline int lpad(int L) { return (L + CH - 1) / CH * CH; }
__host__ __device__ inline size_t lib_floats(int L) { return (size_t)lpad(L) * R + lpad(L) + 2 * R * R + 2 * R; }
__host__ __device__ inline size_t warp_floats() { return (size_t)2 * TP * YST; }

}  // namespace s32

// rec: N x REC floats (workspace).  One warp per tile of 128 pixels, static partition (the work per pixel is fixed).
// CONS false: positivity only -- no nu, the start point is not normalised
template <bool CONS>
__global__ void __launch_bounds__(s32::WARPS * 32, 1)
start_r32_kernel(LibView lib, SolveParams prm, int64_t p_begin, int64_t p_end, float *__restrict__ rec, int warps) {
    using namespace s32;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0]) return;
    const int L = lib.L, Lp = lpad(L);
    float *Acp = smem;                          // [Lp][32] centred library, zero rows beyond L
    float *cv = Acp + (size_t)Lp * R;           // [Lp]
    float *Gis = cv + Lp;                       // [32][32]
    float *Gs = Gis + R * R;                    // [32][32]
    float *Giq = Gs + R * R;                    // [32]
    float *Grs = Giq + R;                       // [32] row sums of G
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float *ybuf = Grs + R + (size_t)warp * warp_floats();      // 2 x [TP][YST]

    for (int e = threadIdx.x; e < Lp * R; e += blockDim.x) Acp[e] = (e < L * R) ? lib.Ac[e] : 0.0f;
    for (int l = threadIdx.x; l < Lp; l += blockDim.x) cv[l] = (l < L) ? lib.c[l] : 0.0f;
    for (int e = threadIdx.x; e < R * R; e += blockDim.x) { Gis[e] = lib.Gi[e]; Gs[e] = lib.Gc[e]; }
    if (threadIdx.x < R) Giq[threadIdx.x] = lib.Giq[threadIdx.x];
    __syncthreads();
    if (threadIdx.x < R) {
        float s = 0.0f;
        for (int j = 0; j < R; ++j) s += Gs[threadIdx.x * R + j];
        Grs[threadIdx.x] = s;
    }
    __syncthreads();
    if (warp >= warps) return;
    const float gdmax = lib.scal[0];
    constexpr bool cons = CONS;
    const float rGiqTot = cons ? rcp_approx(lib.scal[1]) : 0.0f;
    const bool vec_ok = ((L & 3) == 0) && ((prm.ldY & 3) == 0) && ((reinterpret_cast<uintptr_t>(prm.Y) & 15) == 0);
    const int nchunks = Lp / CH;

    for (int64_t tile = (int64_t)blockIdx.x * warps + warp;; tile += (int64_t)gridDim.x * warps) {
        const int64_t p0 = p_begin + tile * TP;
        if (p0 >= p_end) break;
        // ---- stage one chunk of 16 channels for the 128 pixels of the tile: 512 pieces of 16 B, 16 per lane
        auto stage = [&](int cc, float *dst) {
            if (vec_ok) {
#pragma unroll 4
                for (int i = 0; i < 16; ++i) {
                    const int idx = lane + 32 * i, row = idx >> 2, piece = idx & 3;
                    int64_t p = p0 + row;
                    if (p >= p_end) p = p_end - 1;
                    const int l = cc * CH + 4 * piece;
                    const float *src = prm.Y + p * prm.ldY + (l < L ? l : 0);
                    const unsigned nbytes = (l < L) ? 16u : 0u;        // pieces beyond L are zero-filled
                    const unsigned sa = (unsigned)__cvta_generic_to_shared(dst + row * YST + 4 * piece);
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(src), "r"(nbytes) : "memory");
                }
            } else {
                for (int i = 0; i < 64; ++i) {
                    const int idx = lane + 32 * i, row = idx >> 4, ch = idx & 15;
                    int64_t p = p0 + row;
                    if (p >= p_end) p = p_end - 1;
                    const int l = cc * CH + ch;
                    dst[row * YST + ch] = (l < L) ? prm.Y[p * prm.ldY + l] : 0.0f;
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        float2 acc[R][2];        // [endmember][pixel pair]: (pixel lane, lane + 32) and (lane + 64, lane + 96)
#pragma unroll
        for (int r = 0; r < R; ++r) { acc[r][0] = make_float2(0.0f, 0.0f); acc[r][1] = make_float2(0.0f, 0.0f); }
        bool bad[4] = {false, false, false, false};
        stage(0, ybuf);
        for (int cc = 0; cc < nchunks; ++cc) {
            float *cur = ybuf + (cc & 1) * (TP * YST);
            if (cc + 1 < nchunks) {
                stage(cc + 1, ybuf + ((cc + 1) & 1) * (TP * YST));
                asm volatile("cp.async.wait_group 1;" ::: "memory");
            } else {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
            }
            __syncwarp();
#pragma unroll 1
            for (int l4 = 0; l4 < CH / 4; ++l4) {
                float yv[4][4];
                const float4 c4 = *reinterpret_cast<const float4 *>(cv + cc * CH + 4 * l4);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float4 y4 = *reinterpret_cast<const float4 *>(cur + (lane + 32 * j) * YST + 4 * l4);
                    bad[j] |= !isfinite(y4.x) || !isfinite(y4.y) || !isfinite(y4.z) || !isfinite(y4.w);
                    yv[j][0] = y4.x - c4.x; yv[j][1] = y4.y - c4.y; yv[j][2] = y4.z - c4.z; yv[j][3] = y4.w - c4.w;
                }
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    const float *arow = Acp + (size_t)(cc * CH + 4 * l4 + q) * R;
                    const float2 y01 = make_float2(yv[0][q], yv[1][q]), y23 = make_float2(yv[2][q], yv[3][q]);
#pragma unroll
                    for (int r4 = 0; r4 < R / 4; ++r4) {
                        const float4 a4 = *reinterpret_cast<const float4 *>(arow + 4 * r4);
                        acc[4 * r4 + 0][0] = fma2(a4.x, y01, acc[4 * r4 + 0][0]); acc[4 * r4 + 0][1] = fma2(a4.x, y23, acc[4 * r4 + 0][1]);
                        acc[4 * r4 + 1][0] = fma2(a4.y, y01, acc[4 * r4 + 1][0]); acc[4 * r4 + 1][1] = fma2(a4.y, y23, acc[4 * r4 + 1][1]);
                        acc[4 * r4 + 2][0] = fma2(a4.z, y01, acc[4 * r4 + 2][0]); acc[4 * r4 + 2][1] = fma2(a4.z, y23, acc[4 * r4 + 2][1]);
                        acc[4 * r4 + 3][0] = fma2(a4.w, y01, acc[4 * r4 + 3][0]); acc[4 * r4 + 3][1] = fma2(a4.w, y23, acc[4 * r4 + 3][1]);
                    }
                }
            }
            __syncwarp();
        }
        // ---- both pixel pairs wait in shared memory (the stage buffers are free now) and are taken to their start
        //      point one after the other: b, x and G x of a pair are 192 registers
        float2 *park = reinterpret_cast<float2 *>(ybuf) + lane;     // [2][32][32 lanes] float2 (16 KB of the 20 KB stage area)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            park[r * 32] = acc[r][0];
            park[(R + r) * 32] = acc[r][1];
        }
#pragma unroll 1
        for (int pp = 0; pp < 2; ++pp) {
            float2 b2[R];
#pragma unroll
            for (int r = 0; r < R; ++r) b2[r] = park[(pp * R + r) * 32];
            const bool bad0 = pp ? bad[2] : bad[0], bad1 = pp ? bad[3] : bad[1];
            float2 bmax = make_float2(0.0f, 0.0f);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                if (bad0) b2[r].x = 0.0f;
                if (bad1) b2[r].y = 0.0f;
                bmax.x = fmaxf(bmax.x, fabsf(b2[r].x)); bmax.y = fmaxf(bmax.y, fabsf(b2[r].y));
            }
            const float2 sc = make_float2(fmaxf(bmax.x, 1e-3f * gdmax), fmaxf(bmax.y, 1e-3f * gdmax));
            // the pair's slot of the park area is free now: scratch for one vector (x, then G x)
            float2 *scr = park + pp * R * 32;
            // x = Gi b (matrix rows broadcast from shared memory, packed FMAs over the pixel pair); the row loop is
            // ROLLED (the result goes through the scratch vector): straight-line code for both mat-vecs was 50 KB for
            // 8 warps and the kernel stalled on instruction fetch
            float2 sx = make_float2(0.0f, 0.0f);
#pragma unroll 2
            for (int r = 0; r < R; ++r) {
                float2 s0 = make_float2(0.0f, 0.0f), s1 = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int c4 = 0; c4 < R / 4; ++c4) {
                    const float4 g4 = *reinterpret_cast<const float4 *>(Gis + r * R + 4 * c4);
                    s0 = fma2(g4.x, b2[4 * c4 + 0], s0); s1 = fma2(g4.y, b2[4 * c4 + 1], s1);
                    s0 = fma2(g4.z, b2[4 * c4 + 2], s0); s1 = fma2(g4.w, b2[4 * c4 + 3], s1);
                }
                const float2 xr = make_float2(s0.x + s1.x, s0.y + s1.y);
                scr[r * 32] = xr;
                sx.x += xr.x; sx.y += xr.y;
            }
            const float2 mu0 = make_float2((sx.x - 1.0f) * rGiqTot, (sx.y - 1.0f) * rGiqTot);
            float2 x2[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float q = Giq[r];
                const float2 xr = scr[r * 32];
                x2[r] = make_float2(fmaf(-mu0.x, q, xr.x), fmaf(-mu0.y, q, xr.y));
            }
            // G x into the scratch vector; gradient at x: g = G x - b; nu = -g'x; shifts into the interior
            float2 gx = make_float2(0.0f, 0.0f), mnx = make_float2(INFINITY, INFINITY), mng = mnx;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float2 s0 = make_float2(0.0f, 0.0f), s1 = make_float2(0.0f, 0.0f);
#pragma unroll
                for (int c4 = 0; c4 < R / 4; ++c4) {
                    const float4 g4 = *reinterpret_cast<const float4 *>(Gs + r * R + 4 * c4);
                    s0 = fma2(g4.x, x2[4 * c4 + 0], s0); s1 = fma2(g4.y, x2[4 * c4 + 1], s1);
                    s0 = fma2(g4.z, x2[4 * c4 + 2], s0); s1 = fma2(g4.w, x2[4 * c4 + 3], s1);
                }
                const float2 gar = make_float2(s0.x + s1.x, s0.y + s1.y);
                scr[r * 32] = gar;
                const float2 g = make_float2(gar.x - b2[r].x, gar.y - b2[r].y);
                gx.x = fmaf(g.x, x2[r].x, gx.x); gx.y = fmaf(g.y, x2[r].y, gx.y);
                mnx.x = fminf(mnx.x, x2[r].x); mnx.y = fminf(mnx.y, x2[r].y);
                mng.x = fminf(mng.x, g.x); mng.y = fminf(mng.y, g.y);
            }
            float2 nu = cons ? make_float2(-gx.x, -gx.y) : make_float2(0.0f, 0.0f);
            const float2 dp = make_float2(fmaxf(-mnx.x, 0.0f), fmaxf(-mnx.y, 0.0f));
            const float2 dd = make_float2(fmaxf(-(mng.x + nu.x), 0.0f), fmaxf(-(mng.y + nu.y), 0.0f));
            float2 cl = make_float2(nu.x + dd.x, nu.y + dd.y);          // lambda = g + cl
            float2 xl = make_float2(0.0f, 0.0f), sl = xl, sxx = xl, lmx = make_float2(-INFINITY, -INFINITY);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float2 xs = make_float2(x2[r].x + dp.x, x2[r].y + dp.y);
                const float2 gar = scr[r * 32];
                const float2 ls = make_float2(gar.x - b2[r].x + cl.x, gar.y - b2[r].y + cl.y);
                xl.x = fmaf(xs.x, ls.x, xl.x); xl.y = fmaf(xs.y, ls.y, xl.y);
                sl.x += ls.x; sl.y += ls.y; sxx.x += xs.x; sxx.y += xs.y;
                lmx.x = fmaxf(lmx.x, ls.x); lmx.y = fmaxf(lmx.y, ls.y);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int j = 2 * pp + h;
                const int64_t p = p0 + lane + 32 * j;
#define H_(v) (h ? (v).y : (v).x)
                const float sch = H_(sc), bmx = H_(bmax);
                const float xlh = H_(xl);
                const float dp2 = 0.05f * xlh * rcp_approx(fmaxf(H_(sl), 1e-30f));
                const float dd2 = 0.05f * xlh * rcp_approx(fmaxf(H_(sxx), 1e-30f));
                const float xsh = H_(dp) + dp2 + 1e-3f;                     // a = (x + xsh) / sa
                const float lsh = H_(cl) + dd2 + 1e-4f * sch;               // lambda = g + lsh
                const float sa = H_(sxx) + 32.0f * (dp2 + 1e-3f);
                float lam0 = H_(lmx) + dd2 + 1e-4f * sch;
                const float rsa = cons ? 1.0f / sa : 1.0f;
                float nuh = H_(nu);
                const bool flat = !(lam0 > 0.0f) || !isfinite(lam0) || !isfinite(sa);      // degenerate data
                if (flat) { lam0 = fmaxf(bmx, 1e-3f * gdmax); nuh = 0.0f; }
                if (p < p_end) {
                    float *o = rec + (p - p_begin) * REC;
                    float gap = 0.0f, suma = 0.0f;      // a'lambda and sum a of the start point (mu and r_p of iteration 0)
                    // lane-major order of the iteration kernel: position 8 t + s <- row t + 4 s
#pragma unroll
                    for (int t = 0; t < 4; ++t)
#pragma unroll
                        for (int hh = 0; hh < 2; ++hh) {
                            float av[4], lv[4], gv[4];
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int r = t + 16 * hh + 4 * e;
                                const float bb = H_(b2[r]), gg = H_(scr[r * 32]);
                                av[e] = flat ? (1.0f / 32.0f) : (H_(x2[r]) + xsh) * rsa;
                                lv[e] = flat ? lam0 : (gg - bb) + lsh;
                                // G a of the shifted, normalised point, minus b
                                gv[e] = (flat ? Grs[r] * (1.0f / 32.0f) : fmaf(xsh, Grs[r], gg) * rsa) - bb;
                                gap = fmaf(av[e], lv[e], gap); suma += av[e];
                            }
                            *reinterpret_cast<float4 *>(o + 8 * t + 4 * hh) = make_float4(av[0], av[1], av[2], av[3]);
                            *reinterpret_cast<float4 *>(o + 32 + 8 * t + 4 * hh) = make_float4(lv[0], lv[1], lv[2], lv[3]);
                            *reinterpret_cast<float4 *>(o + 64 + 8 * t + 4 * hh) = make_float4(gv[0], gv[1], gv[2], gv[3]);
                        }
                    const bool bd = h ? bad1 : bad0;
                    *reinterpret_cast<float4 *>(o + 96) = make_float4(nuh, sch, lam0, __int_as_float(bd ? LINMIN_INFO_NONFINITE_INPUT : 0));
                    *reinterpret_cast<float4 *>(o + 100) = make_float4(gap * (1.0f / 32.0f), cons ? suma - 1.0f : 0.0f, 0.0f, 0.0f);
                }
#undef H_
            }
        }
        __syncwarp();
    }
}

inline size_t start_r32_smem(int L, int warps) {
    return (s32::lib_floats(L) + (size_t)warps * s32::warp_floats()) * sizeof(float);
}
inline int start_r32_warps(int L) {
    int w = s32::WARPS;
    while (w > 1 && start_r32_smem(L, w) > 226 * 1024) --w;
    return start_r32_smem(L, w) <= 226 * 1024 ? w : 0;
}

inline cudaError_t launch_start_r32(const LibView &lv, const SolveParams &prm, int64_t p_begin, int64_t p_end,
                                    float *rec, int sm_count, cudaStream_t stream) {
    const int warps = start_r32_warps(lv.L);
    if (warps < 1) return cudaErrorInvalidConfiguration;
    const size_t smem = start_r32_smem(lv.L, warps);
    cudaError_t e = lv.cons ? cudaFuncSetAttribute(start_r32_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
                            : cudaFuncSetAttribute(start_r32_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int64_t tiles = (p_end - p_begin + s32::TP - 1) / s32::TP;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((tiles + warps - 1) / warps, sm_count));
    if (lv.cons) start_r32_kernel<true><<<grid, s32::WARPS * 32, smem, stream>>>(lv, prm, p_begin, p_end, rec, warps);
    else start_r32_kernel<false><<<grid, s32::WARPS * 32, smem, stream>>>(lv, prm, p_begin, p_end, rec, warps);
    return cudaGetLastError();
}

}  // namespace linmin
