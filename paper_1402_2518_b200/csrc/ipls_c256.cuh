// ipls_c256.cuh -- projection + IPLS for 65 <= R <= 256: one CTA per pixel, the Newton matrix in shared memory as
// 32 x 32 blocks, blocked Cholesky factorisation with the trailing updates on the tensor cores (sm_100a).
//
// Same iteration as ipls_generic.cuh (read its header: PAPER.md:71-73 names IPLS and prints no steps, DESIGN.md reading
// R1; Mehrotra predictor-corrector on the centred per-pixel QP, nu eliminated through M^-1 1, G a carried along with
// a).  What differs is how M = Gc + diag(lambda / a) is factored and solved with (SURVEY.md 8(a) a2 "warp group for
// large R"; PAPER.md:92 sizes the method by R):
//   * 256 threads, thread i owns entry i of every vector in REGISTERS; shared memory holds the lower block triangle of
//     M (blocks of 32 x 32, row stride 36: conflict-free for the mma fragments and for 16-byte row accesses);
//   * panel p: one warp factors the diagonal block (rows in registers, right-looking, column exchanged through a
//     64-float line) and replaces it by the INVERSE W of its Cholesky factor, so that everything below is a product:
//     L_Ip = M_Ip W' and M_IJ -= L_Ip L_Jp' are 32 x 32 x 32 block products on mma.sync.m16n8k8 in 3 x TF32 (big x small,
//     small x big, big x big: fp32-class accuracy, fp32 accumulate) -- at R = 256 the factorisation is a 256^3/3-flop
//     contraction per iteration, > 95 % of this path's work, the one dense contraction of the method;
//   * the triangular solves use W as well: a block row is a 32 x 32 mat-vec by one warp, followed by rank-32 updates
//     of the right-hand sides by everybody, one CTA barrier per block.
// M is rebuilt every iteration from a zero-padded copy of Gc (LibView::Gpad, stride 32 ceil(R / 32), identity on the
// padded diagonal) with 16-byte cp.async: 148 KB from L2 per iteration.
#pragma once
#include "common.cuh"

namespace linmin {
namespace c256 {

constexpr int NT = 256;            // threads per CTA
constexpr int BS = 36;             // row stride (floats) of a block
constexpr int BLK = 32 * BS;       // floats per block
constexpr unsigned FULL = 0xffffffffu;

__host__ __device__ inline int nblocks(int R) { return (R + 31) >> 5; }
__host__ __device__ inline int blk(int I, int J) { return (I * (I + 1) / 2 + J) * BLK; }      // I >= J
// shared memory (floats): blocks | yc[L4] | xs0[Rp] | xs1[Rp] | dgs[Rp] | line[128] | red[64]
__host__ __device__ inline size_t smem_floats(int L, int R) {
    const int NB = nblocks(R), Rp = 32 * NB, L4 = (L + 3) & ~3;
    return (size_t)(NB * (NB + 1) / 2) * BLK + L4 + 3 * (size_t)Rp + 192;
}

// x = big + small with big the leading 11 significand bits (the tensor core reads the upper 19 bits of a tf32 operand, so
// `small` needs no rounding of its own: 22 of the 24 bits take part; cvt.rna.tf32 is a 6-instruction emulation here)
__device__ __forceinline__ void split_tf32(float x, uint32_t &big, uint32_t &small) {
    big = __float_as_uint(x) & 0xffffe000u;
    small = __float_as_uint(x - __uint_as_float(big));
}
__device__ __forceinline__ void mma_tf32(float (&c)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// One warp: C = X Y' (UPDATE false) or C -= X Y' (UPDATE true: accumulates X Y' - C and stores the negative);
// X, Y, C are 32 x 32 blocks of stride BS; C may alias X (X is read in full first)
template <bool UPDATE>
__device__ __forceinline__ void block_product(float *C, const float *X, const float *Y, int lane) {
    const int g = lane >> 2, t = lane & 3;
    float acc[2][4][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            if (UPDATE) {
                const float2 lo = *reinterpret_cast<const float2 *>(C + (16 * mt + g) * BS + 8 * nt + 2 * t);
                const float2 hi = *reinterpret_cast<const float2 *>(C + (16 * mt + g + 8) * BS + 8 * nt + 2 * t);
                acc[mt][nt][0] = -lo.x; acc[mt][nt][1] = -lo.y; acc[mt][nt][2] = -hi.x; acc[mt][nt][3] = -hi.y;
            } else {
                acc[mt][nt][0] = acc[mt][nt][1] = acc[mt][nt][2] = acc[mt][nt][3] = 0.0f;
            }
        }
    uint32_t ab[4][2][4], as[4][2][4];      // X fragments of all four k-steps (C may alias X)
#pragma unroll
    for (int ks = 0; ks < 4; ++ks)
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
            const float *x = X + (16 * mt + g) * BS + 8 * ks + t;
            split_tf32(x[0], ab[ks][mt][0], as[ks][mt][0]);
            split_tf32(x[8 * BS], ab[ks][mt][1], as[ks][mt][1]);
            split_tf32(x[4], ab[ks][mt][2], as[ks][mt][2]);
            split_tf32(x[8 * BS + 4], ab[ks][mt][3], as[ks][mt][3]);
        }
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            const float *y = Y + (8 * nt + g) * BS + 8 * ks + t;
            uint32_t bb[2], bs[2];
            split_tf32(y[0], bb[0], bs[0]);
            split_tf32(y[4], bb[1], bs[1]);
#pragma unroll
            for (int mt = 0; mt < 2; ++mt) {
                mma_tf32(acc[mt][nt], as[ks][mt], bb);
                mma_tf32(acc[mt][nt], ab[ks][mt], bs);
                mma_tf32(acc[mt][nt], ab[ks][mt], bb);
            }
        }
    }
    __syncwarp();
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) {
            const float sg = UPDATE ? -1.0f : 1.0f;
            *reinterpret_cast<float2 *>(C + (16 * mt + g) * BS + 8 * nt + 2 * t) = make_float2(sg * acc[mt][nt][0], sg * acc[mt][nt][1]);
            *reinterpret_cast<float2 *>(C + (16 * mt + g + 8) * BS + 8 * nt + 2 * t) = make_float2(sg * acc[mt][nt][2], sg * acc[mt][nt][3]);
        }
}

// One warp: B <- W = L^-1 (lower triangular, zeros above the diagonal) for the Cholesky factor L of the 32 x 32 diagonal
// block B (read in full: it is symmetric).  B = L~ D L~' with L~ = E_0 E_1 .. E_30, E_j = I + l_j e_j' (l_j: the
// multipliers of step j), so L~^-T = (I - e_0 l_0')(I - e_1 l_1') .. : lane i holds row i of the Schur complement (m) and
// row i of U = L~^-T (u), and step j is, for both, "entry k -= (entry j / p_j) c_k" with c = column j of the Schur
// complement -- which every lane contributes ONE element of (one conflict-free store, then eight broadcast loads).
// Both rows are kept shifted so that entry j sits in register 0 (each FMA writes one register to the left: no register
// index depends on j, no moves), the column is stored rotated the same way, and the loop is ROLLED on purpose: fully
// unrolled, the sweep was 32 KB of straight-line code run by a single warp and took 11.8 k cycles per block, one
// instruction-cache miss per 128-byte line.  Column j of U is final at step j and goes straight to row j of W,
// scaled by p_j^-1/2 (W = D^-1/2 L~^-1).  A pivot below floorv is clamped (returns true if that happened).
// The sweep is shared by TWO warps (role 0: the rows m and the column exchange; role 1: the rows u and the output), which
// meet at named barrier 1 once per step: 31 FMAs per step and warp instead of 62 on the dependent chain.
__device__ __forceinline__ bool factor_diag(float *B, float *line, float floorv, int lane, int role) {
    float v[32];                                          // role 0: row `lane` of m; role 1: row `lane` of u
    if (role == 0) {
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 x = *reinterpret_cast<const float4 *>(B + lane * BS + 4 * q);
            v[4 * q] = x.x; v[4 * q + 1] = x.y; v[4 * q + 2] = x.z; v[4 * q + 3] = x.w;
        }
        line[lane] = v[0];
    } else {
#pragma unroll
        for (int k = 0; k < 32; ++k) v[k] = (k == lane) ? 1.0f : 0.0f;
    }
    bool clamped = false;
    float c[32];
    asm volatile("bar.sync 1, 64;" ::: "memory");         // (also: B has been read in full; row j is written at step j)
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float4 c4 = *reinterpret_cast<const float4 *>(line + 4 * q);
        c[4 * q] = c4.x; c[4 * q + 1] = c4.y; c[4 * q + 2] = c4.z; c[4 * q + 3] = c4.w;
    }
    // software pipeline: the entry of column j + 1 is computed, stored and the next line requested BEFORE the FMAs of
    // step j, which then cover the store-to-load round trip.  (Taking the next pivot from its owner by shuffle, to get the
    // reciprocal off the chain, was slower: 5.2 k -> 8 k cycles per block.)
#pragma unroll 2
    for (int j = 0; j < 32; ++j) {
        float pj = c[0];
        if (!(pj > floorv)) { pj = floorv; clamped = true; }
        const float lv = -v[0] * rcp_approx(pj);
        float *cbn = line + 32 * ((j + 1) & 1);
        if (role == 0) cbn[(lane - j - 1) & 31] = fmaf(lv, c[1], v[1]);   // column j + 1, rotated: index r = row j + 1 + r
        else B[j * BS + lane] = v[0] * rsqrtf(pj);
        asm volatile("bar.sync 1, 64;" ::: "memory");
        float cn[32];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const float4 c4 = *reinterpret_cast<const float4 *>(cbn + 4 * q);
            cn[4 * q] = c4.x; cn[4 * q + 1] = c4.y; cn[4 * q + 2] = c4.z; cn[4 * q + 3] = c4.w;
        }
#pragma unroll
        for (int r = 1; r < 32; ++r) v[r - 1] = fmaf(lv, c[r], v[r]);
        v[31] = 0.0f;
#pragma unroll
        for (int r = 0; r < 32; ++r) c[r] = cn[r];
    }
    return clamped;
}

// In-place blocked Cholesky of the block lower triangle; on return block (p, p) holds W_pp = L_pp^-1 and the blocks
// below the diagonal hold L.  All 256 threads call it.
__device__ __forceinline__ bool factor_blocks(float *Mb, float *line, int NB, float floorv, int warp, int lane) {
    bool clamped = false;
    // Look-ahead: once the blocks of column p + 1 have their update of panel p, warps 0 and 1 factor the next diagonal
    // block while the other warps finish the trailing update (the diagonal sweep is 32 dependent steps).
    if (warp < 2) clamped |= factor_diag(Mb + blk(0, 0), line, floorv, lane, warp);
    __syncthreads();
    for (int p = 0; p < NB; ++p) {
        for (int I = p + 1 + warp; I < NB; I += NT / 32)
            block_product<false>(Mb + blk(I, p), Mb + blk(I, p), Mb + blk(p, p), lane);
        __syncthreads();
        if (p + 1 >= NB) break;
        for (int I = p + 1 + warp; I < NB; I += NT / 32)               // column p + 1 first
            block_product<true>(Mb + blk(I, p + 1), Mb + blk(I, p), Mb + blk(p + 1, p), lane);
        __syncthreads();
        if (warp < 2) {
            clamped |= factor_diag(Mb + blk(p + 1, p + 1), line, floorv, lane, warp);
        } else {
            int n = 0;
            for (int J = p + 2; J < NB; ++J)
                for (int I = J; I < NB; ++I, ++n)
                    if (n % (NT / 32 - 2) == warp - 2)
                        block_product<true>(Mb + blk(I, J), Mb + blk(I, p), Mb + blk(J, p), lane);
        }
        __syncthreads();
    }
    return clamped;
}

// dot products of one 32-float row (16-byte loads) with one or two 32-float vectors, four accumulators each
template <int NRHS>
__device__ __forceinline__ void row_dot(const float *row, const float *v0, const float *v1, float &r0, float &r1) {
    float s[4] = {0.0f, 0.0f, 0.0f, 0.0f}, u[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float4 a4 = *reinterpret_cast<const float4 *>(row + 4 * q);
        const float4 x4 = *reinterpret_cast<const float4 *>(v0 + 4 * q);
        s[0] = fmaf(a4.x, x4.x, s[0]); s[1] = fmaf(a4.y, x4.y, s[1]); s[2] = fmaf(a4.z, x4.z, s[2]); s[3] = fmaf(a4.w, x4.w, s[3]);
        if (NRHS > 1) {
            const float4 y4 = *reinterpret_cast<const float4 *>(v1 + 4 * q);
            u[0] = fmaf(a4.x, y4.x, u[0]); u[1] = fmaf(a4.y, y4.y, u[1]); u[2] = fmaf(a4.z, y4.z, u[2]); u[3] = fmaf(a4.w, y4.w, u[3]);
        }
    }
    r0 = (s[0] + s[1]) + (s[2] + s[3]);
    r1 = (u[0] + u[1]) + (u[2] + u[3]);
}
// the same down one column of a block (element k at col[k BS])
template <int NRHS>
__device__ __forceinline__ void col_dot(const float *col, const float *v0, const float *v1, float &r0, float &r1) {
    float s[4] = {0.0f, 0.0f, 0.0f, 0.0f}, u[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const float4 x4 = *reinterpret_cast<const float4 *>(v0 + 4 * q);
        const float a0 = col[(4 * q + 0) * BS], a1 = col[(4 * q + 1) * BS], a2 = col[(4 * q + 2) * BS], a3 = col[(4 * q + 3) * BS];
        s[0] = fmaf(a0, x4.x, s[0]); s[1] = fmaf(a1, x4.y, s[1]); s[2] = fmaf(a2, x4.z, s[2]); s[3] = fmaf(a3, x4.w, s[3]);
        if (NRHS > 1) {
            const float4 y4 = *reinterpret_cast<const float4 *>(v1 + 4 * q);
            u[0] = fmaf(a0, y4.x, u[0]); u[1] = fmaf(a1, y4.y, u[1]); u[2] = fmaf(a2, y4.z, u[2]); u[3] = fmaf(a3, y4.w, u[3]);
        }
    }
    r0 = (s[0] + s[1]) + (s[2] + s[3]);
    r1 = (u[0] + u[1]) + (u[2] + u[3]);
}

// (L L') x = rhs in place for NRHS right-hand sides (x0, x1: Rp floats each in shared memory); thread t owns row t.
// Ends with a CTA barrier.
template <int NRHS>
__device__ __forceinline__ void solve_blocks(const float *Mb, int NB, float *x0, float *x1, int tid) {
    const int I = tid >> 5, i = tid & 31;
    // ---- forward, L z = r:  z_p = W_pp r_p, then r_q -= L_qp z_p for q > p
    for (int p = 0; p < NB; ++p) {
        if (I == p) {
            float s0, s1;
            row_dot<NRHS>(Mb + blk(p, p) + i * BS, x0 + 32 * p, x1 + 32 * p, s0, s1);
            __syncwarp();
            x0[tid] = s0;
            if (NRHS > 1) x1[tid] = s1;
        }
        __syncthreads();
        if (I > p && I < NB) {
            float s0, s1;
            row_dot<NRHS>(Mb + blk(I, p) + i * BS, x0 + 32 * p, x1 + 32 * p, s0, s1);
            x0[tid] -= s0;
            if (NRHS > 1) x1[tid] -= s1;
        }
        // (no barrier here: the next diagonal step touches block row p + 1 only, which its own warp has just updated)
        __syncwarp();
    }
    __syncthreads();
    // ---- backward, L' x = z:  x_p = W_pp' z_p, then z_q -= L_pq' x_p for q < p
    for (int p = NB - 1; p >= 0; --p) {
        if (I == p) {
            float s0, s1;
            col_dot<NRHS>(Mb + blk(p, p) + i, x0 + 32 * p, x1 + 32 * p, s0, s1);
            __syncwarp();
            x0[tid] = s0;
            if (NRHS > 1) x1[tid] = s1;
        }
        __syncthreads();
        if (I < p) {
            float s0, s1;
            col_dot<NRHS>(Mb + blk(p, I) + i, x0 + 32 * p, x1 + 32 * p, s0, s1);
            x0[tid] -= s0;
            if (NRHS > 1) x1[tid] -= s1;
        }
        __syncwarp();
    }
    __syncthreads();
}

// CTA reductions of up to three values at once (red: 32 floats, 8 warps x 3 + results)
struct Red {
    float *red;
    int warp, lane;
    template <typename Op>
    __device__ __forceinline__ float one(float v, Op op, float ident) const {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v = op(v, __shfl_xor_sync(FULL, v, o));
        __syncthreads();                          // the previous result has been read by everybody
        if (lane == 0) red[warp] = v;
        __syncthreads();
        float r = (lane < NT / 32) ? red[lane] : ident;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) r = op(r, __shfl_xor_sync(FULL, r, o));
        return __shfl_sync(FULL, r, 0);
    }
    __device__ __forceinline__ float sum(float v) const { return one(v, [](float a, float b) { return a + b; }, 0.0f); }
    __device__ __forceinline__ float max(float v) const { return one(v, [](float a, float b) { return fmaxf(a, b); }, -INFINITY); }
    __device__ __forceinline__ float min(float v) const { return one(v, [](float a, float b) { return fminf(a, b); }, INFINITY); }
    // three sums in one pass
    __device__ __forceinline__ void sum3(float &a, float &b, float &c) const {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_xor_sync(FULL, a, o); b += __shfl_xor_sync(FULL, b, o); c += __shfl_xor_sync(FULL, c, o);
        }
        __syncthreads();
        if (lane == 0) { red[warp] = a; red[8 + warp] = b; red[16 + warp] = c; }
        __syncthreads();
        float r = (lane < 24) ? red[lane] : 0.0f;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) r += __shfl_xor_sync(FULL, r, o);
        a = __shfl_sync(FULL, r, 0); b = __shfl_sync(FULL, r, 8); c = __shfl_sync(FULL, r, 16);
    }
    // two minima in one pass
    __device__ __forceinline__ void min2(float &a, float &b) const {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a = fminf(a, __shfl_xor_sync(FULL, a, o)); b = fminf(b, __shfl_xor_sync(FULL, b, o));
        }
        __syncthreads();
        if (lane == 0) { red[warp] = a; red[8 + warp] = b; }
        __syncthreads();
        float r = (lane < 16) ? red[lane] : INFINITY;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) r = fminf(r, __shfl_xor_sync(FULL, r, o));
        a = __shfl_sync(FULL, r, 0); b = __shfl_sync(FULL, r, 8);
    }
};

}  // namespace c256

// Gpad: zero-padded copy of Gc for the 16-byte staging of ipls_c256_kernel (Rp x Rp, identity on the padded diagonal)
__global__ void pad_gram_kernel(const float *__restrict__ Gc, int R, int Rp, float *__restrict__ Gpad) {
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < Rp * Rp; e += gridDim.x * blockDim.x) {
        const int i = e / Rp, j = e - i * Rp;
        Gpad[e] = (i < R && j < R) ? Gc[(size_t)i * R + j] : (i == j ? 1.0f : 0.0f);
    }
}

// One CTA per pixel (dynamic ticket), 256 threads; thread i owns entry i of a, lambda, b, G a, ...
__global__ void __launch_bounds__(c256::NT, 1)
ipls_c256_kernel(LibView lib, SolveParams prm, unsigned int *__restrict__ counter) {
    using namespace c256;
    extern __shared__ __align__(16) float smem[];
    if (lib.flags[0]) return;
    const int L = lib.L, R = lib.R, NB = nblocks(R), Rp = 32 * NB, L4 = (L + 3) & ~3;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float *Mb = smem;
    float *yc = Mb + (size_t)(NB * (NB + 1) / 2) * BLK;
    float *xs0 = yc + L4, *xs1 = xs0 + Rp, *dgs = xs1 + Rp, *line = dgs + Rp, *redm = line + 128;
    const Red rd{redm, warp, lane};
    __shared__ unsigned int s_ticket;
    const float gdmax = lib.scal[0];
    const float fR = (float)R, tau = 0.995f;
    const bool live = tid < R;
    const bool cons = lib.cons != 0;
    const float giq = live ? lib.Giq[tid] : 0.0f;

    while (true) {
        if (tid == 0) s_ticket = atomicAdd(counter, 1u);
        __syncthreads();
        const int64_t p = (int64_t)s_ticket;
        __syncthreads();
        if (p >= prm.N) break;
        // ---- load spectrum, centre it, detect non-finite input
        const float *y = prm.Y + p * prm.ldY;
        float badf = 0.0f;
        for (int l = tid; l < L; l += NT) {
            const float yv = y[l];
            if (!isfinite(yv)) badf = 1.0f;
            yc[l] = yv - lib.c[l];
        }
        badf = rd.max(badf);                    // (its barriers publish yc)
        if (badf > 0.0f) {
            if (live) prm.coeffs[p * R + tid] = 1.0f / fR;
            if (prm.info && tid == 0) prm.info[p] = LINMIN_INFO_NONFINITE_INPUT;
            continue;
        }
        // ---- projection b = Ac'(y - c)   ("X.S^T")
        float b = 0.0f;
        if (live) {
            float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;
            int l = 0;
#pragma unroll 4
            for (; l + 3 < L; l += 4) {
                s0 = fmaf(lib.Ac[(size_t)(l + 0) * R + tid], yc[l + 0], s0);
                s1 = fmaf(lib.Ac[(size_t)(l + 1) * R + tid], yc[l + 1], s1);
                s2 = fmaf(lib.Ac[(size_t)(l + 2) * R + tid], yc[l + 2], s2);
                s3 = fmaf(lib.Ac[(size_t)(l + 3) * R + tid], yc[l + 3], s3);
            }
            for (; l < L; ++l) s0 = fmaf(lib.Ac[(size_t)l * R + tid], yc[l], s0);
            b = (s0 + s1) + (s2 + s3);
        }
        const float bmax = rd.max(live ? fabsf(b) : 0.0f);
        const float sc = fmaxf(bmax, 1e-3f * gdmax);
        // ---- start (Mehrotra's heuristic, as in ipls_generic.cuh): the sum-constrained LS point of the regularised
        //      problem, x = Gi b - q (1'Gi b - 1)/(1'q), its reduced gradient as multipliers, both shifted inside
        float a, lam, Ga, nu, lam0;
        {
            if (tid < Rp) xs0[tid] = b;         // (padded entries are 0)
            __syncthreads();
            float x = 0.0f;
            if (live) {
                float s0 = 0.0f, s1 = 0.0f, s2 = 0.0f, s3 = 0.0f;
                int j = 0;
#pragma unroll 4
                for (; j + 3 < R; j += 4) {
                    s0 = fmaf(lib.Gi[(size_t)(j + 0) * R + tid], xs0[j + 0], s0);
                    s1 = fmaf(lib.Gi[(size_t)(j + 1) * R + tid], xs0[j + 1], s1);
                    s2 = fmaf(lib.Gi[(size_t)(j + 2) * R + tid], xs0[j + 2], s2);
                    s3 = fmaf(lib.Gi[(size_t)(j + 3) * R + tid], xs0[j + 3], s3);
                }
                for (; j < R; ++j) s0 = fmaf(lib.Gi[(size_t)j * R + tid], xs0[j], s0);
                x = (s0 + s1) + (s2 + s3);
            }
            float sx = x, sq = giq, dummy = 0.0f;
            rd.sum3(sx, sq, dummy);
            const float mu0 = cons ? (sx - 1.0f) / sq : 0.0f;
            x = fmaf(-mu0, giq, x);
            if (tid < Rp) xs1[tid] = x;
            __syncthreads();
            float gxv = 0.0f, rs = 0.0f;     // (G x)_i and the row sum of G
            if (live) {
                float s0 = 0.0f, s1 = 0.0f, r0 = 0.0f, r1 = 0.0f;
                int j = 0;
#pragma unroll 4
                for (; j + 1 < R; j += 2) {
                    const float g0 = lib.Gc[(size_t)(j + 0) * R + tid], g1 = lib.Gc[(size_t)(j + 1) * R + tid];
                    s0 = fmaf(g0, xs1[j + 0], s0); r0 += g0;
                    s1 = fmaf(g1, xs1[j + 1], s1); r1 += g1;
                }
                for (; j < R; ++j) { const float g0 = lib.Gc[(size_t)j * R + tid]; s0 = fmaf(g0, xs1[j], s0); r0 += g0; }
                gxv = s0 + s1; rs = r0 + r1;
            }
            const float gi = gxv - b;
            float gx = live ? gi * x : 0.0f;
            float mnx = live ? x : INFINITY, mng = live ? gi : INFINITY;
            gx = rd.sum(gx);
            rd.min2(mnx, mng);
            nu = cons ? -gx : 0.0f;
            const float dp = fmaxf(-mnx, 0.0f), dd = fmaxf(-(mng + nu), 0.0f);
            const float xi = x + dp, li = gi + nu + dd;
            float xl = live ? xi * li : 0.0f, sl = live ? li : 0.0f, sxx = live ? xi : 0.0f;
            rd.sum3(xl, sl, sxx);
            const float dp2 = 0.05f * xl / fmaxf(sl, 1e-30f), dd2 = 0.05f * xl / fmaxf(sxx, 1e-30f);
            a = xi + dp2 + 1e-3f;
            lam = li + dd2 + 1e-4f * sc;
            const float sa = rd.sum(live ? a : 0.0f);
            lam0 = rd.max(live ? lam : -INFINITY);
            const float rsa = cons ? 1.0f / sa : 1.0f;      // pos: the point is not normalised
            const bool ok = (lam0 > 0.0f) && isfinite(lam0) && isfinite(sa) && isfinite(rsa);
            if (!ok) { lam0 = fmaxf(bmax, 1e-3f * gdmax); nu = 0.0f; }
            if (ok) {
                a *= rsa;
                Ga = fmaf(dp + dp2 + 1e-3f, rs, gxv) * rsa;      // G a of the shifted, normalised point
            } else {                                              // degenerate data: the barycentre
                a = 1.0f / fR; lam = lam0; Ga = rs / fR;
            }
            if (!live) { a = 1.0f; lam = 0.0f; Ga = 0.0f; }
        }
        int iters = 0, flags = 0;
        for (int it = 0;; ++it) {
            // ---- residuals
            const float w = Ga - b + nu;          // G a is carried along with a (Newton identity, see the update)
            float rdmax = live ? fabsf(w - lam) : 0.0f;
            float suma = live ? a : 0.0f, gap = live ? a * lam : 0.0f, dummy = 0.0f;
            rdmax = rd.max(rdmax);
            rd.sum3(suma, gap, dummy);
            const float rp = cons ? suma - 1.0f : 0.0f;
            if (gap <= prm.gap_tol * sc && rdmax <= prm.feas_tol * sc && fabsf(rp) <= prm.feas_tol) {
                flags |= LINMIN_INFO_CONVERGED;
                break;
            }
            if (it >= prm.max_iter) { flags |= LINMIN_INFO_MAX_ITER; break; }
            ++iters;
            const float mu = gap / fR;
            const float di = live ? lam / a : 0.0f;
            // ---- Newton matrix M = Gc + diag(lambda / a): blocks staged from the padded Gram matrix by cp.async
            {
                // a block is 32 rows of 8 16-byte chunks = one chunk per thread
                const int r = tid >> 3, ch = tid & 7;
                int bi = 0;
                for (int I = 0; I < NB; ++I)
                    for (int J = 0; J <= I; ++J, ++bi) {
                        const float *src = lib.Gpad + (size_t)(32 * I + r) * Rp + 32 * J + 4 * ch;
                        const unsigned dst = (unsigned)__cvta_generic_to_shared(Mb + (size_t)bi * BLK + r * BS + 4 * ch);
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src));
                    }
                asm volatile("cp.async.commit_group;");
                asm volatile("cp.async.wait_group 0;");
                __syncthreads();
                if (tid < Rp) Mb[blk(warp, warp) + lane * BS + lane] += di;
                __syncthreads();
            }
            if (factor_blocks(Mb, line, NB, 1e-12f * gdmax, warp, lane)) flags |= LINMIN_INFO_CHOL_REGULARISED;
            // ---- predictor
            if (tid < Rp) { xs0[tid] = live ? -w : 0.0f; xs1[tid] = live ? 1.0f : 0.0f; }
            __syncthreads();
            solve_blocks<2>(Mb, NB, xs0, xs1, tid);
            float u = live ? xs0[tid] : 0.0f;
            const float v = live ? xs1[tid] : 0.0f;
            float su = u, sv = v, dummy2 = 0.0f;
            rd.sum3(su, sv, dummy2);
            float dnu = cons ? (su + rp) / sv : 0.0f;
            float da = u - v * dnu;
            float dl = -lam - di * da;
            float ap = (live && da < 0.0f) ? -a / da : INFINITY;
            float ad = (live && dl < 0.0f) ? -lam / dl : INFINITY;
            rd.min2(ap, ad);
            ap = fminf(1.0f, ap); ad = fminf(1.0f, ad);
            float mua = rd.sum(live ? (a + ap * da) * (lam + ad * dl) : 0.0f) / fR;
            float sg = mua / mu;
            sg = fminf(1.0f, fmaxf(0.0f, sg * sg * sg));
            // ---- corrector
            const float cc = sg * mu - da * dl;
            if (tid < Rp) xs0[tid] = live ? -w + cc / a : 0.0f;
            __syncthreads();
            solve_blocks<1>(Mb, NB, xs0, nullptr, tid);
            u = live ? xs0[tid] : 0.0f;
            su = rd.sum(u);
            dnu = cons ? (su + rp) / sv : 0.0f;
            da = u - v * dnu;
            dl = -lam + cc / a - di * da;
            ap = (live && da < 0.0f) ? -a / da : INFINITY;
            ad = (live && dl < 0.0f) ? -lam / dl : INFINITY;
            rd.min2(ap, ad);
            ap = fminf(1.0f, tau * ap); ad = fminf(1.0f, tau * ad);
            // G da = (r1 - dnu 1) - (lambda/a) o da row by row (M da = r1 - dnu 1, M = G + diag(lambda/a)), r1 = -w + cc/a
            if (live) {
                Ga = fmaf(ap, (-w + cc / a) - dnu - di * da, Ga);
                a = fmaxf(fmaf(ap, da, a), 1e-18f);
                lam = fmaxf(fmaf(ad, dl, lam), 1e-18f * lam0);
            }
            nu = fmaf(ad, dnu, nu);
        }
        // hand-over: zero where the primal-dual indicator says inactive (LINMIN_TAPIA_KAPPA, common.cuh)
        if (live) prm.coeffs[p * R + tid] = (a * sc > LINMIN_TAPIA_KAPPA * lam) ? a : 0.0f;
        if (prm.info && tid == 0) prm.info[p] = flags | (iters << 8);
    }
}

inline cudaError_t launch_ipls_c256(const LibView &lv, const SolveParams &prm, int sm_count, unsigned int *counter,
                                    cudaStream_t stream) {
    const size_t smem = c256::smem_floats(lv.L, lv.R) * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(ipls_c256_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>(prm.N, sm_count));
    ipls_c256_kernel<<<grid, c256::NT, smem, stream>>>(lv, prm, counter);
    return cudaGetLastError();
}
// fits in shared memory?  (R = 256, L <= 4096: 162 KB + vectors)
inline bool ipls_c256_fits(int L, int R) { return c256::smem_floats(L, R) * sizeof(float) + 64 <= 227 * 1024; }

}  // namespace linmin
