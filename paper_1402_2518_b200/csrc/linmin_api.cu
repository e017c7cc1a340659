// linmin_api.cu -- C ABI of liblinmin.so (see include/linmin.h for the contract).
// Host logic only: argument validation, the library handle, kernel launches, the host-buffer pipeline.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"
#include "finish.cuh"
#include "finish_fast.cuh"
#include "ipls_generic.cuh"
#include "ipls_q32.cuh"
#include "ipls_w64.cuh"
#include "ipls_c256.cuh"
#include "precompute.cuh"
#include "whiten.cuh"
#include "detect.cuh"

using namespace linmin;

namespace linmin {
// finish_sweep.cu (own translation unit, own register budget)
cudaError_t launch_finish_sweep_tu(const LibView &lv, const SolveParams &prm, int sm_count,
                                   unsigned int *counter, unsigned int *overflow, const unsigned int *list,
                                   unsigned int *defer, cudaStream_t stream);
inline bool finish_sweep_supported(int L, int R) { return R <= 32 && L <= 256; }
}  // namespace linmin

struct linmin_library {
    int L = 0, R = 0;                // the caller's sizes
    int Ri = 0;                      // endmembers the kernels see: R, or R + 1 with the slack endmember of slo
    int constraint = LINMIN_CONSTRAINT_SUM_TO_ONE, weighting = LINMIN_WEIGHTING_NONE;
    float *W = nullptr;              // weighting: L x L whitening matrix (fp32, lower triangular), Y' = Y W'
    double *Wd = nullptr, *Cd = nullptr;
    int device = 0;
    int sm_count = 0;
    cudaStream_t stream = nullptr;   // stream the handle was created on (frees are ordered on it)
    float *A = nullptr, *At = nullptr, *Ac = nullptr, *c = nullptr, *Gc = nullptr, *Gi = nullptr, *Giq = nullptr;
    linmin_library *pos_twin = nullptr;   // slo at R = 32: the same library under positivity only (launch_solve)
    float *Gpad = nullptr;           // more than 64 endmembers: Gc zero-padded to whole 32 x 32 blocks (ipls_c256.cuh)
    float *scal = nullptr;           // device scalars: gdmax, sum of Giq
    int *flags = nullptr;            // device word: bit 0 = non-finite library
    double *G64 = nullptr, *W64 = nullptr;
    // report fields and the last-use events are the only state a solve call writes; the handle is otherwise
    // immutable after creation (hence `const linmin_library *` in linmin_unmix_lib)
    mutable std::atomic<int> last_launches{0};
    bool timing = false;
    mutable std::atomic<bool> timed{false};
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    // last use per stream: linmin_library_destroy orders its frees after the work of EVERY stream the handle served
    static constexpr int MAX_USE = 16;
    mutable std::mutex use_mu;
    mutable cudaStream_t use_stream[MAX_USE] = {};
    mutable cudaEvent_t use_event[MAX_USE] = {};
    mutable int n_use = 0;
    mutable bool use_overflow = false;   // more streams than slots: destroy synchronises the device instead
};

namespace {

// Staging memory (per-call workspaces, the device buffers of linmin_unmix_host) comes from a memory pool the
// library owns, one per device, created on first use with an unbounded release threshold: a call finds the
// memory of the previous one instead of paying cudaMalloc / cudaFree again (30 ms of a 350 ms host-path step).
// linmin_trim_memory() hands it back.  The application's default pool is not touched.
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};

cudaMemPool_t staging_pool(int dev) {
    if (dev < 0 || dev >= 64) return nullptr;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    if (!g_pools[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { (void)cudaGetLastError(); return nullptr; }
        unsigned long long thr = ~0ull;
        (void)cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        g_pools[dev] = pool;
    }
    return g_pools[dev];
}

cudaError_t staging_alloc(void **p, size_t bytes, cudaStream_t stream) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    cudaMemPool_t pool = staging_pool(dev);
    if (pool) return cudaMallocFromPoolAsync(p, bytes, pool, stream);
    return cudaMallocAsync(p, bytes, stream);
}

int cuda_status(cudaError_t e) {
    if (e == cudaSuccess) return LINMIN_OK;
    if (e == cudaErrorMemoryAllocation) return LINMIN_ERR_OUT_OF_MEMORY;
    return LINMIN_ERR_CUDA;
}

#define CK(call)                                   \
    do {                                           \
        cudaError_t e__ = (call);                  \
        if (e__ != cudaSuccess) {                  \
            (void)cudaGetLastError();              \
            return cuda_status(e__);               \
        }                                          \
    } while (0)

struct Resolved {
    cudaStream_t stream;
    int constraint, weighting;
    const float *cov;
    int64_t ldY, sstride;
    int max_iter;
    float gap_tol, feas_tol;
    int32_t *info;
};

int resolve_opts(const linmin_opts *o, int L, Resolved *r) {
    r->stream = nullptr; r->ldY = L; r->sstride = 0; r->max_iter = 50;
    r->gap_tol = 1e-7f; r->feas_tol = 3e-5f; r->info = nullptr;   // measured optimum of IPLS + finish time
    r->constraint = LINMIN_CONSTRAINT_SUM_TO_ONE; r->weighting = LINMIN_WEIGHTING_NONE; r->cov = nullptr;
    if (!o) return LINMIN_OK;
    if (o->struct_size != sizeof(linmin_opts)) return LINMIN_ERR_INVALID_ARGUMENT;
    if (o->constraint < LINMIN_CONSTRAINT_SUM_TO_ONE || o->constraint > LINMIN_CONSTRAINT_POSITIVITY_ONLY)
        return LINMIN_ERR_INVALID_ARGUMENT;
    if (o->weighting < LINMIN_WEIGHTING_NONE || o->weighting > LINMIN_WEIGHTING_SHARED_DIAGONAL)
        return LINMIN_ERR_INVALID_ARGUMENT;
    r->constraint = o->constraint; r->weighting = o->weighting; r->cov = o->cov;
    r->stream = (cudaStream_t)o->stream;
    if (o->ldY != 0) { if (o->ldY < L) return LINMIN_ERR_INVALID_ARGUMENT; r->ldY = o->ldY; }
    if (o->sigma_pixel_stride != 0) {
        if (o->sigma_pixel_stride < L) return LINMIN_ERR_INVALID_ARGUMENT;
        r->sstride = o->sigma_pixel_stride;
    }
    if (o->max_iter < 0 || o->max_iter > 255) return LINMIN_ERR_INVALID_ARGUMENT;
    if (o->max_iter > 0) r->max_iter = o->max_iter;
    if (o->gap_tol < 0.0f || o->feas_tol < 0.0f || std::isnan(o->gap_tol) || std::isnan(o->feas_tol))
        return LINMIN_ERR_INVALID_ARGUMENT;
    if (o->gap_tol > 0.0f) r->gap_tol = o->gap_tol;
    if (o->feas_tol > 0.0f) r->feas_tol = o->feas_tol;
    r->info = o->info_out;
    return LINMIN_OK;
}

int check_sizes(int64_t N, int L, int R) {
    if (N < 0 || L < 1 || R < 1) return LINMIN_ERR_INVALID_ARGUMENT;
    if (R > LINMIN_MAX_R || L > LINMIN_MAX_L) return LINMIN_ERR_UNSUPPORTED_SIZE;
    if (N >= ((int64_t)1 << 32)) return LINMIN_ERR_UNSUPPORTED_SIZE;   // pixel lists and work tickets are 32-bit
    return LINMIN_OK;
}

LibView view_of(const linmin_library *lib) {
    LibView v;
    v.cons = lib->constraint != LINMIN_CONSTRAINT_POSITIVITY_ONLY;
    v.L = lib->L; v.R = lib->Ri; v.A = lib->A; v.At = lib->At; v.Ac = lib->Ac; v.c = lib->c; v.Gc = lib->Gc;
    v.G64 = lib->G64; v.scal = lib->scal; v.flags = lib->flags; v.Gi = lib->Gi; v.Giq = lib->Giq;
    v.Gpad = lib->Gpad;
    return v;
}

// persistent grid: enough CTAs to fill every SM at the kernel's occupancy, never more than needed
template <typename K>
int persistent_grid(K kernel, int block, size_t smem, int sm_count, int64_t work_items, int items_per_cta) {
    int occ = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, block, smem) != cudaSuccess || occ < 1) {
        (void)cudaGetLastError();
        occ = 1;
    }
    int64_t need = (work_items + items_per_cta - 1) / items_per_cta;
    int64_t cap = (int64_t)sm_count * occ;
    return (int)std::max<int64_t>(1, std::min(need, cap));
}

// Records "the handle was last used on `stream` now" (one event per stream the handle has served); skipped while
// the stream is being captured into a CUDA graph (the graph's owner then keeps the handle alive, include/linmin.h).
void note_use(const linmin_library *lib, cudaStream_t stream) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cs) != cudaSuccess) { (void)cudaGetLastError(); return; }
    if (cs != cudaStreamCaptureStatusNone) return;
    if (stream == lib->stream) return;            // frees are enqueued on that stream anyway
    std::lock_guard<std::mutex> lk(lib->use_mu);
    int slot = -1;
    for (int i = 0; i < lib->n_use; ++i) if (lib->use_stream[i] == stream) slot = i;
    if (slot < 0) {
        if (lib->n_use == linmin_library::MAX_USE) { lib->use_overflow = true; return; }
        cudaEvent_t e = nullptr;
        if (cudaEventCreateWithFlags(&e, cudaEventDisableTiming) != cudaSuccess) { (void)cudaGetLastError(); lib->use_overflow = true; return; }
        slot = lib->n_use++;
        lib->use_stream[slot] = stream; lib->use_event[slot] = e;
    }
    if (cudaEventRecord(lib->use_event[slot], stream) != cudaSuccess) { (void)cudaGetLastError(); lib->use_overflow = true; }
}

// prewhitened: Y is already Y W' (the caller did the renormalisation of this handle's covariance)
int solve_core(const linmin_library *lib, const float *Y, const float *sigma, int64_t N,
               const Resolved &o, float *coeffs, float *csig, float *resid, bool prewhitened,
               bool record_start = true) {
    const int L = lib->L, R = lib->Ri;      // R: the endmembers the kernels see (slack included)
    const bool cons = lib->constraint != LINMIN_CONSTRAINT_POSITIVITY_ONLY;
    LibView lv = view_of(lib);
    struct FreeV { void *p; cudaStream_t s; ~FreeV() { if (p) cudaFreeAsync(p, s); } };
    int launches = 0;
    if (lib->timing && record_start) CK(cudaEventRecord(lib->ev[0], o.stream));
    int64_t ldY = o.ldY, sstride = o.sstride;
    // ---- renormalised problem (eq. 6): Y' = Y W' into a workspace, then the unweighted path on
    //      (A', Y') with unit noise
    float *Yw = nullptr;
    if (lib->weighting != LINMIN_WEIGHTING_NONE && !prewhitened) {
        CK(staging_alloc((void **)&Yw, (size_t)N * L * sizeof(float), o.stream));
        CK(launch_whiten_spectra(Y, o.ldY, N, L, lib->W, lib->weighting == LINMIN_WEIGHTING_SHARED_DIAGONAL, Yw,
                                 lib->sm_count, o.stream));
        ++launches;
        Y = Yw; ldY = L; sigma = nullptr; sstride = 0;
    }
    FreeV free_yw{Yw, o.stream};
    // ---- slo: the kernels work on R + 1 endmembers; their outputs go to internal arrays, the slack is stripped
    float *ci = nullptr, *si = nullptr;
    float *coeffs_user = coeffs, *csig_user = csig;
    if (R != lib->R) {
        CK(staging_alloc((void **)&ci, (size_t)N * R * sizeof(float), o.stream));
        if (csig) CK(staging_alloc((void **)&si, (size_t)N * R * sizeof(float), o.stream));
        coeffs = ci; csig = csig ? si : nullptr;
    }
    FreeV free_ci{ci, o.stream}, free_si{si, o.stream};
    SolveParams prm;
    prm.Y = Y; prm.sigma = sigma; prm.N = N; prm.ldY = ldY; prm.sigma_stride = sstride;
    prm.has_sigma = sigma != nullptr;
    prm.max_iter = o.max_iter; prm.gap_tol = o.gap_tol; prm.feas_tol = o.feas_tol;
    prm.coeffs = coeffs; prm.coeff_sigma = csig; prm.resid = resid; prm.info = o.info;
    // pos: the library is not centred, so the projections b = A'y that set the stopping scale are two orders of magnitude
    // above the gradients that decide the support; with the sto thresholds IPLS handed over supports that needed 1.9
    // repairs per pixel in the finish (0.24 with these; config-4 data: finish 36 -> 11 ms per 2^20 pixels, IPLS 6.2 -> 7.6)
    if (!cons) { prm.gap_tol *= 0.01f; prm.feas_tol *= 0.01f; }

    // ---- K1: projection + IPLS
    // per-call workspace, because one handle may serve several streams: the work counters of the persistent
    // kernels (8 words), then two pixel lists of finish_sweep (count + one entry per pixel each): the overflow
    // list (supports above 16) and the repair list (pixels whose support changes after the first round)
    const bool use_f8 = finish_sweep_supported(L, R);
    const bool use_ff64 = !use_f8 && R > 32 && finish_fast_fits(L, R);      // 33..64 endmembers: finish_fast + its overflow list
    unsigned int *ws = nullptr;
    const size_t ws_words = 8 + (use_f8 ? 2 * ((size_t)N + 1) : (use_ff64 ? (size_t)N + 1 : 0));
    CK(staging_alloc((void **)&ws, ws_words * sizeof(unsigned int), o.stream));
    struct Free { unsigned int *p; cudaStream_t s; ~Free() { cudaFreeAsync(p, s); } } free_ws{ws, o.stream};
    CK(cudaMemsetAsync(ws, 0, std::min<size_t>(9, ws_words) * sizeof(unsigned int), o.stream));
    unsigned int *counters = ws, *overflow = ws + 8, *repair = ws + 8 + ((size_t)N + 1);
    if (use_f8) CK(cudaMemsetAsync(repair, 0, sizeof(unsigned int), o.stream));
    // K1 hands its iterate over with 16-byte stores: a coeffs_out that is only 4-byte aligned (a sub-view of a larger
    // buffer) takes the any-size IPLS kernel instead (scalar stores; same minimiser, the finish is exact either way)
    const bool coeffs16 = (reinterpret_cast<uintptr_t>(coeffs) & 15) == 0;
    if (R == 32 && start_r32_warps(L) > 0 && coeffs16) {
        // K0 (projection + start point, one record per pixel) and K1 (the iteration), in chunks of 2^21 pixels
        // so that the record workspace stays at 0.8 GB whatever N is
        const int64_t chunk = (int64_t)1 << 21;
        const int nchunks = (int)((N + chunk - 1) / chunk);
        float *recbuf = nullptr;
        unsigned int *tickets = nullptr;
        CK(staging_alloc((void **)&recbuf, (size_t)std::min(N, chunk) * s32::REC * sizeof(float), o.stream));
        struct FreeF { void *p; cudaStream_t s; ~FreeF() { cudaFreeAsync(p, s); } } free_rec{recbuf, o.stream};
        CK(staging_alloc((void **)&tickets, (size_t)nchunks * sizeof(unsigned int), o.stream));
        FreeF free_tk{tickets, o.stream};
        CK(cudaMemsetAsync(tickets, 0, (size_t)nchunks * sizeof(unsigned int), o.stream));
        for (int c = 0; c < nchunks; ++c) {
            const int64_t pb = (int64_t)c * chunk, pe = std::min(N, pb + chunk);
            CK(launch_start_r32(lv, prm, pb, pe, recbuf, lib->sm_count, o.stream));
            CK(launch_ipls_q32(lv, prm, pb, pe, recbuf, lib->sm_count, tickets + c, o.stream));
            launches += 2;
        }
    } else if (R > 32 && R <= 64 && ipls_w64_warps(L) > 0) {
        // 33..64 endmembers (CRISM-like config, the paper's 36 / 37 / 44 spectra): one warp per pixel, matrix in registers
        CK(launch_ipls_w64(lv, prm, lib->sm_count, counters, o.stream));
        ++launches;
    } else if (R <= 64) {
        const int teams = 8, block = teams * 32;
        size_t smem = teams * ipls_warp_team_floats(L, R) * sizeof(float);
        CK(cudaFuncSetAttribute(ipls_generic_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int grid = persistent_grid(ipls_generic_kernel<32>, block, smem, lib->sm_count, N, teams);
        ipls_generic_kernel<32><<<grid, block, smem, o.stream>>>(lv, prm);
        CK(cudaGetLastError());
        ++launches;
    } else if (R <= 256 && lib->Gpad && ipls_c256_fits(L, R)) {
        // 65..256 endmembers: one CTA per pixel, blocked Cholesky with the block products on the tensor cores
        CK(launch_ipls_c256(lv, prm, lib->sm_count, counters, o.stream));
        ++launches;
    } else {
        const int block = 256;
        size_t smem = ipls_generic_team_floats(L, R) * sizeof(float);
        CK(cudaFuncSetAttribute(ipls_generic_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int grid = persistent_grid(ipls_generic_kernel<256>, block, smem, lib->sm_count, N, 1);
        ipls_generic_kernel<256><<<grid, block, smem, o.stream>>>(lv, prm);
        CK(cudaGetLastError());
        ++launches;
    }
    if (lib->timing) CK(cudaEventRecord(lib->ev[1], o.stream));
    // ---- K2: exact finish + uncertainty + residual
    auto launch_finish_any = [&](const unsigned int *list) -> int {      // one warp per pixel, any size, any constraint
        const int KMAX = R <= 32 ? R : 64;
        size_t per_warp = (finish_warp_bytes(L, R, KMAX) + 15) & ~(size_t)15;
        int warps = (int)std::min<size_t>(8, (200 * 1024) / per_warp);
        if (warps < 1) return LINMIN_ERR_UNSUPPORTED_SIZE;
        size_t smem = per_warp * warps;
        CK(cudaFuncSetAttribute(finish_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int grid = persistent_grid(finish_kernel, warps * 32, smem, lib->sm_count, N, warps);
        finish_kernel<<<grid, warps * 32, smem, o.stream>>>(lv, prm, KMAX, list);
        CK(cudaGetLastError());
        ++launches;
        return LINMIN_OK;
    };
    if (use_f8) {
        // first round for every pixel (91 % end there), then the others, packed, to their end: a warp's four
        // pixels share every round, so a repair in the main pass would stall the three that are done
        CK(launch_finish_sweep_tu(lv, prm, lib->sm_count, counters + 1, overflow, nullptr, repair, o.stream));
        ++launches;
        CK(launch_finish_sweep_tu(lv, prm, lib->sm_count, counters + 3, overflow, repair, nullptr, o.stream));
        ++launches;
        // pixels whose support outgrew finish_sweep (0.1 % on config 4): one-warp-per-pixel kernels
        CK(launch_finish_fast(lv, prm, lib->sm_count, counters + 2, overflow, nullptr, o.stream));
        ++launches;
    } else if (use_ff64) {
        // one warp per pixel, two endmembers per lane, supports up to 32; wider ones go on to the any-size kernel
        CK(launch_finish_fast(lv, prm, lib->sm_count, counters + 2, nullptr, overflow, o.stream));
        ++launches;
        const int rc = launch_finish_any(overflow);
        if (rc != LINMIN_OK) return rc;
    } else if (R <= 32 && finish_fast_fits(L, R)) {
        CK(launch_finish_fast(lv, prm, lib->sm_count, counters + 2, nullptr, nullptr, o.stream));
        ++launches;
    } else {
        const int rc = launch_finish_any(nullptr);
        if (rc != LINMIN_OK) return rc;
    }
    if (R != lib->R) {
        const int grid = (int)std::min<int64_t>((N * lib->R + 255) / 256, (int64_t)lib->sm_count * 16);
        strip_slack_kernel<<<grid, 256, 0, o.stream>>>(ci, si, N, lib->R, R, coeffs_user, csig_user, o.info);
        CK(cudaGetLastError());
        ++launches;
    }
    if (lib->timing) { CK(cudaEventRecord(lib->ev[2], o.stream)); lib->timed.store(true); }
    lib->last_launches.store(launches);
    note_use(lib, o.stream);
    return LINMIN_OK;
}

// The solve of a handle.  slo at R = 32 has no slack endmember: two passes over the fast kernels, pos into a workspace
// and sto into the caller's arrays, then the per-pixel choice (slo_select_kernel).
int launch_solve(const linmin_library *lib, const float *Y, const float *sigma, int64_t N,
                 const Resolved &o, float *coeffs, float *csig, float *resid) {
    if (!lib->pos_twin) return solve_core(lib, Y, sigma, N, o, coeffs, csig, resid, false);
    const int L = lib->L, R = lib->R;
    struct FreeV { void *p; cudaStream_t s; ~FreeV() { if (p) cudaFreeAsync(p, s); } };
    Resolved oc = o;
    float *Yw = nullptr;
    int extra = 0;
    // timing report: the call starts here and ends after the selection; the first interval then holds the whitening,
    // the whole pos pass and the IPLS kernels of the sto pass, the second the sto finish and the selection
    if (lib->timing) CK(cudaEventRecord(lib->ev[0], o.stream));
    if (lib->weighting != LINMIN_WEIGHTING_NONE) {
        CK(staging_alloc((void **)&Yw, (size_t)N * L * sizeof(float), o.stream));
        CK(launch_whiten_spectra(Y, o.ldY, N, L, lib->W, lib->weighting == LINMIN_WEIGHTING_SHARED_DIAGONAL, Yw,
                                 lib->sm_count, o.stream));
        ++extra;
        Y = Yw; sigma = nullptr; oc.ldY = L; oc.sstride = 0;
    }
    FreeV free_yw{Yw, o.stream};
    float *cp = nullptr, *sp = nullptr, *rp = nullptr;
    int32_t *ip = nullptr;
    CK(staging_alloc((void **)&cp, (size_t)N * R * sizeof(float), o.stream));
    FreeV f0{cp, o.stream};
    if (csig) CK(staging_alloc((void **)&sp, (size_t)N * R * sizeof(float), o.stream));
    FreeV f1{sp, o.stream};
    if (resid) CK(staging_alloc((void **)&rp, (size_t)N * sizeof(float), o.stream));
    FreeV f2{rp, o.stream};
    if (o.info) CK(staging_alloc((void **)&ip, (size_t)N * sizeof(int32_t), o.stream));
    FreeV f3{ip, o.stream};
    Resolved op = oc;
    op.info = ip;
    int rc = solve_core(lib->pos_twin, Y, sigma, N, op, cp, sp, rp, true);
    if (rc != LINMIN_OK) return rc;
    rc = solve_core(lib, Y, sigma, N, oc, coeffs, csig, resid, true, false);
    if (rc != LINMIN_OK) return rc;
    const int grid = (int)std::min<int64_t>((N + 7) / 8, (int64_t)lib->sm_count * 16);
    slo_select_kernel<<<grid, 256, 0, o.stream>>>(N, R, cp, sp, rp, ip, coeffs, csig, resid, o.info);
    CK(cudaGetLastError());
    if (lib->timing) CK(cudaEventRecord(lib->ev[2], o.stream));
    lib->last_launches.store(lib->last_launches.load() + lib->pos_twin->last_launches.load() + extra + 1);
    return LINMIN_OK;
}

// Once-per-library precompute, all of it on the device and enqueued on `stream`: copy of A,
// centred library, transposed copy, Gram matrices, start-point data.  No host round trip; `wait_check` adds the
// ONE synchronisation linmin_library_create documents (to return LINMIN_ERR_LIBRARY_NONFINITE).
int library_create_impl(const float *A, int L, int R, cudaStream_t stream, bool on_host, bool wait_check,
                        int constraint, int weighting, const float *cov, linmin_library **out) {
    *out = nullptr;
    if (weighting != LINMIN_WEIGHTING_NONE && !cov) return LINMIN_ERR_INVALID_ARGUMENT;
    // slo: a slack endmember (sto on [A | 0]) -- except at R = 32, where the fast kernels exist for exactly
    // 32 endmembers: there slo is the pos solution where its sum stays below one and the sto solution elsewhere
    const bool twin = constraint == LINMIN_CONSTRAINT_SUM_LOWER_THAN_ONE && R == 32 && start_r32_warps(L) > 0 &&
                      finish_sweep_supported(L, R);
    const int Ri = (constraint == LINMIN_CONSTRAINT_SUM_LOWER_THAN_ONE && !twin) ? R + 1 : R;
    if (Ri > LINMIN_MAX_R) return LINMIN_ERR_UNSUPPORTED_SIZE;
    const bool cons = constraint != LINMIN_CONSTRAINT_POSITIVITY_ONLY;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    linmin_library *lib = new (std::nothrow) linmin_library();
    if (!lib) return LINMIN_ERR_OUT_OF_MEMORY;
    lib->L = L; lib->R = R; lib->Ri = Ri; lib->constraint = constraint; lib->weighting = weighting;
    lib->device = dev; lib->stream = stream;
    float *Araw = nullptr, *covd = nullptr;       // device copies of the caller's arrays (released below)
    auto fail = [&](int code) {
        if (Araw) cudaFreeAsync(Araw, stream);
        if (covd) cudaFreeAsync(covd, stream);
        linmin_library_destroy(lib);
        return code;
    };
#define CKF(call)                                                 \
    do {                                                          \
        cudaError_t e__ = (call);                                 \
        if (e__ != cudaSuccess) { (void)cudaGetLastError(); return fail(cuda_status(e__)); } \
    } while (0)
    CKF(cudaDeviceGetAttribute(&lib->sm_count, cudaDevAttrMultiProcessorCount, dev));
    const size_t LR = (size_t)L * Ri, RR = (size_t)Ri * Ri, LL = (size_t)L * L;
    CKF(cudaMallocAsync((void **)&lib->A, LR * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->At, LR * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->Ac, LR * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->c, (size_t)L * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->Gc, RR * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->Gi, RR * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->Giq, (size_t)Ri * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->scal, 4 * sizeof(float), stream));
    CKF(cudaMallocAsync((void **)&lib->G64, RR * sizeof(double), stream));
    CKF(cudaMallocAsync((void **)&lib->W64, RR * sizeof(double), stream));
    CKF(cudaMallocAsync((void **)&lib->flags, sizeof(int), stream));
    CKF(cudaMemsetAsync(lib->flags, 0, sizeof(int), stream));
    CKF(cudaMallocAsync((void **)&Araw, (size_t)L * R * sizeof(float), stream));
    CKF(cudaMemcpyAsync(Araw, A, (size_t)L * R * sizeof(float), on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, stream));
    if (weighting != LINMIN_WEIGHTING_NONE) {
        // renormalised problem: C = Rc Rc', W = Rc^-1, A' = W A
        const size_t ncov = (weighting == LINMIN_WEIGHTING_SHARED_DIAGONAL) ? (size_t)L : LL;
        CKF(cudaMallocAsync((void **)&covd, ncov * sizeof(float), stream));
        CKF(cudaMemcpyAsync(covd, cov, ncov * sizeof(float), on_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, stream));
        CKF(cudaMallocAsync((void **)&lib->W, LL * sizeof(float), stream));
        CKF(cudaMallocAsync((void **)&lib->Wd, LL * sizeof(double), stream));
        CKF(cudaMallocAsync((void **)&lib->Cd, LL * sizeof(double), stream));
        whitening_matrix_kernel<<<1, 1024, 0, stream>>>(covd, weighting == LINMIN_WEIGHTING_SHARED_DIAGONAL ? 1 : 2, L,
                                                        lib->Cd, lib->Wd, lib->W, lib->flags);
        CKF(cudaGetLastError());
    }
    {
        int block = 256;
        // the library the kernels see: whitened, with the slack endmember of slo as a last, all-zero column
        whiten_library_kernel<<<(int)((LR + block - 1) / block), block, 0, stream>>>(Araw, L, R, Ri, lib->Wd, lib->A);
        CKF(cudaGetLastError());
        int grid = (L * 32 + block - 1) / block;
        // pos: no centring (it is only valid under sum a = 1) and no shift of the fp64 Gram matrix
        center_library_kernel<<<grid, block, 0, stream>>>(lib->A, Araw, L, Ri, R, cons ? 1 : 0, lib->Ac, lib->c, lib->flags);
        CKF(cudaGetLastError());
        transpose_library_kernel<<<(int)((LR + block - 1) / block), block, 0, stream>>>(lib->A, L, Ri, lib->At);
        CKF(cudaGetLastError());
        grid = (int)((RR + block - 1) / block);
        gram_kernel<<<grid, block, 0, stream>>>(lib->A, lib->Ac, L, Ri, lib->G64, lib->Gc);
        CKF(cudaGetLastError());
        // start point data of IPLS: inverse of the regularised centred Gram matrix, its row sums, gdmax
        start_data_kernel<<<1, 1024, 0, stream>>>(lib->Gc, Ri, lib->W64, lib->Gi, lib->Giq, lib->scal, lib->G64, cons ? 1 : 0);
        CKF(cudaGetLastError());
        if (Ri > 64) {
            const int Rp = 32 * c256::nblocks(Ri);
            CKF(cudaMallocAsync((void **)&lib->Gpad, (size_t)Rp * Rp * sizeof(float), stream));
            pad_gram_kernel<<<(Rp * Rp + block - 1) / block, block, 0, stream>>>(lib->Gc, Ri, Rp, lib->Gpad);
            CKF(cudaGetLastError());
        }
    }
    cudaFreeAsync(Araw, stream); Araw = nullptr;
    if (covd) { cudaFreeAsync(covd, stream); covd = nullptr; }
    if (twin) {     // (same A, same covariance: its non-finite / covariance flags are this handle's)
        const int rc = library_create_impl(A, L, R, stream, on_host, false, LINMIN_CONSTRAINT_POSITIVITY_ONLY, weighting, cov,
                                           &lib->pos_twin);
        if (rc < 0) return fail(rc);
    }
    if (wait_check) {
        int hflags = 0;
        CKF(cudaMemcpyAsync(&hflags, lib->flags, sizeof(int), cudaMemcpyDeviceToHost, stream));
        CKF(cudaStreamSynchronize(stream));
        if (hflags & 1) return fail(LINMIN_ERR_LIBRARY_NONFINITE);
        if (hflags & 2) return fail(LINMIN_ERR_COVARIANCE);
    }
    *out = lib;
    return (Ri > L) ? LINMIN_WARN_RANK_DEFICIENT : LINMIN_OK;
#undef CKF
}

}  // namespace

extern "C" {

int linmin_version(void) { return LINMIN_VERSION; }

int linmin_trim_memory(void) {
    std::lock_guard<std::mutex> lk(g_pool_mu);
    for (cudaMemPool_t pool : g_pools)
        if (pool && cudaMemPoolTrimTo(pool, 0) != cudaSuccess) { (void)cudaGetLastError(); return LINMIN_ERR_CUDA; }
    return LINMIN_OK;
}

const char *linmin_strerror(int code) {
    switch (code) {
        case LINMIN_OK: return "ok";
        case LINMIN_ERR_INVALID_ARGUMENT: return "invalid argument";
        case LINMIN_ERR_UNSUPPORTED_SIZE: return "unsupported size (R > 256 or L > 512)";
        case LINMIN_ERR_NOT_IMPLEMENTED: return "option not implemented (unused: every option of linmin.h is built)";
        case LINMIN_ERR_CUDA: return "CUDA runtime error (no device, or a failed call)";
        case LINMIN_ERR_OUT_OF_MEMORY: return "out of device memory";
        case LINMIN_ERR_LIBRARY_NONFINITE: return "library A contains a non-finite value";
        case LINMIN_ERR_COVARIANCE: return "noise covariance is not finite or not positive definite";
        case LINMIN_ERR_STATIC_SCRATCH: return "more than 64 endmembers: beyond the fixed scratch array of linmin_detection_thresholds_static";
        case LINMIN_WARN_RANK_DEFICIENT: return "warning: R > L, the minimiser may be non-unique";
        default: return "unknown status code";
    }
}

int linmin_library_create(const float *A, int32_t L, int32_t R, const linmin_opts *opts, linmin_library **lib) {
    if (!lib) return LINMIN_ERR_INVALID_ARGUMENT;
    *lib = nullptr;
    if (!A) return LINMIN_ERR_INVALID_ARGUMENT;
    int rc = check_sizes(0, L, R);
    if (rc != LINMIN_OK) return rc;
    Resolved o;
    rc = resolve_opts(opts, L, &o);
    if (rc != LINMIN_OK) return rc;
    return library_create_impl(A, L, R, o.stream, false, true, o.constraint, o.weighting, o.cov, lib);
}

void linmin_library_destroy(linmin_library *lib) {
    if (!lib) return;
    cudaStream_t s = lib->stream;
    {   // the frees below are ordered on the creation stream: make it wait for the last work of every other stream
        std::lock_guard<std::mutex> lk(lib->use_mu);
        if (lib->use_overflow) cudaDeviceSynchronize();
        for (int i = 0; i < lib->n_use; ++i) {
            cudaStreamWaitEvent(s, lib->use_event[i], 0);
            cudaEventDestroy(lib->use_event[i]);
        }
        lib->n_use = 0;
    }
    if (lib->pos_twin) linmin_library_destroy(lib->pos_twin);      // (its frees go to the same stream, after the waits above)
    void *bufs[] = {lib->A, lib->At, lib->Ac, lib->c, lib->Gc, lib->Gi, lib->Giq, lib->scal, lib->G64, lib->W64, lib->flags,
                    lib->W, lib->Wd, lib->Cd, lib->Gpad};
    for (void *q : bufs) if (q) cudaFreeAsync(q, s);
    for (int i = 0; i < 3; ++i) if (lib->ev[i]) cudaEventDestroy(lib->ev[i]);
    (void)cudaGetLastError();
    delete lib;
}

int linmin_library_last_launches(const linmin_library *lib) { return lib ? lib->last_launches.load() : 0; }

int linmin_library_enable_timing(linmin_library *lib, int enable) {
    if (!lib) return LINMIN_ERR_INVALID_ARGUMENT;
    if (enable && !lib->ev[0])
        for (int i = 0; i < 3; ++i) CK(cudaEventCreate(&lib->ev[i]));
    lib->timing = enable != 0;
    lib->timed.store(false);
    return LINMIN_OK;
}

int linmin_library_last_timing(const linmin_library *lib, float *ipls_ms, float *finish_ms) {
    if (!lib || !lib->timing || !lib->timed.load()) return LINMIN_ERR_INVALID_ARGUMENT;
    CK(cudaEventSynchronize(lib->ev[2]));
    float a = 0.0f, b = 0.0f;
    CK(cudaEventElapsedTime(&a, lib->ev[0], lib->ev[1]));
    CK(cudaEventElapsedTime(&b, lib->ev[1], lib->ev[2]));
    if (ipls_ms) *ipls_ms = a;
    if (finish_ms) *finish_ms = b;
    return LINMIN_OK;
}

int linmin_unmix_lib(const linmin_library *lib, const float *Y, const float *sigma, int64_t N,
                     const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out, float *resid_out) {
    if (!lib) return LINMIN_ERR_INVALID_ARGUMENT;
    if (N < 0) return LINMIN_ERR_INVALID_ARGUMENT;
    Resolved o;
    int rc = resolve_opts(opts, lib->L, &o);
    if (rc != LINMIN_OK) return rc;
    // constraint and weighting are properties of the handle: opts must agree with it (or be NULL)
    if (opts && (o.constraint != lib->constraint || o.weighting != lib->weighting)) return LINMIN_ERR_INVALID_ARGUMENT;
    if (N >= ((int64_t)1 << 32)) return LINMIN_ERR_UNSUPPORTED_SIZE;
    if (N == 0) { lib->last_launches.store(0); return LINMIN_OK; }
    if (!Y || !coeffs_out) return LINMIN_ERR_INVALID_ARGUMENT;
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev != lib->device) return LINMIN_ERR_INVALID_ARGUMENT;     // the handle's memory lives on another device
    return launch_solve(lib, Y, sigma, N, o, coeffs_out, coeff_sigma_out, resid_out);
}

int linmin_unmix(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L, int32_t R,
                 const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out, float *resid_out) {
    int rc = check_sizes(N, L, R);
    if (rc != LINMIN_OK) return rc;
    if (!A) return LINMIN_ERR_INVALID_ARGUMENT;
    Resolved o;
    rc = resolve_opts(opts, L, &o);
    if (rc != LINMIN_OK) return rc;
    if (N > 0 && (!Y || !coeffs_out)) return LINMIN_ERR_INVALID_ARGUMENT;
    linmin_library *lib = nullptr;
    // everything is enqueued on the caller's stream and the call returns: no synchronisation, no host arithmetic.
    // A non-finite library can therefore not be reported through the status: the solve kernels return at once on
    // the device flag and the outputs are poisoned instead (NaN, LINMIN_INFO_LIBRARY_NONFINITE).
    int wrc = library_create_impl(A, L, R, o.stream, false, false, o.constraint, o.weighting, o.cov, &lib);
    if (wrc < 0) return wrc;
    rc = LINMIN_OK;
    if (N > 0) {
        rc = launch_solve(lib, Y, sigma, N, o, coeffs_out, coeff_sigma_out, resid_out);
        if (rc == LINMIN_OK) {
            const int grid = (int)std::min<int64_t>((N * R + 255) / 256, (int64_t)lib->sm_count * 8);
            poison_outputs_kernel<<<grid, 256, 0, o.stream>>>(lib->flags, N, R, coeffs_out, coeff_sigma_out, resid_out, o.info);
            if (cudaGetLastError() != cudaSuccess) rc = LINMIN_ERR_CUDA;
        }
    }
    linmin_library_destroy(lib);   // stream-ordered frees: safe while the kernels are still queued
    return rc != LINMIN_OK ? rc : wrc;
}

int linmin_unmix_host(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L, int32_t R,
                      const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out, float *resid_out) {
    int rc = check_sizes(N, L, R);
    if (rc != LINMIN_OK) return rc;
    if (!A) return LINMIN_ERR_INVALID_ARGUMENT;
    Resolved o;
    rc = resolve_opts(opts, L, &o);
    if (rc != LINMIN_OK) return rc;
    if (N > 0 && (!Y || !coeffs_out)) return LINMIN_ERR_INVALID_ARGUMENT;

    const int NBUF = 3;
    cudaStream_t st[NBUF] = {nullptr, nullptr, nullptr};
    float *dY[NBUF] = {}, *dS[NBUF] = {}, *dC[NBUF] = {}, *dCS[NBUF] = {}, *dR[NBUF] = {};
    int32_t *dI[NBUF] = {};
    float *dSshared = nullptr;
    linmin_library *lib = nullptr;
    int wrc = LINMIN_OK;
    int64_t chunk = std::min<int64_t>(N, (int64_t)1 << 18);   // 2^16: 334 ms, 2^18: 330 ms, 2^20: 358 ms per config-4 step
    auto cleanup = [&]() {
        for (int b = 0; b < NBUF; ++b) {
            if (st[b]) {
                float *bufs[5] = {dY[b], dS[b], dC[b], dCS[b], dR[b]};
                for (float *q : bufs) if (q) cudaFreeAsync(q, st[b]);
                if (dI[b]) cudaFreeAsync(dI[b], st[b]);
                cudaStreamSynchronize(st[b]);
                cudaStreamDestroy(st[b]);
            }
        }
        if (dSshared) cudaFree(dSshared);
        if (lib) { cudaStreamSynchronize(lib->stream); linmin_library_destroy(lib); }
        (void)cudaGetLastError();
    };
#define CKH(call)                                                                   \
    do {                                                                            \
        cudaError_t e__ = (call);                                                   \
        if (e__ != cudaSuccess) { (void)cudaGetLastError(); cleanup(); return cuda_status(e__); } \
    } while (0)
    wrc = library_create_impl(A, L, R, nullptr, true, true, o.constraint, o.weighting, o.cov, &lib);
    if (wrc < 0) { lib = nullptr; return wrc; }
    if (N == 0) { cleanup(); return wrc; }
    const bool per_pixel_sigma = sigma && o.sstride != 0;
    if (sigma && !per_pixel_sigma) {
        CKH(cudaMalloc((void **)&dSshared, (size_t)L * sizeof(float)));
        CKH(cudaMemcpy(dSshared, sigma, (size_t)L * sizeof(float), cudaMemcpyHostToDevice));
    }
    for (int b = 0; b < NBUF; ++b) {
        CKH(cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking));
        CKH(staging_alloc((void **)&dY[b], (size_t)chunk * L * sizeof(float), st[b]));
        if (per_pixel_sigma) CKH(staging_alloc((void **)&dS[b], (size_t)chunk * L * sizeof(float), st[b]));
        CKH(staging_alloc((void **)&dC[b], (size_t)chunk * R * sizeof(float), st[b]));
        if (coeff_sigma_out) CKH(staging_alloc((void **)&dCS[b], (size_t)chunk * R * sizeof(float), st[b]));
        if (resid_out) CKH(staging_alloc((void **)&dR[b], (size_t)chunk * sizeof(float), st[b]));
        if (o.info) CKH(staging_alloc((void **)&dI[b], (size_t)chunk * sizeof(int32_t), st[b]));
    }
    int bi = 0;
    for (int64_t p0 = 0; p0 < N; p0 += chunk, bi = (bi + 1) % NBUF) {
        int64_t n = std::min(chunk, N - p0);
        cudaStream_t s = st[bi];
        // stream order makes reuse of buffer set `bi` safe: its previous D2H copies precede these H2D
        CKH(cudaMemcpy2DAsync(dY[bi], (size_t)L * sizeof(float), Y + p0 * o.ldY, (size_t)o.ldY * sizeof(float),
                              (size_t)L * sizeof(float), (size_t)n, cudaMemcpyHostToDevice, s));
        if (per_pixel_sigma)
            CKH(cudaMemcpy2DAsync(dS[bi], (size_t)L * sizeof(float), sigma + p0 * o.sstride,
                                  (size_t)o.sstride * sizeof(float), (size_t)L * sizeof(float), (size_t)n,
                                  cudaMemcpyHostToDevice, s));
        Resolved oc = o;
        oc.stream = s; oc.ldY = L; oc.sstride = per_pixel_sigma ? L : 0; oc.info = dI[bi];
        const float *sg = per_pixel_sigma ? dS[bi] : dSshared;
        rc = launch_solve(lib, dY[bi], sg, n, oc, dC[bi], dCS[bi], dR[bi]);
        if (rc != LINMIN_OK) { cleanup(); return rc; }
        CKH(cudaMemcpyAsync(coeffs_out + p0 * R, dC[bi], (size_t)n * R * sizeof(float), cudaMemcpyDeviceToHost, s));
        if (coeff_sigma_out)
            CKH(cudaMemcpyAsync(coeff_sigma_out + p0 * R, dCS[bi], (size_t)n * R * sizeof(float), cudaMemcpyDeviceToHost, s));
        if (resid_out)
            CKH(cudaMemcpyAsync(resid_out + p0, dR[bi], (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, s));
        if (o.info)
            CKH(cudaMemcpyAsync(o.info + p0, dI[bi], (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    }
    for (int b = 0; b < NBUF; ++b) CKH(cudaStreamSynchronize(st[b]));
    cleanup();
    return wrc;
#undef CKH
}

// ---------------------------------------------------------------- NEXT rows 3-4: detect.cuh

int linmin_additional_spectra(const float *wavelength, int32_t L, int32_t n_extra, float *out, int32_t ld_out,
                              int32_t col0, void *stream) {
    if (!out || L < 1 || (n_extra != 4 && n_extra != 12) || col0 < 0 || ld_out < col0 + n_extra) return LINMIN_ERR_INVALID_ARGUMENT;
    if (L > LINMIN_MAX_L) return LINMIN_ERR_UNSUPPORTED_SIZE;
    additional_spectra_kernel<<<(L + 127) / 128, 128, 0, (cudaStream_t)stream>>>(wavelength, L, n_extra, out, ld_out, col0);
    CK(cudaGetLastError());
    return LINMIN_OK;
}

int linmin_detection_thresholds(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                float *thresholds_out, void *stream) {
    return linmin_detection_thresholds_ex(coeffs, present, N, R, 0, thresholds_out, stream);
}

int linmin_detection_thresholds_ex(const float *coeffs, const unsigned char *present, int64_t N, int32_t R,
                                   int32_t whole_class, float *thresholds_out, void *stream) {
    if (!coeffs || !present || !thresholds_out || N < 0 || R < 1) return LINMIN_ERR_INVALID_ARGUMENT;
    if (whole_class != 0 && whole_class != 1) return LINMIN_ERR_INVALID_ARGUMENT;
    if (R > LINMIN_MAX_R) return LINMIN_ERR_UNSUPPORTED_SIZE;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int block = R * std::max(1, 256 / R);
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N * R + block - 1) / block, (int64_t)sms * 8));
    double *part = nullptr;
    CK(staging_alloc((void **)&part, (size_t)grid * R * 6 * sizeof(double), st));
    threshold_partial_kernel<<<grid, block, (size_t)block * 6 * sizeof(double), st>>>(coeffs, present, N, R, whole_class, part);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        threshold_final_kernel<<<(R + 63) / 64, 64, 0, st>>>(part, grid, R, thresholds_out);
        e = cudaGetLastError();
    }
    cudaFreeAsync(part, st);
    CK(e);
    return LINMIN_OK;
}

int linmin_detect(const float *coeffs, const float *coeff_sigma, const float *resid, const float *thresholds,
                  float rms_max, int64_t N, int32_t R, unsigned char *mask_out, unsigned long long *counts_out, void *stream) {
    if (!coeffs || !coeff_sigma || !resid || !thresholds || !mask_out || N < 0 || R < 1) return LINMIN_ERR_INVALID_ARGUMENT;
    if (R > LINMIN_MAX_R) return LINMIN_ERR_UNSUPPORTED_SIZE;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (counts_out) CK(cudaMemsetAsync(counts_out, 0, (size_t)R * sizeof(unsigned long long), st));
    if (N == 0) return LINMIN_OK;
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N * R + 255) / 256, (int64_t)sms * 8));
    detect_kernel<<<grid, 256, (size_t)R * sizeof(unsigned int), st>>>(coeffs, coeff_sigma, resid, thresholds, rms_max, N, R,
                                                                        mask_out, counts_out);
    CK(cudaGetLastError());
    return LINMIN_OK;
}

int linmin_second_pass(const float *A, const float *Y, const float *sigma, int64_t N, int32_t L, int32_t R,
                       const unsigned char *keep, const linmin_opts *opts, float *coeffs_out, float *coeff_sigma_out,
                       float *resid_out) {
    int rc = check_sizes(N, L, R);
    if (rc != LINMIN_OK) return rc;
    if (!A || !keep || (N > 0 && (!Y || !coeffs_out))) return LINMIN_ERR_INVALID_ARGUMENT;
    Resolved o;
    rc = resolve_opts(opts, L, &o);
    if (rc != LINMIN_OK) return rc;
    // the size of the sub-library decides every allocation below: the one place where the host reads device data
    std::vector<unsigned char> hk((size_t)R);
    CK(cudaMemcpyAsync(hk.data(), keep, (size_t)R, cudaMemcpyDeviceToHost, o.stream));
    CK(cudaStreamSynchronize(o.stream));
    std::vector<int> idx;
    for (int i = 0; i < R; ++i) if (hk[i]) idx.push_back(i);
    const int Rs = (int)idx.size();
    if (Rs < 1) return LINMIN_ERR_INVALID_ARGUMENT;
    int *didx = nullptr;
    float *sub = nullptr, *cs = nullptr, *ss = nullptr;
    struct FreeV { void *p; cudaStream_t s; ~FreeV() { if (p) cudaFreeAsync(p, s); } };
    CK(staging_alloc((void **)&didx, (size_t)Rs * sizeof(int), o.stream));
    FreeV f0{didx, o.stream};
    CK(cudaMemcpyAsync(didx, idx.data(), (size_t)Rs * sizeof(int), cudaMemcpyHostToDevice, o.stream));
    CK(cudaStreamSynchronize(o.stream));     // idx is a host vector that dies with this call
    CK(staging_alloc((void **)&sub, (size_t)L * Rs * sizeof(float), o.stream));
    FreeV f1{sub, o.stream};
    gather_columns_kernel<<<(L * Rs + 255) / 256, 256, 0, o.stream>>>(A, L, R, didx, Rs, sub);
    CK(cudaGetLastError());
    if (N == 0) return LINMIN_OK;
    CK(staging_alloc((void **)&cs, (size_t)N * Rs * sizeof(float), o.stream));
    FreeV f2{cs, o.stream};
    if (coeff_sigma_out) CK(staging_alloc((void **)&ss, (size_t)N * Rs * sizeof(float), o.stream));
    FreeV f3{ss, o.stream};
    rc = linmin_unmix(sub, Y, sigma, N, L, Rs, opts, cs, ss, resid_out);
    if (rc < 0) return rc;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((N * Rs + 255) / 256, (int64_t)sms * 8));
    CK(cudaMemsetAsync(coeffs_out, 0, (size_t)N * R * sizeof(float), o.stream));
    scatter_columns_kernel<<<grid, 256, 0, o.stream>>>(cs, N, Rs, didx, R, coeffs_out);
    CK(cudaGetLastError());
    if (coeff_sigma_out) {
        CK(cudaMemsetAsync(coeff_sigma_out, 0, (size_t)N * R * sizeof(float), o.stream));
        scatter_columns_kernel<<<grid, 256, 0, o.stream>>>(ss, N, Rs, didx, R, coeff_sigma_out);
        CK(cudaGetLastError());
    }
    return rc;
}

int linmin_autofit(const float *A, int32_t L, int32_t R, void *stream, float *resid_ls_out, float *resid_nn_out) {
    int rc = check_sizes(0, L, R);
    if (rc != LINMIN_OK) return rc;
    if (!A || R < 2 || (!resid_ls_out && !resid_nn_out)) return LINMIN_ERR_INVALID_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    struct FreeV { void *p; cudaStream_t s; ~FreeV() { if (p) cudaFreeAsync(p, s); } };
    if (resid_ls_out) {
        double *Q = nullptr;
        CK(staging_alloc((void **)&Q, (size_t)R * L * (R - 1) * sizeof(double), st));
        FreeV fq{Q, st};
        autofit_ls_kernel<<<R, 256, 0, st>>>(A, L, R, Q, resid_ls_out);
        CK(cudaGetLastError());
    }
    if (resid_nn_out) {
        // eq. 7 under positivity: R problems of R - 1 endmembers through the pos option of the solver (N = 1 each)
        float *Sn = nullptr, *yrow = nullptr, *a = nullptr;
        CK(staging_alloc((void **)&Sn, (size_t)L * (R - 1) * sizeof(float), st));
        FreeV f0{Sn, st};
        CK(staging_alloc((void **)&yrow, (size_t)L * sizeof(float), st));
        FreeV f1{yrow, st};
        CK(staging_alloc((void **)&a, (size_t)(R - 1) * sizeof(float), st));
        FreeV f2{a, st};
        Resolved o;
        resolve_opts(nullptr, L, &o);
        o.stream = st; o.constraint = LINMIN_CONSTRAINT_POSITIVITY_ONLY;
        for (int n = 0; n < R; ++n) {
            drop_column_kernel<<<(L * (R - 1) + 255) / 256, 256, 0, st>>>(A, L, R, n, Sn, yrow);
            CK(cudaGetLastError());
            linmin_library *lib = nullptr;
            int wrc = library_create_impl(Sn, L, R - 1, st, false, false, LINMIN_CONSTRAINT_POSITIVITY_ONLY,
                                          LINMIN_WEIGHTING_NONE, nullptr, &lib);
            if (wrc < 0) return wrc;
            rc = launch_solve(lib, yrow, nullptr, 1, o, a, nullptr, nullptr);
            if (rc == LINMIN_OK) {
                autofit_residue_kernel<<<(L + 127) / 128, 128, 0, st>>>(A, L, R, n, Sn, a, resid_nn_out);
                if (cudaGetLastError() != cudaSuccess) rc = LINMIN_ERR_CUDA;
            }
            linmin_library_destroy(lib);
            if (rc != LINMIN_OK) return rc;
        }
    }
    return LINMIN_OK;
}

}  // extern "C"
