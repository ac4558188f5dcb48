// disc_api.cu -- context, argument validation, launch plumbing and the extern "C" boundary of
// include/disc.h.  Every step of the path runs in the kernels of moments.cuh / field.cuh / pyramid.cuh;
// this file only sizes grids, picks template instances and enqueues launches on the caller's stream.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/disc.h"
#include "launch.h"
#include "mask.cuh"
#include "pyramid.cuh"

using namespace disc;

namespace {

struct Level {
    int nx, ny, nz;
    size_t N;
    float* ct;       // pyramid copy (levels >= 1); level 0 uses the caller's pointer
    float* cbct;     // idem
    float* zhat;     // cached CBCT patch z-score (I_s - mu_s)/sigma_s of this level   [N]
    float* m;        // warped CT                                                        [N]
    float* sp;       // corrected CBCT                                                   [N]
    float* disp;     // field of this level (levels >= 1; level 0 uses the caller's)     [3N]
    float* scratch;  // field after the x,y Gaussian passes                              [3N]
    // NEXT-1 / diagnostics (allocated by disc_set_mask / disc_set_diagnostics)
    float* mu_s;     // CBCT patch mean                                                  [N]
    float* var_s;    // CBCT patch variance                                              [N]
    float* A;        // a(x): E(M) while it is being computed                            [N]
    float* B;        // b(x): VAR(M) while it is being computed                          [N]
    unsigned char* xi;  // 0 free, 255 masked and unfilled, k = filled in pass k         [N bytes]
    unsigned* fill_list;  // work lists of the fill passes: odd passes [0, N), even passes [N, 2N)  (N < 2^32)  [2N]
    unsigned* fill_queued;  // one bit per voxel: already on the next pass's list          [ceil(N/32)]
};

thread_local char g_create_error[256] = "";

}  // namespace

struct disc_ctx {
    int dims[3];
    float spacing[3];
    int R[3];         // patch radius per axis (R[0] == R[1])
    int fac[3];       // pyramid factor per axis, 1 or 2
    float sigma;
    int levels, iters;
    int K;
    int force_mode;   // 1 Thirion (default), 2 double force
    float stop_eps;   // < 0: stopping criterion off (default)
    StopCtl* d_stop;  // device-side state of the criterion
    int runs_host[DISC_MAX_LEVELS];   // iterations per level when the criterion is off
    DevInfo di;       // device the context was created on, and its SM count
    GaussTaps taps;
    Level lv[DISC_MAX_LEVELS];
    // NEXT-1: reliability mask and interpolation of a, b
    int mask_on;
    float mask_hu0, mask_a_min, mask_a_max;   // < 0: derived from the images
    int fill_radius, max_fill_passes;
    float fill_h;
    int diag_on;      // Fig. 9 (e), (f): mean a, mean b per iteration
    MaskCtl* d_mask;
    int fill_grid;       // blocks of k_fill_list (all resident: it is a cooperative launch)
    double* d_partial;   // block partials of the deterministic reductions   [2 * kReduceBlocks]
    double* d_mean_a;    // [levels * iters], level-major from the coarsest level
    double* d_mean_b;
    float* cbct_shift;   // CBCT + Delta HU at level 0                       [N_0]
    float* h2d_ct;    // device staging for disc_register_host
    float* h2d_cbct;
    float* d_out_disp;
    float* d_out_corr;
    unsigned long long launches;
    char err[256];
};

namespace {

disc_status fail(disc_ctx* c, disc_status st, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c ? c->err : g_create_error, 256, fmt, ap);
    va_end(ap);
    return st;
}

disc_status check_launch(disc_ctx* c, const char* what) {
    c->launches++;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
    return DISC_OK;
}

#define DISC_TRY(expr)                         \
    do {                                       \
        disc_status _s = (expr);               \
        if (_s != DISC_OK) return _s;          \
    } while (0)

#define DISC_NEED(c, cond, msg)                                             \
    do {                                                                    \
        if (!(cond)) return fail((c), DISC_ERR_INVALID_ARG, "%s", (msg));   \
    } while (0)

bool level_ok(const disc_ctx* c, int level) { return level >= 0 && level < c->levels; }

const IterCtl kNoCtl = {nullptr, 0};
constexpr int kReduceBlocks = 592;   // grid of the grid-stride reductions (4 per SM on a B200)

// every entry point runs on the device the context was created on (scratch, attributes and grid sizes belong to it)
disc_status check_device(disc_ctx* c) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(c, DISC_ERR_CUDA, "cudaGetDevice failed");
    if (dev != c->di.dev)
        return fail(c, DISC_ERR_INVALID_ARG, "context belongs to CUDA device %d, current device is %d", c->di.dev, dev);
    return DISC_OK;
}

template <int MODE>
disc_status launch_moments(disc_ctx* c, const Level& L, const float* vol, const float* aux, float* out0,
                           float* out1, IterCtl ctl, cudaStream_t st) {
    if (!launch_moments_any(c->di, c->R[0], c->R[2], MODE, vol, aux, out0, out1, L.nx, L.ny, L.nz, DISC_EPS_VAR, ctl, st))
        return fail(c, DISC_ERR_UNSUPPORTED, "no moments kernel for patch radius (%d,%d,%d)", c->R[0], c->R[1], c->R[2]);
    return check_launch(c, "k_moments");
}

// force: 0 = plain smoothing, otherwise the context's force mode
disc_status launch_force_gxy(disc_ctx* c, bool force, const Level& L, const float* m, const float* s, const float* rin,
                             float* rout, IterCtl ctl, cudaStream_t st, StopReq stop = StopReq{nullptr, 0, 0.f}) {
    const int FORCE = force ? c->force_mode : 0;
    if (!launch_force_gxy_any(c->di, c->K, FORCE, m, s, rin, rout, L.nx, L.ny, L.nz, DISC_EPS_DEN, c->taps, ctl, stop, st))
        return fail(c, DISC_ERR_UNSUPPORTED, "Gaussian radius %d unsupported", c->K);
    return check_launch(c, "k_force_gxy");
}

template <bool WARP>
disc_status launch_gz_warp(disc_ctx* c, const Level& L, const float* rin, float* rout, const float* moving,
                           float* mout, IterCtl ctl, cudaStream_t st) {
    if (!launch_gz_warp_any(c->di, c->K, WARP, rin, rout, moving, mout, L.nx, L.ny, L.nz, c->taps, ctl, st))
        return fail(c, DISC_ERR_UNSUPPORTED, "Gaussian radius %d unsupported", c->K);
    return check_launch(c, "k_gz_warp");
}

disc_status launch_warp(disc_ctx* c, const Level& L, const float* moving, const float* r, float* out, cudaStream_t st) {
    launch_warp_kernel(moving, r, out, L.nx, L.ny, L.nz, st);
    return check_launch(c, "k_warp");
}

disc_status launch_downsample(disc_ctx* c, const Level& fine, const float* in, float* out, cudaStream_t st) {
    const int* f = c->fac;
    const int mx = fine.nx / f[0], my = fine.ny / f[1], mz = fine.nz / f[2];
    dim3 grid((mx + 127) / 128, my, mz);
    // 8-byte loads of the two x neighbours need an even row length (it is: nx = 2 mx) and an 8-byte aligned base
    if (f[0] == 2 && (reinterpret_cast<uintptr_t>(in) & 7u) == 0)
        k_downsample<true><<<grid, 128, 0, st>>>(in, out, mx, my, mz, f[0], f[1], f[2]);
    else
        k_downsample<false><<<grid, 128, 0, st>>>(in, out, mx, my, mz, f[0], f[1], f[2]);
    return check_launch(c, "k_downsample");
}

disc_status launch_upsample(disc_ctx* c, const Level& coarse, const float* in, float* out, cudaStream_t st) {
    const int* f = c->fac;
    const int nx = f[0] * coarse.nx, ny = f[1] * coarse.ny, nz = f[2] * coarse.nz;
    if (f[0] == 2 && f[1] == 2 && f[2] == 2 && (reinterpret_cast<uintptr_t>(out) & 7u) == 0) {   // 8-byte stores of x pairs
        dim3 grid2((coarse.nx + 127) / 128, coarse.ny, 3 * coarse.nz);
        k_upsample_field_222<<<grid2, 128, 0, st>>>(in, out, coarse.nx, coarse.ny, coarse.nz);
        return check_launch(c, "k_upsample_field_222");
    }
    dim3 grid((nx + 127) / 128, ny, 3 * nz);
    k_upsample_field<<<grid, 128, 0, st>>>(in, out, coarse.nx, coarse.ny, coarse.nz, f[0], f[1], f[2]);
    return check_launch(c, "k_upsample_field");
}


// ---------------------------------------------------------------- NEXT-1 plumbing
bool ab_path(const disc_ctx* c) { return c->mask_on || c->diag_on; }

// grid of the cooperative fill kernel: every block must be resident at once
disc_status fill_grid_for(disc_ctx* c, int* grid) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fill_list, 256, 0) != cudaSuccess || per_sm < 1)
        return fail(c, DISC_ERR_CUDA, "no resident block of the fill kernel: %s", cudaGetErrorString(cudaGetLastError()));
    *grid = per_sm * c->di.n_sm;
    return DISC_OK;
}

// Fig.-9 slots of iterations that a run does not reach (early stop, disc_iterate on one level) read NaN, not the
// previous run's averages: all-ones bytes are a quiet NaN in fp64.
disc_status clear_diagnostics(disc_ctx* c, cudaStream_t st) {
    if (!c->diag_on || !c->d_mean_a) return DISC_OK;
    const size_t nd = (size_t)c->levels * (c->iters > 0 ? c->iters : 1) * sizeof(double);
    if (cudaMemsetAsync(c->d_mean_a, 0xff, nd, st) != cudaSuccess || cudaMemsetAsync(c->d_mean_b, 0xff, nd, st) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "cudaMemsetAsync (diagnostics) failed");
    return DISC_OK;
}

// frees the mask / diagnostics buffers and nulls the pointers (so that a later alloc_ab starts from scratch)
void free_ab(disc_ctx* c) {
    for (int l = 0; l < DISC_MAX_LEVELS; ++l) {
        Level& L = c->lv[l];
        cudaFree(L.mu_s); cudaFree(L.var_s); cudaFree(L.A); cudaFree(L.B); cudaFree(L.xi); cudaFree(L.fill_list); cudaFree(L.fill_queued);
        L.mu_s = L.var_s = L.A = L.B = nullptr; L.xi = nullptr; L.fill_list = nullptr; L.fill_queued = nullptr;
    }
    cudaFree(c->d_mask); cudaFree(c->d_partial); cudaFree(c->d_mean_a); cudaFree(c->d_mean_b); cudaFree(c->cbct_shift);
    c->d_mask = nullptr; c->d_partial = nullptr; c->d_mean_a = c->d_mean_b = nullptr; c->cbct_shift = nullptr;
}

// all or nothing: c->d_mask != NULL means every buffer below exists
disc_status alloc_ab(disc_ctx* c) {
    if (c->d_mask) return DISC_OK;
    bool ok = cudaMalloc(&c->d_mask, sizeof(MaskCtl)) == cudaSuccess && cudaMemset(c->d_mask, 0, sizeof(MaskCtl)) == cudaSuccess &&
              cudaMalloc(&c->d_partial, sizeof(double) * 2 * kReduceBlocks) == cudaSuccess;
    const size_t nd = (size_t)c->levels * (c->iters > 0 ? c->iters : 1);
    ok = ok && cudaMalloc(&c->d_mean_a, sizeof(double) * nd) == cudaSuccess && cudaMalloc(&c->d_mean_b, sizeof(double) * nd) == cudaSuccess &&
         cudaMemset(c->d_mean_a, 0, sizeof(double) * nd) == cudaSuccess && cudaMemset(c->d_mean_b, 0, sizeof(double) * nd) == cudaSuccess;
    ok = ok && cudaMalloc(&c->cbct_shift, c->lv[0].N * sizeof(float)) == cudaSuccess;
    for (int l = 0; ok && l < c->levels; ++l) {
        Level& L = c->lv[l];
        const size_t b = L.N * sizeof(float);
        ok = cudaMalloc(&L.mu_s, b) == cudaSuccess && cudaMalloc(&L.var_s, b) == cudaSuccess && cudaMalloc(&L.A, b) == cudaSuccess &&
             cudaMalloc(&L.B, b) == cudaSuccess && cudaMalloc(&L.xi, L.N) == cudaSuccess;
        if (ok && L.N <= 0xffffffffull)
            ok = cudaMalloc(&L.fill_list, 2 * L.N * sizeof(unsigned)) == cudaSuccess &&
                 cudaMalloc(&L.fill_queued, (L.N + 31) / 32 * sizeof(unsigned)) == cudaSuccess;
    }
    if (!ok) {
        cudaGetLastError();
        free_ab(c);   // a retry must not find d_mask set with the other buffers missing
        return fail(c, DISC_ERR_ALLOC, "cudaMalloc failed (mask / diagnostics buffers)");
    }
    return DISC_OK;
}

unsigned reduce_grid(size_t N) {
    const size_t b = (N + 255) / 256;
    return (unsigned)(b < (size_t)kReduceBlocks ? b : (size_t)kReduceBlocks);
}

// the CBCT patch moments of a level (they never change within it)
disc_status cache_cbct_moments(disc_ctx* c, const Level& L, const float* cbct, cudaStream_t st) {
    return launch_moments<kModeMoments>(c, L, cbct, nullptr, L.mu_s, L.var_s, kNoCtl, st);
}

// A1 steps 1-3 with explicit a, b: moments of m, Eqs. (5)-(6), [Eq. (7), Eqs. (8)-(10)], a I_s + b.
// out = nullptr: diagnostics only.  slot < 0: no diagnostics.
disc_status correct_ab(disc_ctx* c, const Level& L, const float* cbct, const float* m, float* out, bool use_mask, int slot,
                       IterCtl ctl, cudaStream_t st) {
    DISC_TRY(launch_moments<kModeMoments>(c, L, m, nullptr, L.A, L.B, ctl, st));
    const unsigned g = reduce_grid(L.N);
    if (use_mask) {
        k_fill_reset<<<1, 1, 0, st>>>(c->d_mask, ctl);
        DISC_TRY(check_launch(c, "k_fill_reset"));
        // one round per block (each round of the list append holds three block barriers: a grid-stride loop of 55 rounds
        // ran them back to back, 157 us at 256x256x128; independent blocks overlap them)
        const size_t nb = (L.N + 255) / 256;
        const unsigned gm = (unsigned)(nb < 0x7fffffffull ? nb : 0x7fffffffull);
        k_ab_mask<true><<<gm, 256, 0, st>>>(m, cbct, L.mu_s, L.var_s, L.A, L.B, L.xi, L.N, DISC_EPS_VAR, c->d_mask, ctl, L.fill_list, L.fill_queued);
        DISC_TRY(check_launch(c, "k_ab_mask"));
        const float inv_h2 = 1.f / (c->fill_h * c->fill_h);
        if (L.fill_list) {
            // all passes in one cooperative launch over the compacted list of masked voxels
            const float* a_cbct = cbct; float* a_A = L.A; float* a_B = L.B; unsigned char* a_xi = L.xi;
            unsigned* a_list = L.fill_list; unsigned* a_list2 = L.fill_list + L.N; unsigned* a_q = L.fill_queued;
            int a_nx = L.nx, a_ny = L.ny, a_nz = L.nz, a_rt = c->fill_radius, a_max = c->max_fill_passes;
            float a_h = inv_h2; MaskCtl* a_ctl = c->d_mask; IterCtl a_ictl = ctl;
            void* args[] = {&a_cbct, &a_A, &a_B, &a_xi, &a_list, &a_list2, &a_q, &a_nx, &a_ny, &a_nz, &a_rt, &a_h, &a_max, &a_ctl, &a_ictl};
            cudaError_t e = cudaLaunchCooperativeKernel((const void*)k_fill_list, dim3(c->fill_grid), dim3(256), args, 0, st);
            if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "k_fill_list: %s", cudaGetErrorString(e));
            DISC_TRY(check_launch(c, "k_fill_list"));
        } else {
            dim3 grid((L.nx + 127) / 128, L.ny, L.nz);
            for (int p = 1; p <= c->max_fill_passes; ++p) {
                k_fill_pass<<<grid, 128, 0, st>>>(cbct, L.A, L.B, L.xi, L.nx, L.ny, L.nz, c->fill_radius, inv_h2, p, c->d_mask, ctl);
                DISC_TRY(check_launch(c, "k_fill_pass"));
            }
        }
    } else {
        k_ab_mask<false><<<g, 256, 0, st>>>(m, cbct, L.mu_s, L.var_s, L.A, L.B, nullptr, L.N, DISC_EPS_VAR, c->d_mask, ctl, nullptr, nullptr);
        DISC_TRY(check_launch(c, "k_ab"));
    }
    k_apply_ab<<<g, 256, 0, st>>>(cbct, L.A, L.B, out, L.N, c->d_partial, c->d_mask, slot >= 0 ? c->d_mean_a : nullptr,
                                  c->d_mean_b, slot >= 0 ? slot : 0, ctl);
    return check_launch(c, "k_apply_ab");
}

// Delta HU, HU_0 and (unless given) a_m, a_min, a_max from the two full-resolution images, into the device-side
// MaskCtl.  `cbct` may be the unshifted image: the shift changes no variance.
disc_status mask_parameters(disc_ctx* c, const float* ct, const float* cbct, cudaStream_t st) {
    Level& L = c->lv[0];
    if (cudaMemsetAsync(c->d_mask, 0, sizeof(MaskCtl), st) != cudaSuccess) return fail(c, DISC_ERR_CUDA, "cudaMemsetAsync failed");
    k_sum2<<<reduce_grid(L.N), 256, 0, st>>>(ct, cbct, L.N, c->d_partial, c->d_mask, c->mask_hu0);
    DISC_TRY(check_launch(c, "k_sum2"));
    if (c->mask_a_min < 0.f) {
        DISC_TRY(launch_moments<kModeMoments>(c, L, cbct, nullptr, L.mu_s, L.var_s, kNoCtl, st));
        DISC_TRY(launch_moments<kModeMoments>(c, L, ct, nullptr, L.A, L.B, kNoCtl, st));     // r = 0: I_m = CT
        for (int p = 0; p < 4; ++p) {
            k_select_hist<<<reduce_grid(L.N), 256, 0, st>>>(L.var_s, L.B, L.N, DISC_EPS_VAR, p, c->d_mask);
            DISC_TRY(check_launch(c, "k_select_hist"));
            k_select_step<<<1, 1, 0, st>>>(p, c->d_mask);
            DISC_TRY(check_launch(c, "k_select_step"));
        }
    }
    k_mask_set<<<1, 1, 0, st>>>(c->d_mask, c->mask_hu0, c->mask_a_min, c->mask_a_max);
    return check_launch(c, "k_mask_set");
}

// n_iters x { correct, force+update+Gxy, Gz+warp } on level L; on entry L.m must hold warp(ct, disp).
// With final_warp the last iteration also refreshes L.m (needed when the caller goes on using it).
disc_status iterate_level(disc_ctx* c, Level& L, const float* ct, const float* cbct, float* disp, int n_iters,
                          bool final_warp, cudaStream_t st) {
    const int level = (int)(&L - c->lv);
    const bool stop = c->stop_eps >= 0.f;
    c->runs_host[level] = n_iters;
    if (stop) { launch_stop_reset(c->d_stop, st); DISC_TRY(check_launch(c, "k_stop_reset")); }
    disc_status rc = DISC_OK;
    for (int k = 0; k < n_iters && rc == DISC_OK; ++k) {
        // with the criterion on, every kernel of iteration k falls through once an earlier iteration has tripped it;
        // the field and L.m then stay those of the last iteration run (its z pass always refreshes L.m: k + 1 < n_iters)
        const IterCtl ctl = stop ? IterCtl{&c->d_stop->stop_iter, k} : kNoCtl;
        const int slot = c->diag_on && k < c->iters ? (c->levels - 1 - level) * c->iters + k : -1;
        if (c->mask_on) {
            rc = correct_ab(c, L, cbct, L.m, L.sp, true, slot, ctl, st);                       // A1 steps 1,2,3
        } else {
            rc = launch_moments<kModeCorrect>(c, L, L.m, L.zhat, L.sp, nullptr, ctl, st);     // A1 steps 1,3
            if (rc == DISC_OK && slot >= 0) rc = correct_ab(c, L, cbct, L.m, nullptr, false, slot, ctl, st);   // Fig. 9 only
        }
        // A1 steps 4,5,6(x,y); with the criterion on, the same kernel adds up sum|dr|, sum|r| of the iteration and its
        // last block takes the decision (l^(k)): kernels of later iterations fall through
        const StopReq sreq = stop ? StopReq{c->d_stop, k, c->stop_eps} : StopReq{nullptr, 0, 0.f};
        if (rc == DISC_OK) rc = launch_force_gxy(c, true, L, L.m, L.sp, disp, L.scratch, ctl, st, sreq);
        if (rc == DISC_OK) {
            if (k + 1 < n_iters || final_warp)
                rc = launch_gz_warp<true>(c, L, L.scratch, disp, ct, L.m, ctl, st);            // A1 step 6(z) + next I_m^(k)
            else
                rc = launch_gz_warp<false>(c, L, L.scratch, disp, nullptr, nullptr, ctl, st);
        }
    }
    if (rc == DISC_OK && stop) { launch_stop_record(c->d_stop, level, n_iters, st); rc = check_launch(c, "k_stop_record"); }
    return rc;
}

void free_ctx(disc_ctx* c) {
    for (int l = 0; l < DISC_MAX_LEVELS; ++l) {
        Level& L = c->lv[l];
        cudaFree(L.ct); cudaFree(L.cbct); cudaFree(L.zhat); cudaFree(L.m); cudaFree(L.sp);
        cudaFree(L.disp); cudaFree(L.scratch);
        cudaFree(L.mu_s); cudaFree(L.var_s); cudaFree(L.A); cudaFree(L.B); cudaFree(L.xi);
    }
    cudaFree(c->d_mask); cudaFree(c->d_partial); cudaFree(c->d_mean_a); cudaFree(c->d_mean_b); cudaFree(c->cbct_shift);
    cudaFree(c->d_stop);
    cudaFree(c->h2d_ct); cudaFree(c->h2d_cbct); cudaFree(c->d_out_disp); cudaFree(c->d_out_corr);
    delete c;
}

}  // namespace

// =====================================================================================
extern "C" {

disc_status disc_create(disc_ctx** out, const int dims[3], const float spacing[3], int patch_radius,
                        float sigma_smooth, int levels, int iters) {
    const int R3[3] = {patch_radius, patch_radius, patch_radius}, f3[3] = {2, 2, 2};
    return disc_create_ex(out, dims, spacing, R3, sigma_smooth, levels, iters, f3);
}

disc_status disc_create_ex(disc_ctx** out, const int dims[3], const float spacing[3], const int patch_radius[3],
                           float sigma_smooth, int levels, int iters, const int pyramid_factor[3]) {
    if (!out) return fail(nullptr, DISC_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    if (!dims || !spacing || !patch_radius || !pyramid_factor)
        return fail(nullptr, DISC_ERR_INVALID_ARG, "dims/spacing/patch_radius/pyramid_factor is NULL");
    if (levels < 1 || levels > DISC_MAX_LEVELS) return fail(nullptr, DISC_ERR_INVALID_ARG, "levels must be in 1..%d", DISC_MAX_LEVELS);
    for (int i = 0; i < 3; ++i) {
        if (dims[i] < 1) return fail(nullptr, DISC_ERR_INVALID_ARG, "dims[%d] < 1", i);
        if (!(spacing[i] > 0.f)) return fail(nullptr, DISC_ERR_INVALID_ARG, "spacing[%d] <= 0", i);
        if (pyramid_factor[i] != 1 && pyramid_factor[i] != 2)
            return fail(nullptr, DISC_ERR_INVALID_ARG, "pyramid_factor[%d] must be 1 or 2", i);
        if (pyramid_factor[i] == 2 && dims[i] % (1 << (levels - 1)) != 0)
            return fail(nullptr, DISC_ERR_INVALID_ARG, "dims[%d]=%d not divisible by 2^(levels-1)", i, dims[i]);
        if (patch_radius[i] < 0) return fail(nullptr, DISC_ERR_INVALID_ARG, "patch_radius < 0");
    }
    if (!(sigma_smooth > 0.f)) return fail(nullptr, DISC_ERR_INVALID_ARG, "sigma_smooth <= 0");
    if (iters < 0) return fail(nullptr, DISC_ERR_INVALID_ARG, "iters < 0");
    for (int i = 0; i < 3; ++i)
        if (patch_radius[i] > DISC_MAX_PATCH_RADIUS)
            return fail(nullptr, DISC_ERR_UNSUPPORTED, "patch_radius %d > %d", patch_radius[i], DISC_MAX_PATCH_RADIUS);
    if (patch_radius[0] != patch_radius[1])
        return fail(nullptr, DISC_ERR_UNSUPPORTED, "patch radii along x and y must be equal (%d != %d)", patch_radius[0], patch_radius[1]);
    const int K = (int)std::ceil(3.0 * (double)sigma_smooth);
    if (K > DISC_MAX_GAUSS_RADIUS)
        return fail(nullptr, DISC_ERR_UNSUPPORTED, "Gaussian radius ceil(3 sigma) = %d > %d", K, DISC_MAX_GAUSS_RADIUS);

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    int major = 0;
    e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
    if (major != 10) return fail(nullptr, DISC_ERR_UNSUPPORTED, "device compute capability %d.x, this library is sm_100a only", major);
    if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, DISC_ERR_UNSUPPORTED, "device ordinal %d >= %d", dev, kMaxDevices);

    disc_ctx* c = new (std::nothrow) disc_ctx();
    if (!c) return fail(nullptr, DISC_ERR_ALLOC, "out of host memory");
    std::memset(c, 0, sizeof(*c));
    for (int i = 0; i < 3; ++i) { c->dims[i] = dims[i]; c->spacing[i] = spacing[i]; }
    c->di.dev = dev;
    c->di.n_sm = 148;
    cudaDeviceGetAttribute(&c->di.n_sm, cudaDevAttrMultiProcessorCount, dev);
    for (int i = 0; i < 3; ++i) { c->R[i] = patch_radius[i]; c->fac[i] = pyramid_factor[i]; }
    c->sigma = sigma_smooth; c->levels = levels; c->iters = iters; c->K = K;
    c->force_mode = DISC_FORCE_THIRION;
    c->stop_eps = -1.f;
    if (cudaMalloc(&c->d_stop, sizeof(StopCtl)) != cudaSuccess || cudaMemset(c->d_stop, 0, sizeof(StopCtl)) != cudaSuccess) {
        cudaGetLastError();
        free_ctx(c);
        return fail(nullptr, DISC_ERR_ALLOC, "cudaMalloc failed (stop control)");
    }
    // Gaussian taps: fp64, normalised to sum 1, then rounded to fp32 (reading A10)
    {
        double w[kMaxGaussTaps], sum = 0.0;
        for (int i = -K; i <= K; ++i) { w[i + K] = std::exp(-(double)(i * i) / (2.0 * (double)sigma_smooth * (double)sigma_smooth)); sum += w[i + K]; }
        for (int i = 0; i < 2 * K + 1; ++i) c->taps.w[i] = (float)(w[i] / sum);
    }
    for (int l = 0; l < levels; ++l) {
        Level& L = c->lv[l];
        L.nx = dims[0]; L.ny = dims[1]; L.nz = dims[2];
        for (int i = 0; i < l; ++i) { L.nx /= c->fac[0]; L.ny /= c->fac[1]; L.nz /= c->fac[2]; }
        L.N = (size_t)L.nx * L.ny * L.nz;
        const size_t b = L.N * sizeof(float);
        bool ok = cudaMalloc(&L.zhat, b) == cudaSuccess && cudaMalloc(&L.m, b) == cudaSuccess &&
                  cudaMalloc(&L.sp, b) == cudaSuccess && cudaMalloc(&L.scratch, 3 * b) == cudaSuccess;
        if (ok && l > 0)
            ok = cudaMalloc(&L.ct, b) == cudaSuccess && cudaMalloc(&L.cbct, b) == cudaSuccess &&
                 cudaMalloc(&L.disp, 3 * b) == cudaSuccess;
        if (!ok) {
            cudaGetLastError();
            free_ctx(c);
            return fail(nullptr, DISC_ERR_ALLOC, "cudaMalloc failed at level %d", l);
        }
    }
    *out = c;
    return DISC_OK;
}

void disc_destroy(disc_ctx* ctx) {
    if (!ctx) return;
    cudaDeviceSynchronize();
    free_ctx(ctx);
}

const char* disc_last_error(const disc_ctx* ctx) { return ctx ? ctx->err : g_create_error; }

unsigned long long disc_launch_count(const disc_ctx* ctx) { return ctx ? ctx->launches : 0ull; }

disc_status disc_set_force(disc_ctx* c, int mode) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_NEED(c, mode == DISC_FORCE_THIRION || mode == DISC_FORCE_DOUBLE, "force mode must be DISC_FORCE_THIRION or DISC_FORCE_DOUBLE");
    c->force_mode = mode;
    return DISC_OK;
}

disc_status disc_set_stop(disc_ctx* c, float eps) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_NEED(c, eps == eps, "eps is NaN");
    c->stop_eps = eps >= 0.f ? eps : -1.f;
    return DISC_OK;
}

disc_status disc_iterations_run(disc_ctx* c, int* out_host) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_NEED(c, out_host, "NULL pointer");
    if (c->stop_eps >= 0.f) {
        int runs[DISC_MAX_LEVELS];
        cudaError_t e = cudaDeviceSynchronize();
        if (e == cudaSuccess) e = cudaMemcpy(runs, c->d_stop->runs, sizeof(runs), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "reading the stop control: %s", cudaGetErrorString(e));
        for (int l = 0; l < c->levels; ++l) out_host[l] = runs[l];
    } else {
        for (int l = 0; l < c->levels; ++l) out_host[l] = c->runs_host[l];
    }
    return DISC_OK;
}

disc_status disc_set_mask(disc_ctx* c, int enable, float hu0, float a_min, float a_max, int fill_radius, float h,
                          int max_fill_passes) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    if (!enable) { c->mask_on = 0; return DISC_OK; }
    DISC_NEED(c, hu0 == hu0 && a_min == a_min && a_max == a_max && h == h, "NaN parameter");
    DISC_NEED(c, a_min < 0.f || a_max >= a_min, "a_max < a_min");
    DISC_NEED(c, fill_radius >= 1 && fill_radius <= 8, "fill_radius must be in 1..8");
    DISC_NEED(c, h > 0.f, "h <= 0");
    DISC_NEED(c, max_fill_passes >= 1 && max_fill_passes <= 254, "max_fill_passes must be in 1..254");
    DISC_TRY(alloc_ab(c));
    DISC_TRY(fill_grid_for(c, &c->fill_grid));
    c->mask_on = 1;
    c->mask_hu0 = hu0 >= 0.f ? hu0 : -1.f;
    c->mask_a_min = a_min >= 0.f ? a_min : -1.f;
    c->mask_a_max = a_min >= 0.f ? a_max : -1.f;
    c->fill_radius = fill_radius; c->fill_h = h; c->max_fill_passes = max_fill_passes;
    // the given parameters go to the device-side control block now, so that the fine-grained calls can be used without
    // disc_mask_params / disc_register; the derived ones are (re)computed there by those two
    MaskCtl h0;
    std::memset(&h0, 0, sizeof(h0));
    h0.hu0 = hu0 >= 0.f ? hu0 : 0.f;
    h0.a_m = 1.f;
    h0.a_min = a_min >= 0.f ? a_min : 0.5f;
    h0.a_max = a_min >= 0.f ? a_max : 1.5f;
    if (cudaMemcpy(c->d_mask, &h0, sizeof(h0), cudaMemcpyHostToDevice) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "cudaMemcpy (mask parameters) failed");
    return DISC_OK;
}

disc_status disc_mask_params(disc_ctx* c, const float* ct, const float* cbct, float out_host[5], void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, c->mask_on, "the mask is off (disc_set_mask)");
    DISC_NEED(c, ct && cbct && out_host, "NULL pointer");
    cudaStream_t st = (cudaStream_t)stream;
    DISC_TRY(mask_parameters(c, ct, cbct, st));
    MaskCtl h;
    cudaError_t e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpy(&h, c->d_mask, sizeof(h), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "reading the mask parameters: %s", cudaGetErrorString(e));
    out_host[0] = (float)h.delta_hu; out_host[1] = h.hu0; out_host[2] = h.a_m; out_host[3] = h.a_min; out_host[4] = h.a_max;
    return DISC_OK;
}

disc_status disc_get_ab(disc_ctx* c, int level, float* out_a, float* out_b, unsigned char* out_xi, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, c->d_mask, "neither the mask nor the diagnostics are on");
    const Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    if (out_a) e = cudaMemcpyAsync(out_a, L.A, L.N * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && out_b) e = cudaMemcpyAsync(out_b, L.B, L.N * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess && out_xi) e = cudaMemcpyAsync(out_xi, L.xi, L.N, cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "copy failed: %s", cudaGetErrorString(e));
    return DISC_OK;
}

disc_status disc_set_diagnostics(disc_ctx* c, int enable) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    if (enable) DISC_TRY(alloc_ab(c));
    c->diag_on = enable ? 1 : 0;
    return DISC_OK;
}

disc_status disc_get_diagnostics(disc_ctx* c, double* mean_a_host, double* mean_b_host) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, c->diag_on && c->d_mean_a, "the diagnostics are off (disc_set_diagnostics)");
    DISC_NEED(c, mean_a_host && mean_b_host, "NULL pointer");
    const size_t nd = (size_t)c->levels * (c->iters > 0 ? c->iters : 1) * sizeof(double);
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemcpy(mean_a_host, c->d_mean_a, nd, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(mean_b_host, c->d_mean_b, nd, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "reading the diagnostics: %s", cudaGetErrorString(e));
    return DISC_OK;
}

disc_status disc_warp(disc_ctx* c, int level, const float* moving, const float* disp, float* out, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, moving && disp && out, "NULL pointer");
    return launch_warp(c, c->lv[level], moving, disp, out, (cudaStream_t)stream);
}

disc_status disc_correct_intensity(disc_ctx* c, int level, const float* cbct, const float* ct_warped,
                                   float* out_corrected, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, cbct && ct_warped && out_corrected, "NULL pointer");
    Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    if (c->mask_on) {   // Eqs. (5)-(10) with the mask parameters the context holds (disc_set_mask / disc_mask_params)
        DISC_TRY(cache_cbct_moments(c, L, cbct, st));
        return correct_ab(c, L, cbct, ct_warped, out_corrected, true, -1, kNoCtl, st);
    }
    DISC_TRY(launch_moments<kModeZscore>(c, L, cbct, nullptr, L.zhat, nullptr, kNoCtl, st));
    return launch_moments<kModeCorrect>(c, L, ct_warped, L.zhat, out_corrected, nullptr, kNoCtl, st);
}

disc_status disc_demons_step(disc_ctx* c, int level, const float* m_warped, const float* s_corrected,
                             float* disp_inout, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, m_warped && s_corrected && disp_inout, "NULL pointer");
    Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    DISC_TRY(launch_force_gxy(c, true, L, m_warped, s_corrected, disp_inout, L.scratch, kNoCtl, st));
    return launch_gz_warp<false>(c, L, L.scratch, disp_inout, nullptr, nullptr, kNoCtl, st);
}

disc_status disc_iterate(disc_ctx* c, int level, const float* ct, const float* cbct, float* disp_inout,
                         int n_iters, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, ct && cbct && disp_inout, "NULL pointer");
    DISC_NEED(c, n_iters >= 0, "n_iters < 0");
    Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    // only this level runs: the counts of the others read 0
    for (int l = 0; l < DISC_MAX_LEVELS; ++l) c->runs_host[l] = 0;
    if (c->stop_eps >= 0.f && cudaMemsetAsync(c->d_stop->runs, 0, sizeof(c->d_stop->runs), st) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "cudaMemsetAsync failed");
    DISC_TRY(clear_diagnostics(c, st));
    if (!c->mask_on) DISC_TRY(launch_moments<kModeZscore>(c, L, cbct, nullptr, L.zhat, nullptr, kNoCtl, st));
    if (ab_path(c)) DISC_TRY(cache_cbct_moments(c, L, cbct, st));
    DISC_TRY(launch_warp(c, L, ct, disp_inout, L.m, st));
    return iterate_level(c, L, ct, cbct, disp_inout, n_iters, true, st);
}

disc_status disc_profile_iteration(disc_ctx* c, int level, const float* ct, const float* cbct, float* disp_inout,
                                   int n_iters, float ms_per_kernel[3], void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, ct && cbct && disp_inout && ms_per_kernel, "NULL pointer");
    DISC_NEED(c, n_iters >= 1 && n_iters <= 4096, "n_iters must be in 1..4096");
    Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    const int ne = 4 * n_iters;
    cudaEvent_t* ev = new (std::nothrow) cudaEvent_t[ne];
    if (!ev) return fail(c, DISC_ERR_ALLOC, "out of host memory");
    for (int i = 0; i < ne; ++i)
        if (cudaEventCreate(&ev[i]) != cudaSuccess) {
            for (int j = 0; j < i; ++j) cudaEventDestroy(ev[j]);
            delete[] ev;
            return fail(c, DISC_ERR_CUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
        }
    disc_status rc = launch_moments<kModeZscore>(c, L, cbct, nullptr, L.zhat, nullptr, kNoCtl, st);
    if (rc == DISC_OK) rc = launch_warp(c, L, ct, disp_inout, L.m, st);
    for (int k = 0; k < n_iters && rc == DISC_OK; ++k) {
        cudaEventRecord(ev[4 * k + 0], st);
        rc = launch_moments<kModeCorrect>(c, L, L.m, L.zhat, L.sp, nullptr, kNoCtl, st);
        cudaEventRecord(ev[4 * k + 1], st);
        if (rc == DISC_OK) rc = launch_force_gxy(c, true, L, L.m, L.sp, disp_inout, L.scratch, kNoCtl, st);
        cudaEventRecord(ev[4 * k + 2], st);
        if (rc == DISC_OK) rc = launch_gz_warp<true>(c, L, L.scratch, disp_inout, ct, L.m, kNoCtl, st);
        cudaEventRecord(ev[4 * k + 3], st);
    }
    cudaError_t e = cudaStreamSynchronize(st);
    if (rc == DISC_OK && e != cudaSuccess) rc = fail(c, DISC_ERR_CUDA, "stream sync: %s", cudaGetErrorString(e));
    if (rc == DISC_OK) {
        double acc[3] = {0, 0, 0};
        for (int k = 0; k < n_iters; ++k)
            for (int j = 0; j < 3; ++j) {
                float ms = 0.f;
                cudaEventElapsedTime(&ms, ev[4 * k + j], ev[4 * k + j + 1]);
                acc[j] += ms;
            }
        for (int j = 0; j < 3; ++j) ms_per_kernel[j] = (float)(acc[j] / n_iters);
    }
    for (int i = 0; i < ne; ++i) cudaEventDestroy(ev[i]);
    delete[] ev;
    return rc;
}

disc_status disc_register(disc_ctx* c, const float* ct, const float* cbct, float* out_disp,
                          float* out_corrected_cbct, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, ct && cbct && out_disp, "NULL pointer");
    cudaStream_t st = (cudaStream_t)stream;
    const int nl = c->levels;
    // pyramids
    const float* pct[DISC_MAX_LEVELS];
    const float* pcb[DISC_MAX_LEVELS];
    pct[0] = ct; pcb[0] = cbct;
    DISC_TRY(clear_diagnostics(c, st));
    if (c->mask_on) {
        // A1 "Globally adjust the intensity of CBCT" and the mask parameters
        DISC_TRY(mask_parameters(c, ct, cbct, st));
        k_shift<<<reduce_grid(c->lv[0].N), 256, 0, st>>>(cbct, c->cbct_shift, c->lv[0].N, c->d_mask);
        DISC_TRY(check_launch(c, "k_shift"));
        pcb[0] = c->cbct_shift;
    }
    for (int l = 1; l < nl; ++l) {
        DISC_TRY(launch_downsample(c, c->lv[l - 1], pct[l - 1], c->lv[l].ct, st));
        DISC_TRY(launch_downsample(c, c->lv[l - 1], pcb[l - 1], c->lv[l].cbct, st));
        pct[l] = c->lv[l].ct; pcb[l] = c->lv[l].cbct;
    }
    for (int l = nl - 1; l >= 0; --l) {
        Level& L = c->lv[l];
        float* r = l == 0 ? out_disp : L.disp;
        if (l == nl - 1) {
            if (cudaMemsetAsync(r, 0, 3 * L.N * sizeof(float), st) != cudaSuccess)
                return fail(c, DISC_ERR_CUDA, "cudaMemsetAsync failed");
        } else {
            DISC_TRY(launch_upsample(c, c->lv[l + 1], c->lv[l + 1].disp, r, st));
        }
        if (!c->mask_on) DISC_TRY(launch_moments<kModeZscore>(c, L, pcb[l], nullptr, L.zhat, nullptr, kNoCtl, st));
        if (ab_path(c)) DISC_TRY(cache_cbct_moments(c, L, pcb[l], st));
        DISC_TRY(launch_warp(c, L, pct[l], r, L.m, st));
        const bool need_m = (l == 0 && out_corrected_cbct != nullptr);
        DISC_TRY(iterate_level(c, L, pct[l], pcb[l], r, c->iters, need_m, st));
        if (need_m) {                                                                  // reading A12
            if (c->mask_on) DISC_TRY(correct_ab(c, L, pcb[l], L.m, out_corrected_cbct, true, -1, kNoCtl, st));
            else DISC_TRY(launch_moments<kModeCorrect>(c, L, L.m, L.zhat, out_corrected_cbct, nullptr, kNoCtl, st));
        }
    }
    return DISC_OK;
}

disc_status disc_register_host(disc_ctx* c, const float* ct_host, const float* cbct_host, float* out_disp_host,
                               float* out_corr_host, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, ct_host && cbct_host && out_disp_host, "NULL pointer");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t b = c->lv[0].N * sizeof(float);
    if (!c->h2d_ct) {
        bool ok = cudaMalloc(&c->h2d_ct, b) == cudaSuccess && cudaMalloc(&c->h2d_cbct, b) == cudaSuccess &&
                  cudaMalloc(&c->d_out_disp, 3 * b) == cudaSuccess && cudaMalloc(&c->d_out_corr, b) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return fail(c, DISC_ERR_ALLOC, "cudaMalloc (host staging) failed"); }
    }
    if (cudaMemcpyAsync(c->h2d_ct, ct_host, b, cudaMemcpyHostToDevice, st) != cudaSuccess ||
        cudaMemcpyAsync(c->h2d_cbct, cbct_host, b, cudaMemcpyHostToDevice, st) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "H2D copy failed: %s", cudaGetErrorString(cudaGetLastError()));
    DISC_TRY(disc_register(c, c->h2d_ct, c->h2d_cbct, c->d_out_disp, out_corr_host ? c->d_out_corr : nullptr, stream));
    if (cudaMemcpyAsync(out_disp_host, c->d_out_disp, 3 * b, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "D2H copy failed");
    if (out_corr_host && cudaMemcpyAsync(out_corr_host, c->d_out_corr, b, cudaMemcpyDeviceToHost, st) != cudaSuccess)
        return fail(c, DISC_ERR_CUDA, "D2H copy failed");
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(c, DISC_ERR_CUDA, "stream sync: %s", cudaGetErrorString(e));
    return DISC_OK;
}

disc_status disc_box_moments(disc_ctx* c, int level, const float* vol, float* mean, float* var, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, vol && mean && var, "NULL pointer");
    return launch_moments<kModeMoments>(c, c->lv[level], vol, nullptr, mean, var, kNoCtl, (cudaStream_t)stream);
}

disc_status disc_force_update(disc_ctx* c, int level, const float* m, const float* s, float* disp_inout, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, m && s && disp_inout, "NULL pointer");
    const Level& L = c->lv[level];
    launch_force_update(c->force_mode, m, s, disp_inout, L.nx, L.ny, L.nz, DISC_EPS_DEN, (cudaStream_t)stream);
    return check_launch(c, "k_force_update");
}

disc_status disc_smooth_field(disc_ctx* c, int level, float* disp_inout, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_ok(c, level), "level out of range");
    DISC_NEED(c, disp_inout, "NULL pointer");
    Level& L = c->lv[level];
    cudaStream_t st = (cudaStream_t)stream;
    DISC_TRY(launch_force_gxy(c, false, L, nullptr, nullptr, disp_inout, L.scratch, kNoCtl, st));
    return launch_gz_warp<false>(c, L, L.scratch, disp_inout, nullptr, nullptr, kNoCtl, st);
}

disc_status disc_downsample(disc_ctx* c, int level_from, const float* vol, float* out, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_from >= 0 && level_from + 1 < c->levels, "level_from out of range");
    DISC_NEED(c, vol && out, "NULL pointer");
    return launch_downsample(c, c->lv[level_from], vol, out, (cudaStream_t)stream);
}

disc_status disc_upsample_field(disc_ctx* c, int level_from, const float* disp, float* out, void* stream) {
    if (!c) return DISC_ERR_INVALID_ARG;
    DISC_TRY(check_device(c));
    DISC_NEED(c, level_from >= 1 && level_from < c->levels, "level_from out of range");
    DISC_NEED(c, disp && out, "NULL pointer");
    return launch_upsample(c, c->lv[level_from], disp, out, (cudaStream_t)stream);
}

}  // extern "C"

// =====================================================================================
// disc_smooth_field_noalloc: Gaussian regularisation for callers that may not allocate device memory (include/disc.h).
// The buffer between the x,y pass and the z pass is this fixed array instead of a context's cudaMalloc'ed scratch.
// In HOST code the name below is only a handle for cudaGetSymbolAddress: it is not a device address and must never be
// handed to a kernel; the launches get the address looked up once per device in noalloc_device().
static __device__ __align__(256) float g_noalloc_scratch[3 * (size_t)DISC_NOALLOC_MAX_VOXELS];

namespace {

struct NoAllocDev {
    bool ready;
    float* scratch;   // device address of g_noalloc_scratch on this device
    DevInfo di;
};
NoAllocDev g_noalloc_dev[kMaxDevices];   // zero-initialised; guarded by g_noalloc_mutex
std::mutex g_noalloc_mutex;

// Per-device set-up, done by the first call on the current device: no allocation, only queries.
disc_status noalloc_device(const NoAllocDev** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, DISC_ERR_UNSUPPORTED, "device ordinal %d >= %d", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoAllocDev& d = g_noalloc_dev[dev];
    if (!d.ready) {
        int major = 0, n_sm = 0;
        e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
        if (major != 10) return fail(nullptr, DISC_ERR_UNSUPPORTED, "device compute capability %d.x, this library is sm_100a only", major);
        float* p = nullptr;
        e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);   // the array's address on the CURRENT device
        if (e != cudaSuccess || !p)
            return fail(nullptr, DISC_ERR_CUDA, "cudaGetSymbolAddress(built-in scratch) on device %d: %s", dev, cudaGetErrorString(e));
        d.scratch = p;
        d.di.dev = dev;
        d.di.n_sm = n_sm;
        d.ready = true;
    }
    *out = &d;
    return DISC_OK;
}

}  // namespace

extern "C" disc_status disc_smooth_field_noalloc(const int dims[3], float sigma_smooth, float* disp_inout, void* stream) {
    if (!dims || !disp_inout) return fail(nullptr, DISC_ERR_INVALID_ARG, "dims or disp_inout is NULL");
    for (int i = 0; i < 3; ++i)
        if (dims[i] < 1) return fail(nullptr, DISC_ERR_INVALID_ARG, "dims[%d] < 1", i);
    const unsigned long long N = (unsigned long long)dims[0] * (unsigned long long)dims[1] * (unsigned long long)dims[2];
    if ((unsigned long long)dims[0] * dims[1] > (unsigned long long)DISC_NOALLOC_MAX_VOXELS || N > (unsigned long long)DISC_NOALLOC_MAX_VOXELS)
        return fail(nullptr, DISC_ERR_INVALID_ARG,
                    "%d x %d x %d voxels exceed the built-in scratch of disc_smooth_field_noalloc (DISC_NOALLOC_MAX_VOXELS = %d): "
                    "use a context and disc_smooth_field", dims[0], dims[1], dims[2], (int)DISC_NOALLOC_MAX_VOXELS);
    if (!(sigma_smooth > 0.f)) return fail(nullptr, DISC_ERR_INVALID_ARG, "sigma_smooth <= 0");
    const int K = (int)std::ceil(3.0 * (double)sigma_smooth);
    if (K > DISC_MAX_GAUSS_RADIUS)
        return fail(nullptr, DISC_ERR_UNSUPPORTED, "Gaussian radius ceil(3 sigma) = %d > %d", K, DISC_MAX_GAUSS_RADIUS);
    const NoAllocDev* d = nullptr;
    DISC_TRY(noalloc_device(&d));
    // taps exactly as disc_create forms them: fp64, normalised to sum 1, then rounded to fp32 (reading A10)
    GaussTaps taps;
    std::memset(&taps, 0, sizeof(taps));
    {
        double w[kMaxGaussTaps], sum = 0.0;
        for (int i = -K; i <= K; ++i) { w[i + K] = std::exp(-(double)(i * i) / (2.0 * (double)sigma_smooth * (double)sigma_smooth)); sum += w[i + K]; }
        for (int i = 0; i < 2 * K + 1; ++i) taps.w[i] = (float)(w[i] / sum);
    }
    cudaStream_t st = (cudaStream_t)stream;
    const StopReq no_stop = {nullptr, 0, 0.f};
    // x,y passes: disp_inout -> built-in array (all 3 N floats written); z pass: built-in array -> disp_inout
    if (!launch_force_gxy_any(d->di, K, 0, nullptr, nullptr, disp_inout, d->scratch, dims[0], dims[1], dims[2], DISC_EPS_DEN, taps,
                              kNoCtl, no_stop, st))
        return fail(nullptr, DISC_ERR_UNSUPPORTED, "Gaussian radius %d unsupported", K);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "k_force_gxy (no-alloc): %s", cudaGetErrorString(e));
    if (!launch_gz_warp_any(d->di, K, false, d->scratch, disp_inout, nullptr, nullptr, dims[0], dims[1], dims[2], taps, kNoCtl, st))
        return fail(nullptr, DISC_ERR_UNSUPPORTED, "Gaussian radius %d unsupported", K);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, DISC_ERR_CUDA, "k_gz_warp (no-alloc): %s", cudaGetErrorString(e));
    return DISC_OK;
}
