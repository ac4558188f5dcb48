/*
 * disc.h -- C-ABI of the B200-native DISC hot path (CT -> CBCT demons registration with
 * simultaneous patch-moment intensity correction; Zhen et al., arxiv 1204.6295).
 * Citations are PAPER.md:LINE of that paper's text; "reading Ax" refers to DESIGN.md.
 *
 * Plain C: no C++ types, no exceptions, no torch types.  One GPU (sm_100a), one context per
 * stream at a time.  Nothing here runs on the CPU: without a CUDA device every compute call
 * returns DISC_ERR_CUDA / DISC_ERR_UNSUPPORTED -- there is no fallback.
 *
 * Conventions
 *   dims = (nx, ny, nz), x fastest: idx = (z*ny + y)*nx + x.  All volumes are float32.
 *   A displacement field is planar: disp[c*N + idx], c = 0,1,2 <-> x,y,z, in VOXEL units of the
 *   level it lives on (reading A13).  Level 0 is the finest; level l has dims >> l.
 *   The moving image is the CT, the static image the CBCT.  The field is a
 *   pull-back: warped(x) = ct(x + r(x)), so for cbct(x) = ct(x + u(x)) the
 *   registration returns r ~ u (reading A1).
 *   Unless a parameter says HOST, every pointer is a DEVICE pointer owned by the caller; the
 *   library never frees or keeps it after the call's work has run.  Inputs are never written.
 *   Outputs must not alias inputs except where a parameter is named *_inout.
 *   `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Every call only
 *   enqueues work on it and returns; the library never synchronises (except disc_destroy and
 *   disc_register_host, which say so).  Scratch lives in the context, so one context must not
 *   be used from two streams concurrently.
 *   Errors: argument errors are detected before any launch and return DISC_ERR_INVALID_ARG;
 *   launch/runtime failures return DISC_ERR_CUDA; disc_last_error() gives a message.
 */
#ifndef DISC_H
#define DISC_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct disc_ctx disc_ctx; /* opaque, owned by the library */

typedef enum {
    DISC_OK = 0,
    DISC_ERR_INVALID_ARG = 1,
    DISC_ERR_UNSUPPORTED = 2, /* no sm_100 device, patch radius > 12 or Rx != Ry, Gaussian radius > 12 */
    DISC_ERR_ALLOC = 3,
    DISC_ERR_CUDA = 4
} disc_status;

/* Limits of this build. */
#define DISC_MAX_PATCH_RADIUS 12
#define DISC_MAX_GAUSS_RADIUS 12 /* ceil(3*sigma) <= 12, i.e. sigma <= 4 */
#define DISC_MAX_LEVELS 8

/* Regularisers (readings A5, A7): a = 0 where var_s <= DISC_EPS_VAR [HU^2];
 * force denominator |g|^2 + d^2 + DISC_EPS_DEN [HU^2]. */
#define DISC_EPS_VAR 1e-6f
#define DISC_EPS_DEN 1e-3f

/*
 * disc_create -- problem statement of the paper (Alg. A1 :175-198).
 *   dims          (nx, ny, nz) of level 0, each >= 1 and divisible by 2^(levels-1).   HOST
 *   spacing       voxel size in mm, each > 0.  Validated and stored; the hot path works in voxel
 *                 units (Eq. (1) has no spacing term; reading A13).          HOST
 *   patch_radius  R >= 0; the patch is the cube of side 2R+1 truncated to the volume (PAPER.md:87-89,
 *                 reading A4), the same R in voxels at every level.
 *   sigma_smooth  Gaussian sigma in voxels, > 0; support K = ceil(3 sigma), replicate border (A10).
 *   levels        pyramid levels >= 1, factor 2 per level in all three axes (A9).
 *   iters         iterations per level >= 0 (fixed count instead of the stopping test, A14).
 * Allocates all scratch (pyramid copies, warped CT, corrected CBCT, cached CBCT patch z-score,
 * second field buffer) on the current CUDA device.  Returns DISC_ERR_UNSUPPORTED if the current
 * device is not compute capability 10.x.
 */
disc_status disc_create(disc_ctx** out, const int dims[3], const float spacing[3], int patch_radius,
                        float sigma_smooth, int levels, int iters);

/*
 * disc_create_ex -- the same with the clinical geometry of the paper: a non-cubic patch and a pyramid
 * that need not halve every axis.
 *   patch_radius    (Rx, Ry, Rz) >= 0, HOST: the patch is the box of side 2R_c + 1 along axis c.  The paper's patches are
 *                   3x3x3 ... 25x25x7, i.e. radii up to (12, 12, 3); all have Rx == Ry, and that is
 *                   what this build supports: Rx != Ry, or a radius > DISC_MAX_PATCH_RADIUS -> DISC_ERR_UNSUPPORTED.
 *   pyramid_factor  (fx, fy, fz), each 1 or 2, HOST: level l has dims[c] / f_c^l voxels along axis c (each must divide).
 *                   The paper's clinical volumes (256x256x68 at 0.94x0.94x2.5 mm) were down-sampled in the transverse
 *                   plane only: factor (2, 2, 1).  Down: block mean over fx*fy*fz voxels; up: trilinear at
 *                   i/2 - 1/4 along the halved axes, identity along the others; component c of the field is scaled by
 *                   f_c, because it is in voxel units of its own axis (reading A9).
 *   spacing         recorded, never used by the iteration: Eq. (1) has no spacing term and the paper runs
 *                   its anisotropic volumes with the same formula, so gradients are per voxel, the Gaussian sigma is in
 *                   voxels on every axis and the field is in voxels of its own axis (reading A13).
 * Everything else as disc_create, which is disc_create_ex with (R, R, R) and (2, 2, 2).
 */
disc_status disc_create_ex(disc_ctx** out, const int dims[3], const float spacing[3], const int patch_radius[3],
                           float sigma_smooth, int levels, int iters, const int pyramid_factor[3]);

/* Synchronises the device, frees the context and its scratch.  NULL is allowed. */
void disc_destroy(disc_ctx* ctx);

/* Message of the last error of this context (ctx == NULL: of the calling thread's last failed disc_create or
 * disc_smooth_field_noalloc).  The string is owned by the library and valid until the next call on the same context. */
const char* disc_last_error(const disc_ctx* ctx);

/* Number of CUDA kernels this context has launched so far (bench.py's gpu_launches). */
unsigned long long disc_launch_count(const disc_ctx* ctx);

/* Force variant used by disc_force_update, disc_demons_step, disc_iterate and disc_register from now on.
 *   DISC_FORCE_THIRION (default): the passive force, first term of Eq. (1) with the corrected CBCT s'
 *                      (north_star (c); reading A2):  dr = d grad(s') / (|grad s'|^2 + d^2 + eps)
 *   DISC_FORCE_DOUBLE: both terms of Eq. (1), the paper's double-force demons:
 *                      dr = d grad(s') / (|grad s'|^2 + d^2 + eps) + d grad(m) / (|grad m|^2 + d^2 + eps)
 * with d = s' - m (sign: reading A1), m the deformed CT of the current iteration, both gradients central
 * differences with clamped indices (A8), eps = DISC_EPS_DEN in both denominators (A7).
 * Host-side state only, no launch.  Any other mode -> DISC_ERR_INVALID_ARG. */
#define DISC_FORCE_THIRION 1
#define DISC_FORCE_DOUBLE 2
disc_status disc_set_force(disc_ctx* ctx, int mode);

/* Stopping criterion of the paper (Alg. A1 :187), used by disc_iterate and disc_register
 * from now on.  eps >= 0 enables it, eps < 0 disables it (default: fixed iteration counts, north_star).
 * Inside a level, every iteration k = 0,1,.. evaluates  l(k) = sum_x |dr(x)| / sum_x |r(x)|  from the increment that
 * iteration's force is about to add and the field before the update (Euclidean norm per voxel, reading A16;
 * l = +inf while the field is zero).  The first iteration k >= 10 with  l(k-10) - l(k) <= eps  is completed and is the
 * level's last; `iters` of disc_create stays the per-level maximum.  (The text's condition is followed; Alg. A1's
 * `while` prints it inverted.)  The paper's value is eps = 1e-4.
 * The test runs on the device (the paper's "comparison kernel"): the force kernel of the iteration adds the two sums up
 * while it evaluates the force, and its last block sets a flag; the kernels of the remaining iterations are still
 * enqueued but return at once, so there is no host synchronisation.  Host-side state only, no launch. */
disc_status disc_set_stop(disc_ctx* ctx, float eps);

/*
 * Reliability mask and interpolation / extrapolation of a, b (Alg. A1 step 2).
 * With enable != 0, disc_register, disc_iterate and disc_correct_intensity replace the direct correction by
 *   a = STD(M)/STD(S), b = E(M) - a E(S)                                   Eqs. (5)-(6)
 *   xi = 1 where |I_m^(k) - I_s| > HU_0 or a < a_min or a > a_max          Eq. (7),
 *   a = b = 0 where xi = 1, then, repeated until nothing is left: every voxel with xi = 1 takes the average of the
 *   a, b of the available voxels (xi = 0, or filled by an earlier pass) in the cube T of radius fill_radius around
 *   it, weighted by w_i = exp(-(I_s(i) - I_s(x))^2 / h^2)                  Eqs. (8)-(10)
 *   I'_s = a I_s + b
 * and disc_register first shifts the CBCT by Delta HU = mean(CT) - mean(CBCT) (Alg. A1 "globally adjust").
 *   hu0             HU_0 [HU]; < 0: 2 |Delta HU|
 *   a_min, a_max    bounds of a; a_min < 0: 0.5 a_m and 1.5 a_m with a_m the median of A computed before the DIR from the
 *                   full-resolution images.  Reading A17: the median runs over the voxels where both patch
 *                   variances exceed DISC_EPS_VAR and is the lower median.
 *   fill_radius     radius of T in voxels, 1..8 (its size is lost from the text: "a relative small size")
 *   h               Eq. (10) [HU], > 0 (never given in the text)
 *   max_fill_passes 1..254; readings A18: a pass reads only what was available when it started; the weights are
 *                   normalised by the largest one (same quotient, no underflow); passes stop when nothing is left, when a
 *                   pass fills nothing or after max_fill_passes, and what is then still unfilled keeps a = b = 0.
 * Everything is decided on the device (parameters, "anything left"): the iteration gets no host synchronisation.
 * The passes of one correction run in ONE cooperative launch over a compacted list of the xi = 1 voxels (grid barrier between
 * passes), so a correction with few masked voxels costs little more than the unmasked one.
 * disc_set_mask itself allocates 5 N words + N bytes per level on first use and copies the given parameters to the
 * device (a blocking cudaMemcpy of a few bytes); until disc_mask_params or disc_register has derived them, a parameter
 * given as < 0 reads HU_0 = 0, a_min = 0.5, a_max = 1.5.  enable == 0 switches back.
 */
disc_status disc_set_mask(disc_ctx* ctx, int enable, float hu0, float a_min, float a_max, int fill_radius, float h,
                          int max_fill_passes);

/* The parameters the mask derives from the two full-resolution images (device pointers), computed now and kept for
 * later fine-grained calls: out_host = {Delta HU, HU_0, a_m, a_min, a_max} (HOST, 5 floats).  SYNCHRONISES `stream`. */
disc_status disc_mask_params(disc_ctx* ctx, const float* ct, const float* cbct, float out_host[5], void* stream);

/* a(x), b(x) and the mask of `level` as the last correction left them -- after an early stop (disc_set_stop) those of the
 * last iteration run -- (device buffers, each may be NULL): out_a, out_b [N_level] floats, out_xi [N_level] bytes --
 * 0: xi = 0, k in 1..254: xi = 1, filled in pass k, 255: xi = 1, never filled. */
disc_status disc_get_ab(disc_ctx* ctx, int level, float* out_a, float* out_b, unsigned char* out_xi, void* stream);

/* Fig. 9 (e), (f) of the paper: the averages of a and of b over all voxels in every iteration of
 * disc_register.  disc_get_diagnostics SYNCHRONISES the device and writes levels*iters doubles each (HOST), level-major
 * from the COARSEST level, `iters` slots per level; the slot of an iteration the last disc_register / disc_iterate did not
 * run (stopping criterion tripped earlier, other level) reads NaN.  Without the mask this costs one more moments launch
 * per iteration. */
disc_status disc_set_diagnostics(disc_ctx* ctx, int enable);
disc_status disc_get_diagnostics(disc_ctx* ctx, double* mean_a_host, double* mean_b_host);

/* Iterations actually run per level by the last disc_register / disc_iterate on this context:
 * out_host[level], level = 0 .. levels-1 (HOST array of `levels` ints).  SYNCHRONISES the device when the
 * stopping criterion is enabled; without it the counts are the requested ones. */
disc_status disc_iterations_run(disc_ctx* ctx, int* out_host);

/* ---- the steps of one iteration, in execution order b -> a -> c+d (Alg. A1) ---- */

/* (b) out(x) = moving(x + disp(x)), trilinear, sample position clamped to the volume
 * ("update the moving image", kernel 5 :171; reading A11).
 * moving [N_level], disp [3*N_level], out [N_level]. */
disc_status disc_warp(disc_ctx* ctx, int level, const float* moving, const float* disp, float* out, void* stream);

/* (a) out = a*(cbct - mu_cbct) + mu_ct with a = STD(ct patch)/STD(cbct patch), patch moments over
 * the truncated cube of radius R (PAPER.md:95 Eq. 3, :117-119 Eqs. 5-6, :141; readings A4, A5):
 * a = 0 where var_cbct <= DISC_EPS_VAR.  cbct, ct_warped, out_corrected: [N_level]. */
disc_status disc_correct_intensity(disc_ctx* ctx, int level, const float* cbct, const float* ct_warped,
                                   float* out_corrected, void* stream);

/* (c)+(d) = Alg. A1 steps 4-6: disp += (s-m) grad s / (|grad s|^2 + (s-m)^2 + eps)
 * (Eq. 1 first term; readings A1, A2, A7, A8), then disp <- G_sigma * disp (A3, A10).
 * m_warped, s_corrected: [N_level]; disp_inout: [3*N_level], updated in place. */
disc_status disc_demons_step(disc_ctx* ctx, int level, const float* m_warped, const float* s_corrected,
                             float* disp_inout, void* stream);

/* The whole registration (Alg. A1, fixed `iters` per level): builds both pyramids
 * (2x2x2 means), r = 0 at the coarsest level, per level `iters` x {warp, correct, force+update,
 * smooth}, up-samples r between levels (x2 trilinear, values doubled), and finally
 * out_corrected_cbct = correct(cbct, warp(ct, out_disp)) (reading A12).
 * ct, cbct: [N_0]; out_disp: [3*N_0]; out_corrected_cbct: [N_0] or NULL. */
disc_status disc_register(disc_ctx* ctx, const float* ct, const float* cbct, float* out_disp,
                          float* out_corrected_cbct, void* stream);

/* Same as disc_register with HOST buffers (pageable or pinned): copies ct and cbct to the device,
 * registers, copies the results back and SYNCHRONISES `stream` before returning.
 * This is the end-to-end entry point bench.py times ("e2e"). */
disc_status disc_register_host(disc_ctx* ctx, const float* ct_host, const float* cbct_host, float* out_disp_host,
                               float* out_corrected_cbct_host, void* stream);

/* `n_iters` iterations of {correct, force+update, smooth, warp} at one level, starting from
 * disp_inout (the fused steady-state loop of disc_register; what bench.py times as iterations/s).
 * ct, cbct: [N_level] images of that level; disp_inout [3*N_level].  After the call the context's
 * warped-CT buffer holds warp(ct, disp_inout). */
disc_status disc_iterate(disc_ctx* ctx, int level, const float* ct, const float* cbct, float* disp_inout,
                         int n_iters, void* stream);

/* Measurement aid for bench.py's roofline object: runs `n_iters` iterations exactly as disc_iterate does, with a
 * CUDA event pair around every kernel on `stream`, SYNCHRONISES the stream and writes the mean duration in
 * milliseconds of each of the three per-iteration kernels to ms_per_kernel (HOST, 3 floats):
 * [0] moments+correct, [1] force+update+Gaussian x,y, [2] Gaussian z + warp. */
disc_status disc_profile_iteration(disc_ctx* ctx, int level, const float* ct, const float* cbct, float* disp_inout,
                                   int n_iters, float ms_per_kernel[3], void* stream);

/* ---- finer-grained exports (BASELINE.json config 5 per-kernel sweep, and tests) ---- */

/* Patch mean and population variance of `vol` over the truncated cube of radius R (Eq. 3, A4).
 * mean, var: [N_level] float32. */
disc_status disc_box_moments(disc_ctx* ctx, int level, const float* vol, float* mean, float* var, void* stream);

/* Step (c) alone: disp_inout += force(m, s). */
disc_status disc_force_update(disc_ctx* ctx, int level, const float* m, const float* s, float* disp_inout, void* stream);

/* Step (d) alone: disp_inout <- G_sigma * disp_inout. */
disc_status disc_smooth_field(disc_ctx* ctx, int level, float* disp_inout, void* stream);

/* Block mean from level_from to level_from+1 over the context's pyramid factor, 2x2x2 by default (
 * reading A9).  vol [N_level_from], out [N_level_from+1]. */
disc_status disc_downsample(disc_ctx* ctx, int level_from, const float* vol, float* out, void* stream);

/* Up-sampling of a field from level_from to level_from-1: trilinear at i/2 - 1/4 (clamped) with the value doubled
 * along every axis the pyramid halves (reading A9).  disp [3*N_level_from], out [3*N_level_from-1]. */
disc_status disc_upsample_field(disc_ctx* ctx, int level_from, const float* disp, float* out, void* stream);

/* ---- an entry point for callers that are not allowed to allocate device memory ---- */

/*
 * disc_smooth_field_noalloc -- step (d), disp_inout <- G_sigma * disp_inout (readings A3, A10), computed by
 * the same two kernels as disc_smooth_field and bit-identical to it, but WITHOUT a context and without any allocation.
 *
 * Who needs it.  Every other compute call needs a disc_ctx, and disc_create obtains the scratch of all kernels with
 * cudaMalloc.  Some hosts of this library cannot do that: an application that carves the GPU's memory up itself at
 * start-up and forbids library-side cudaMalloc, or a latency-bound treatment-room loop (re-regularising a field between
 * two beam deliveries) in which cudaMalloc / cudaFree are unacceptable because they synchronise the whole device and
 * stall the other streams.  For them the field buffer the x,y pass hands to the z pass (3 N floats) lives in a
 * fixed array inside libdisc.so instead of in a context.
 *
 *   dims          (nx, ny, nz), each >= 1, HOST.  nx*ny*nz must not exceed DISC_NOALLOC_MAX_VOXELS (the size of the
 *                 built-in array); a larger volume is rejected with DISC_ERR_INVALID_ARG and a message that names both
 *                 numbers -- use a context and disc_smooth_field for it.
 *   sigma_smooth  Gaussian sigma in voxels, > 0, ceil(3 sigma) <= DISC_MAX_GAUSS_RADIUS (else DISC_ERR_UNSUPPORTED).
 *   disp_inout    DEVICE, 3*nx*ny*nz floats, planar, owned by the caller, updated in place.
 *   stream        cudaStream_t of the CURRENT device; the call only enqueues two kernels on it and returns.
 *
 * Cost: the array is 3 * DISC_NOALLOC_MAX_VOXELS floats = 12 MiB of device memory, and every GPU on which this
 * library gets loaded keeps that much reserved until the process exits, whether or not this function is ever called.
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress), the device's compute
 * capability and SM count, and keeps them; that is host-side set-up, not an allocation, but it talks to the driver, so
 * make the first call on each device during start-up, before any stream capture is begun.  Later calls do no set-up.
 * Sharing: there is ONE array per device and every call on that device uses it.  Two calls whose kernels may overlap
 * on the GPU (different streams without an ordering between them, or two host threads) race on it and both results
 * are undefined; calls on one stream, or ordered by events, are fine.  The array keeps whatever the last call left in
 * it; nothing in it has to start at zero, because the x,y pass writes all 3 N floats before the z pass reads them.
 * Errors go to disc_last_error(NULL) of the calling thread.  This function calls no cudaMalloc, no cudaFree and no
 * library routine that allocates.
 */
#define DISC_NOALLOC_MAX_VOXELS (1 << 20) /* 128 x 128 x 64, config 2's finest level */
disc_status disc_smooth_field_noalloc(const int dims[3], float sigma_smooth, float* disp_inout, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* DISC_H */
