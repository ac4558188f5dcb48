// launch.h -- internal C++ interface between disc_api.cu and the separately compiled kernel
// translation units (moments_tu.cu, field_tu.cu; each is built several times for a range of R / K so
// that the template instances compile in parallel).  The *_any functions return false when no
// instance exists for the requested radius.
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace disc {

constexpr int kMomTX = 32, kMomTY = 16;  // (x,y) tile of the plain-load moments kernel
constexpr int kMomMaxRTile32 = 7;        // largest R whose z ring fits tensor memory with the 32x32 tile (moments_v2.cuh)

enum MomentsMode {
    kModeMoments = 0,  // out0 = mean, out1 = var                                   (disc_box_moments)
    kModeZscore = 1,   // out0 = (v - mu)/sigma, 0 where var <= eps_var              (cached per level from the CBCT)
    kModeCorrect = 2   // out0 = sigma_m * aux + mu_m  (aux = CBCT z-score)          (per-iteration correction)
};


// Stop control handed to every kernel launched from this host thread ({nullptr, 0}: criterion off); set by
// disc_api.cu around the launches of one iteration.
extern thread_local IterCtl g_iter_ctl;
// sum|dr|, sum|r| of the iteration -> l^(k), criterion check in the last block (field.cuh k_force_norms)
void launch_force_norms(int force, const float* m, const float* s, const float* r, int nx, int ny, int nz, float eps_den,
                        StopCtl* ctl, int iter, float stop_eps, int n_sm, cudaStream_t st);
void launch_stop_reset(StopCtl* ctl, cudaStream_t st);
void launch_stop_record(StopCtl* ctl, int level, int n_iters, cudaStream_t st);

bool launch_moments_any(int R, int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx,
                        int ny, int nz, int zchunk, float eps_var, cudaStream_t st);
// force = 0 none (plain smoothing), 1 Thirion / passive, 2 double (ForceMode in field.cuh)
bool launch_force_gxy_any(int K, int force, int txb, const float* m, const float* s, const float* rin, float* rout,
                          int nx, int ny, int nz, int yseg, float eps_den, const GaussTaps& taps, cudaStream_t st);
bool launch_gz_warp_any(int K, bool warp, const float* rin, float* rout, const float* moving, float* mout, int nx,
                        int ny, int nz, int zchunk, const GaussTaps& taps, cudaStream_t st);
void launch_force_update(int force, const float* m, const float* s, float* r, int nx, int ny, int nz, float eps_den,
                         cudaStream_t st);
void launch_warp_kernel(const float* moving, const float* r, float* out, int nx, int ny, int nz, cudaStream_t st);

// per-translation-unit entry points (defined by moments_tu.cu / field_tu.cu with -DDISC_TU=n)
#define DISC_DECL_TU(n)                                                                                                  \
    bool launch_moments_tu##n(int R, int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx,     \
                              int ny, int nz, int zchunk, float eps_var, cudaStream_t st);                              \
    bool launch_force_gxy_tu##n(int K, int force, int txb, const float* m, const float* s, const float* rin,           \
                                float* rout, int nx, int ny, int nz, int yseg, float eps_den, const GaussTaps& taps,    \
                                cudaStream_t st);                                                                        \
    bool launch_gz_warp_tu##n(int K, bool warp, const float* rin, float* rout, const float* moving, float* mout,        \
                              int nx, int ny, int nz, int zchunk, const GaussTaps& taps, cudaStream_t st);
DISC_DECL_TU(0) DISC_DECL_TU(1) DISC_DECL_TU(2) DISC_DECL_TU(3)
#undef DISC_DECL_TU

}  // namespace disc
