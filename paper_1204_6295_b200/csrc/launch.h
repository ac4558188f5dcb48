// launch.h -- internal C++ interface between disc_api.cu and the separately compiled kernel
// translation units (moments_tu.cu, field_tu.cu; each is built several times for a range of R / K so
// that the template instances compile in parallel).  The *_any functions return false when no
// instance exists for the requested radius.
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace disc {

constexpr int kMomTX = 32, kMomTY = 16;  // (x,y) tile of the plain-load moments kernel
constexpr int kMaxDevices = 64;          // per-device "attribute set" flags of the launchers

// What a launcher needs to know about the context's device (set in disc_create).
struct DevInfo {
    int dev;    // CUDA device ordinal the context lives on
    int n_sm;   // its multiprocessor count
};

enum MomentsMode {
    kModeMoments = 0,  // out0 = mean, out1 = var                                   (disc_box_moments)
    kModeZscore = 1,   // out0 = (v - mu)/sigma, 0 where var <= eps_var              (cached per level from the CBCT)
    kModeCorrect = 2   // out0 = sigma_m * aux + mu_m  (aux = CBCT z-score)          (per-iteration correction)
};

// The stopping criterion's request to the force kernel of iteration `iter` (ctl == nullptr: criterion off): the fused
// tile kernel adds sum|dr|, sum|r| up itself (block partials, last block decides); the plain-load fallback launches
// k_force_norms first.
struct StopReq {
    StopCtl* ctl;
    int iter;
    float eps;
};

// sum|dr|, sum|r| of the iteration -> l^(k), criterion check in the last block (field.cuh k_force_norms)
void launch_force_norms(int force, const float* m, const float* s, const float* r, int nx, int ny, int nz, float eps_den,
                        StopCtl* ctl, int iter, float stop_eps, int n_sm, cudaStream_t st);
void launch_stop_reset(StopCtl* ctl, cudaStream_t st);
void launch_stop_record(StopCtl* ctl, int level, int n_iters, cudaStream_t st);

// Every iteration kernel takes the stop control of its iteration by value ({nullptr, 0}: criterion off).
// rxy: patch radius along x and y, rz: along z; zchunk <= 0: the launcher picks the z chunk.
bool launch_moments_any(const DevInfo& di, int rxy, int rz, int mode, const float* vol, const float* aux, float* out0,
                        float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st);
// force = 0 none (plain smoothing), 1 Thirion / passive, 2 double (ForceMode in field.cuh)
bool launch_force_gxy_any(const DevInfo& di, int K, int force, const float* m, const float* s, const float* rin,
                          float* rout, int nx, int ny, int nz, float eps_den, const GaussTaps& taps, IterCtl ctl,
                          StopReq stop, cudaStream_t st);
bool launch_gz_warp_any(const DevInfo& di, int K, bool warp, const float* rin, float* rout, const float* moving,
                        float* mout, int nx, int ny, int nz, const GaussTaps& taps, IterCtl ctl, cudaStream_t st);
void launch_force_update(int force, const float* m, const float* s, float* r, int nx, int ny, int nz, float eps_den,
                         cudaStream_t st);
void launch_warp_kernel(const float* moving, const float* r, float* out, int nx, int ny, int nz, cudaStream_t st);

// per-translation-unit entry points (defined by moments_tu.cu / field_tu.cu with -DDISC_TU=n)
#define DISC_DECL_TU(n)                                                                                                  \
    bool launch_moments_tu##n(const DevInfo& di, int rxy, int rz, int mode, const float* vol, const float* aux,         \
                              float* out0, float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl,             \
                              cudaStream_t st);                                                                          \
    bool launch_force_gxy_tu##n(const DevInfo& di, int K, int force, const float* m, const float* s, const float* rin,  \
                                float* rout, int nx, int ny, int nz, float eps_den, const GaussTaps& taps, IterCtl ctl, \
                                StopReq stop, cudaStream_t st);                                                                        \
    bool launch_gz_warp_tu##n(const DevInfo& di, int K, bool warp, const float* rin, float* rout, const float* moving,  \
                              float* mout, int nx, int ny, int nz, const GaussTaps& taps, IterCtl ctl, cudaStream_t st);
DISC_DECL_TU(0) DISC_DECL_TU(1) DISC_DECL_TU(2) DISC_DECL_TU(3)
#undef DISC_DECL_TU

}  // namespace disc
