// moments_tu.cu -- instantiates k_moments<R, MODE> for R in [DISC_R_LO, DISC_R_HI]; built once per range
// (-DDISC_TU=n -DDISC_R_LO=a -DDISC_R_HI=b) so the instances compile in parallel.
#include "launch.h"
#include "moments.cuh"

#define DISC_CAT2(a, b) a##b
#define DISC_CAT(a, b) DISC_CAT2(a, b)

namespace disc {

template <int R>
static void launch_r(int mode, const float* vol, const float* aux, float* out0, float* out1, int nx, int ny, int nz,
                     int zchunk, float eps_var, cudaStream_t st) {
    dim3 grid((nx + kMomTX - 1) / kMomTX, (ny + kMomTY - 1) / kMomTY, (nz + zchunk - 1) / zchunk);
    constexpr int NT = MomCfg<R>::NT;
    if (mode == kModeMoments)
        k_moments<R, kModeMoments><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var);
    else if (mode == kModeZscore)
        k_moments<R, kModeZscore><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var);
    else
        k_moments<R, kModeCorrect><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var);
}

bool DISC_CAT(launch_moments_tu, DISC_TU)(int R, int mode, const float* vol, const float* aux, float* out0,
                                          float* out1, int nx, int ny, int nz, int zchunk, float eps_var,
                                          cudaStream_t st) {
    switch (R) {
#define DISC_CASE(r)                                                              \
    case r:                                                                       \
        if (r >= DISC_R_LO && r <= DISC_R_HI) {                                   \
            launch_r<(r >= DISC_R_LO && r <= DISC_R_HI) ? r : DISC_R_LO>(mode, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st); \
            return true;                                                          \
        }                                                                         \
        return false;
        DISC_CASE(0) DISC_CASE(1) DISC_CASE(2) DISC_CASE(3) DISC_CASE(4) DISC_CASE(5)
        DISC_CASE(6) DISC_CASE(7) DISC_CASE(8) DISC_CASE(9) DISC_CASE(10)
#undef DISC_CASE
    }
    return false;
}

}  // namespace disc
