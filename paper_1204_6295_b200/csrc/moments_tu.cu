// moments_tu.cu -- instantiates k_moments<R, MODE> for R in [DISC_R_LO, DISC_R_HI]; built once per range
// (-DDISC_TU=n -DDISC_R_LO=a -DDISC_R_HI=b) so the instances compile in parallel.
#include "launch.h"
#include "moments.cuh"
#include "moments_v2.cuh"

#define DISC_CAT2(a, b) a##b
#define DISC_CAT(a, b) DISC_CAT2(a, b)

namespace disc {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point: no link-time dependency on libcuda
static EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

template <int R, int TY>
static bool launch_r_v2(int mode, const float* vol, const float* aux, float* out0, float* out1, int nx, int ny,
                        int nz, int zchunk, float eps_var, cudaStream_t st) {
    using C = MomV2Cfg<R, TY>;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return false;
    CUtensorMap tmap, tmap_aux;
    const cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
    const cuuint64_t gstr[2] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * ny * 4};
    const cuuint32_t box[3] = {(cuuint32_t)C::PXB, (cuuint32_t)C::PY, 1};
    const cuuint32_t box_aux[3] = {(cuuint32_t)C::TX, (cuuint32_t)TY, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    // per-voxel operand of the evaluation: the volume itself (z-score), the cached z-score (correction)
    const float* per_voxel = mode == kModeCorrect ? aux : vol;
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(vol), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS ||
        enc(&tmap_aux, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(per_voxel), gdim, gstr, box_aux, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    static bool configured[3] = {false, false, false};
    dim3 grid((nx + C::TX - 1) / C::TX, (ny + TY - 1) / TY, (nz + zchunk - 1) / zchunk);
#define DISC_LAUNCH_MODE(M)                                                                                         \
    {                                                                                                               \
        if (!configured[M]) {                                                                                       \
            cudaFuncSetAttribute(k_moments_v2<R, TY, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes); \
            configured[M] = true;                                                                                   \
        }                                                                                                           \
        k_moments_v2<R, TY, M><<<grid, C::NT, C::smem_bytes, st>>>(tmap, tmap_aux, out0, out1, nx, ny, nz, zchunk, eps_var, g_iter_ctl); \
    }
    if (mode == kModeMoments) DISC_LAUNCH_MODE(kModeMoments)
    else if (mode == kModeZscore) DISC_LAUNCH_MODE(kModeZscore)
    else DISC_LAUNCH_MODE(kModeCorrect)
#undef DISC_LAUNCH_MODE
    return true;
}

template <int R>
static bool launch_r_tma(int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx,
                         int ny, int nz, int zchunk, float eps_var, cudaStream_t st) {
    if constexpr (R <= kMomMaxRTile32) {
        if (ty == 32) return launch_r_v2<R, 32>(mode, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st);
    }
    return launch_r_v2<R, 16>(mode, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st);
}

template <int R>
static void launch_r(int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx, int ny, int nz,
                     int zchunk, float eps_var, cudaStream_t st) {
    // TMA path: rows must be 16-byte multiples and the base 16-byte aligned (tensor-map requirements)
    if (nx % 4 == 0 && (reinterpret_cast<uintptr_t>(vol) & 15u) == 0 &&
        (mode != kModeCorrect || (reinterpret_cast<uintptr_t>(aux) & 15u) == 0) &&
        launch_r_tma<R>(mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st))
        return;
    dim3 grid((nx + kMomTX - 1) / kMomTX, (ny + kMomTY - 1) / kMomTY, (nz + zchunk - 1) / zchunk);
    constexpr int NT = MomCfg<R>::NT;
    if (mode == kModeMoments)
        k_moments<R, kModeMoments><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, g_iter_ctl);
    else if (mode == kModeZscore)
        k_moments<R, kModeZscore><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, g_iter_ctl);
    else
        k_moments<R, kModeCorrect><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, g_iter_ctl);
}

// one radius: launches if R lies in this unit's range (the discarded branch is never instantiated)
template <int R>
static bool case_r(int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx, int ny,
                   int nz, int zchunk, float eps_var, cudaStream_t st) {
    if constexpr (R >= DISC_R_LO && R <= DISC_R_HI) {
        launch_r<R>(mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st);
        return true;
    } else {
        return false;
    }
}

bool DISC_CAT(launch_moments_tu, DISC_TU)(int R, int mode, int ty, const float* vol, const float* aux,
                                          float* out0, float* out1, int nx, int ny, int nz, int zchunk,
                                          float eps_var, cudaStream_t st) {
    switch (R) {
#define DISC_CASE(r) \
    case r: return case_r<r>(mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st);
        DISC_CASE(0) DISC_CASE(1) DISC_CASE(2) DISC_CASE(3) DISC_CASE(4) DISC_CASE(5)
        DISC_CASE(6) DISC_CASE(7) DISC_CASE(8) DISC_CASE(9) DISC_CASE(10)
#undef DISC_CASE
    }
    return false;
}

}  // namespace disc
