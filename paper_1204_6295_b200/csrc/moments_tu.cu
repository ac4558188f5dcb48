// moments_tu.cu -- instantiates k_moments_v3<R, TY, MODE> and the plain-load k_moments<R, MODE> for R in [DISC_R_LO, DISC_R_HI]; built once per range
// (-DDISC_TU=n -DDISC_R_LO=a -DDISC_R_HI=b) so the instances compile in parallel.
#include "launch.h"
#include "moments.cuh"
#include "moments_blk.cuh"
#include "moments_v3.cuh"

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

// Tiled fp32 tensor map of an (nx, ny, nz) volume with a (bx, by, bz) box, out-of-volume elements read as zero.
// A map encodes nothing but the base address, the shape and the box, so it can be reused whenever those recur -- in the
// iteration loop the source is always the context's warped-CT buffer of the level, and cuTensorMapEncodeTiled per launch
// was pure host overhead (the coarse levels are launch-bound).  Small per-thread cache, least recently used out.
static bool tensor_map_3d(EncodeTiledFn enc, const float* vol, int nx, int ny, int nz, int bx, int by, int bz,
                          CUtensorMap* out) {
    struct Entry {
        const float* vol;
        int d[6];
        unsigned long long used;
        CUtensorMap map;
    };
    constexpr int kEntries = 16;
    static thread_local Entry cache[kEntries] = {};
    static thread_local unsigned long long tick = 0;
    const int d[6] = {nx, ny, nz, bx, by, bz};
    int victim = 0;
    ++tick;
    for (int i = 0; i < kEntries; ++i) {
        Entry& e = cache[i];
        if (e.used && e.vol == vol && e.d[0] == d[0] && e.d[1] == d[1] && e.d[2] == d[2] && e.d[3] == d[3] &&
            e.d[4] == d[4] && e.d[5] == d[5]) {
            e.used = tick;
            *out = e.map;
            return true;
        }
        if (e.used < cache[victim].used) victim = i;
    }
    const cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
    const cuuint64_t gstr[2] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * ny * 4};
    const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz};
    const cuuint32_t estr[3] = {1, 1, 1};
    Entry& e = cache[victim];
    if (enc(&e.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(vol), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
        e.used = 0;
        return false;
    }
    e.vol = vol;
    for (int i = 0; i < 6; ++i) e.d[i] = d[i];
    e.used = tick;
    *out = e.map;
    return true;
}

// the plain definition for everything the sliding-window kernels do not cover (moments.cuh)
static void launch_moments_direct(int rx, int ry, int rz, int mode, const float* vol, const float* aux, float* out0,
                                  float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    dim3 grid((nx + 127) / 128, ny, nz);
    if (mode == kModeMoments)
        k_moments_direct<kModeMoments><<<grid, 128, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, rx, ry, rz, eps_var, ctl);
    else if (mode == kModeZscore)
        k_moments_direct<kModeZscore><<<grid, 128, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, rx, ry, rz, eps_var, ctl);
    else
        k_moments_direct<kModeCorrect><<<grid, 128, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, rx, ry, rz, eps_var, ctl);
}

// z chunk of the marching kernels: minimise (waves of CTAs) x (slices marched per CTA, with the 2 rz halo and a few
// slices of pipeline fill).  `slots` = CTAs resident on the device at once.
static int pick_zchunk(long long tiles, long long slots, int nz, int rz) {
    double best = 1e300;
    int best_zc = nz;
    for (int nchunk = 1; nchunk <= nz; ++nchunk) {
        const int zc = (nz + nchunk - 1) / nchunk;
        const long long ctas = tiles * ((nz + zc - 1) / zc);
        const long long waves = (ctas + slots - 1) / slots;
        const double cost = (double)waves * (zc + 2 * rz + 4);
        if (cost < best) { best = cost; best_zc = zc; }
        if (zc == 1) break;
    }
    return best_zc;
}

template <int R, int TY>
static bool launch_r_v3(const DevInfo& di, int rz, int mode, const float* vol, const float* aux, float* out0,
                        float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    using C = MomV3Cfg<R, TY>;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return false;
    CUtensorMap tmap;
    if (!tensor_map_3d(enc, vol, nx, ny, nz, C::PXB, C::PY, 1, &tmap)) return false;
    // per-voxel operand of the evaluation: the volume itself (z-score), the cached z-score (correction)
    const float* pv = mode == kModeCorrect ? aux : vol;
    const long long tiles = (long long)((nx + C::TX - 1) / C::TX) * ((ny + TY - 1) / TY);
    const int zchunk = pick_zchunk(tiles, di.n_sm, nz, rz);
    dim3 grid((nx + C::TX - 1) / C::TX, (ny + TY - 1) / TY, (nz + zchunk - 1) / zchunk);
    static bool configured[3][kMaxDevices] = {};
#define DISC_LAUNCH_MODE(M)                                                                                              \
    {                                                                                                                    \
        if (!configured[M][di.dev]) {   /* the opt-in is per device */                                                   \
            /* on failure the flag stays clear and the launch fails with an error the caller's cudaGetLastError reports */ \
            if (cudaFuncSetAttribute(k_moments_v3<R, TY, M>, cudaFuncAttributeMaxDynamicSharedMemorySize,               \
                                     (int)C::smem_bytes) == cudaSuccess)                                                 \
                configured[M][di.dev] = true;                                                                            \
        }                                                                                                                \
        k_moments_v3<R, TY, M><<<grid, C::NT, C::smem_bytes, st>>>(tmap, pv, out0, out1, nx, ny, nz, rz, zchunk, eps_var, ctl); \
    }
    if (mode == kModeMoments) DISC_LAUNCH_MODE(kModeMoments)
    else if (mode == kModeZscore) DISC_LAUNCH_MODE(kModeZscore)
    else DISC_LAUNCH_MODE(kModeCorrect)
#undef DISC_LAUNCH_MODE
    return true;
}

// Small volumes (the coarse pyramid levels): the block kernel of moments_blk.cuh.  A block is 32 x by x bz outputs;
// (by, bz) is the largest block whose raw tile + pair buffer fit shared memory, and the kernel is taken only while
// the whole grid is at most two waves of one CTA per SM -- beyond that the marching kernel's O(1) halo wins.
template <int R>
static bool launch_r_blk(const DevInfo& di, int rz, int mode, const float* vol, const float* aux, float* out0,
                         float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    using C = MomBlkCfg<R>;
    if (2 * rz + 1 > kMaxWz) return false;
    constexpr size_t kSmemMax = 216 * 1024;
    static const int cand[][2] = {{8, 4}, {8, 2}, {4, 4}, {4, 2}};
    int by = 0, bz = 0;
    for (const auto& c : cand)
        if (C::smem_bytes(c[0] + 2 * R, c[1] + 2 * rz) <= kSmemMax) { by = c[0]; bz = c[1]; break; }
    if (by * bz < 16) return false;
    const long long ctas = (long long)((nx + C::TX - 1) / C::TX) * ((ny + by - 1) / by) * ((nz + bz - 1) / bz);
    if (ctas > 2LL * di.n_sm) return false;
    const int py = by + 2 * R, pz = bz + 2 * rz;
    if (py > 256 || pz > 256) return false;
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return false;
    CUtensorMap tmap;
    if (!tensor_map_3d(enc, vol, nx, ny, nz, C::PXB, py, pz, &tmap)) return false;
    const float* pv = mode == kModeCorrect ? aux : vol;
    dim3 grid((nx + C::TX - 1) / C::TX, (ny + by - 1) / by, (nz + bz - 1) / bz);
    const size_t smem = C::smem_bytes(py, pz);
    static bool configured[3][kMaxDevices] = {};
#define DISC_LAUNCH_MODE(M)                                                                                              \
    {                                                                                                                    \
        if (!configured[M][di.dev]) {   /* the opt-in is per device */                                                   \
            if (cudaFuncSetAttribute(k_moments_blk<R, M>, cudaFuncAttributeMaxDynamicSharedMemorySize,                  \
                                     (int)kSmemMax) == cudaSuccess)                                                      \
                configured[M][di.dev] = true;                                                                            \
        }                                                                                                                \
        k_moments_blk<R, M><<<grid, C::NT, smem, st>>>(tmap, pv, out0, out1, nx, ny, nz, rz, by, bz, eps_var, ctl);      \
    }
    if (mode == kModeMoments) DISC_LAUNCH_MODE(kModeMoments)
    else if (mode == kModeZscore) DISC_LAUNCH_MODE(kModeZscore)
    else DISC_LAUNCH_MODE(kModeCorrect)
#undef DISC_LAUNCH_MODE
    return true;
}

// the TMA kernel with the tile height the z window allows: 32 rows while the ring of 2 rz + 1 slots fits tensor
// memory, 16 rows beyond (possible only when the tile + halo still has 32 rows, R >= 8)
template <int R>
static bool launch_r_tma(const DevInfo& di, int rz, int mode, const float* vol, const float* aux, float* out0,
                         float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    const int wz = 2 * rz + 1;
    if (wz <= MomV3Cfg<R, 32>::WZ_MAX)
        return launch_r_v3<R, 32>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
    if constexpr (R >= 8) {
        if (wz <= MomV3Cfg<R, 16>::WZ_MAX)
            return launch_r_v3<R, 16>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
    }
    return false;
}

template <int R>
static bool launch_r(const DevInfo& di, int rz, int mode, const float* vol, const float* aux, float* out0, float* out1,
                     int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    if (di.dev < 0 || di.dev >= kMaxDevices) return false;
    // TMA path: rows must be 16-byte multiples and the base 16-byte aligned (tensor-map requirements)
    if (nx % 4 == 0 && (reinterpret_cast<uintptr_t>(vol) & 15u) == 0 &&
        (launch_r_blk<R>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st) ||
         launch_r_tma<R>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st)))
        return true;
    if constexpr (R <= 10) {
        if (rz == R) {   // plain-load sliding-window kernel: cubic patches, any nx
            const long long tiles = (long long)((nx + kMomTX - 1) / kMomTX) * ((ny + kMomTY - 1) / kMomTY);
            const int zchunk = pick_zchunk(tiles, 2LL * di.n_sm, nz, rz);
            dim3 grid((nx + kMomTX - 1) / kMomTX, (ny + kMomTY - 1) / kMomTY, (nz + zchunk - 1) / zchunk);
            constexpr int NT = MomCfg<R>::NT;
            if (mode == kModeMoments)
                k_moments<R, kModeMoments><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, ctl);
            else if (mode == kModeZscore)
                k_moments<R, kModeZscore><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, ctl);
            else
                k_moments<R, kModeCorrect><<<grid, NT, 0, st>>>(vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, ctl);
            return true;
        }
    }
    launch_moments_direct(R, R, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
    return true;
}

// one radius: launches if R lies in this unit's range (the discarded branch is never instantiated)
template <int R>
static bool case_r(const DevInfo& di, int rz, int mode, const float* vol, const float* aux, float* out0, float* out1,
                   int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    if constexpr (R >= DISC_R_LO && R <= DISC_R_HI) {
        return launch_r<R>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
    } else {
        return false;
    }
}

bool DISC_CAT(launch_moments_tu, DISC_TU)(const DevInfo& di, int rxy, int rz, int mode, const float* vol,
                                          const float* aux, float* out0, float* out1, int nx, int ny, int nz,
                                          float eps_var, IterCtl ctl, cudaStream_t st) {
    switch (rxy) {
#define DISC_CASE(r) \
    case r: return case_r<r>(di, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
        DISC_CASE(0) DISC_CASE(1) DISC_CASE(2) DISC_CASE(3) DISC_CASE(4) DISC_CASE(5) DISC_CASE(6)
        DISC_CASE(7) DISC_CASE(8) DISC_CASE(9) DISC_CASE(10) DISC_CASE(11) DISC_CASE(12)
#undef DISC_CASE
    }
    return false;
}

}  // namespace disc
