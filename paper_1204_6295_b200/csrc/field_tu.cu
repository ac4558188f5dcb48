// field_tu.cu -- instantiates the force+Gxy and Gz+warp kernels (field.cuh, field_v3.cuh) for K in [DISC_K_LO, DISC_K_HI]; built
// once per range (-DDISC_TU=n -DDISC_K_LO=a -DDISC_K_HI=b).  TU 0 also holds the K-independent kernels.
#include <cstdlib>

#include "field.cuh"
#include "field_v3.cuh"
#include "launch.h"

#define DISC_CAT2(a, b) a##b
#define DISC_CAT(a, b) DISC_CAT2(a, b)

namespace disc {

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

template <int K, int FORCE>
static void launch_fg(int txb, const float* m, const float* s, const float* rin, float* rout, int nx, int ny, int nz,
                      int yseg, float eps_den, const GaussTaps& taps, cudaStream_t st) {
    const bool vec_ok = nx % 4 == 0 && aligned16(rin) && aligned16(rout) && (!FORCE || (aligned16(m) && aligned16(s))) &&
                        3ull * nx * ny * nz < 0xffffffffull;   // the tile kernel indexes voxels with 32 bits
    static int n_sm = 0;
    if (!n_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    }
    if (vec_ok) {
        using C = FgT4Cfg<K>;
        static bool configured = false;  // one attribute call per instance (idempotent, so a race is harmless)
        if (!configured) {
            cudaFuncSetAttribute(k_force_gxy_t4<K, FORCE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
            configured = true;
        }
        const long long n_tiles = (long long)((nx + C::TX - 1) / C::TX) * ((ny + C::TY - 1) / C::TY) * nz;
        const int grid = (int)(n_tiles < (long long)C::OCC * n_sm ? n_tiles : (long long)C::OCC * n_sm);   // persistent: OCC CTAs per SM
        k_force_gxy_t4<K, FORCE><<<grid, C::NT, C::smem_bytes, st>>>(m, s, rin, rout, nx, ny, nz, eps_den, taps, g_iter_ctl);
        return;
    }
    dim3 grid((nx + txb - 1) / txb, (ny + yseg - 1) / yseg, nz);
    if (txb == 128)
        k_force_gxy<K, FORCE, 128><<<grid, 128, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, g_iter_ctl);
    else if (txb == 64)
        k_force_gxy<K, FORCE, 64><<<grid, 64, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, g_iter_ctl);
    else
        k_force_gxy<K, FORCE, 32><<<grid, 32, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, g_iter_ctl);
}

template <int K, bool WARP, int LZ>
static void launch_gzd(const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                       const GaussTaps& taps, cudaStream_t st) {
    const size_t plane = (size_t)nx * ny;
    dim3 grid((unsigned)((plane + kGzdThreads - 1) / kGzdThreads), (nz + LZ - 1) / LZ, 1);
    k_gz_warp_d<K, WARP, LZ><<<grid, kGzdThreads, 0, st>>>(rin, rout, moving, mout, nx, ny, nz, taps, g_iter_ctl);
}

template <int K, bool WARP, int LZ>
static void launch_gzd2(const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                        const GaussTaps& taps, cudaStream_t st) {
    const size_t pairs = (size_t)nx * ny / 2;
    dim3 grid((unsigned)((pairs + kGzdThreads - 1) / kGzdThreads), (nz + LZ - 1) / LZ, 1);
    k_gz_warp_d2<K, WARP, LZ><<<grid, kGzdThreads, 0, st>>>(rin, rout, moving, mout, nx, ny, nz, taps, g_iter_ctl);
}

static inline bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

template <int K, bool WARP>
static void launch_gz(const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                      int zchunk, const GaussTaps& taps, cudaStream_t st) {
    // zchunk = output slices per thread (4 or 8) + 100 * (columns per thread, 1 or 2), chosen by the caller
    const int lz = zchunk % 100, two = zchunk / 100 >= 2;
    if (two && nx % 2 == 0 && aligned8(rin) && aligned8(rout) && (!WARP || aligned8(mout))) {
        if (lz >= 8) launch_gzd2<K, WARP, 8>(rin, rout, moving, mout, nx, ny, nz, taps, st);
        else launch_gzd2<K, WARP, 4>(rin, rout, moving, mout, nx, ny, nz, taps, st);
        return;
    }
    if (lz >= 8) launch_gzd<K, WARP, 8>(rin, rout, moving, mout, nx, ny, nz, taps, st);
    else launch_gzd<K, WARP, 4>(rin, rout, moving, mout, nx, ny, nz, taps, st);
}

// one Gaussian radius: launches if K lies in this unit's range (the discarded branch is never instantiated)
template <int K>
static bool case_fg(int force, int txb, const float* m, const float* s, const float* rin, float* rout, int nx, int ny,
                    int nz, int yseg, float eps_den, const GaussTaps& taps, cudaStream_t st) {
    if constexpr (K >= DISC_K_LO && K <= DISC_K_HI) {
        if (force == kForceDouble) launch_fg<K, kForceDouble>(txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st);
        else if (force == kForceSingle) launch_fg<K, kForceSingle>(txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st);
        else launch_fg<K, kForceNone>(txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st);
        return true;
    } else {
        return false;
    }
}

template <int K>
static bool case_gz(bool warp, const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                    int zchunk, const GaussTaps& taps, cudaStream_t st) {
    if constexpr (K >= DISC_K_LO && K <= DISC_K_HI) {
        if (warp) launch_gz<K, true>(rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st);
        else launch_gz<K, false>(rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st);
        return true;
    } else {
        return false;
    }
}

#define DISC_FOR_K(X) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12)

bool DISC_CAT(launch_force_gxy_tu, DISC_TU)(int K, int force, int txb, const float* m, const float* s,
                                            const float* rin, float* rout, int nx, int ny, int nz, int yseg,
                                            float eps_den, const GaussTaps& taps, cudaStream_t st) {
    switch (K) {
#define DISC_CASE(k) \
    case k: return case_fg<k>(force, txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st);
        DISC_FOR_K(DISC_CASE)
#undef DISC_CASE
    }
    return false;
}

bool DISC_CAT(launch_gz_warp_tu, DISC_TU)(int K, bool warp, const float* rin, float* rout, const float* moving,
                                          float* mout, int nx, int ny, int nz, int zchunk, const GaussTaps& taps,
                                          cudaStream_t st) {
    switch (K) {
#define DISC_CASE(k) \
    case k: return case_gz<k>(warp, rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st);
        DISC_FOR_K(DISC_CASE)
#undef DISC_CASE
    }
    return false;
}

#if DISC_TU == 0
void launch_force_update(int force, const float* m, const float* s, float* r, int nx, int ny, int nz, float eps_den,
                         cudaStream_t st) {
    dim3 grid((nx + 255) / 256, ny, nz);
    if (force == kForceDouble) k_force_update<kForceDouble><<<grid, 256, 0, st>>>(m, s, r, nx, ny, nz, eps_den);
    else k_force_update<kForceSingle><<<grid, 256, 0, st>>>(m, s, r, nx, ny, nz, eps_den);
}

void launch_force_norms(int force, const float* m, const float* s, const float* r, int nx, int ny, int nz, float eps_den,
                        StopCtl* ctl, int iter, float stop_eps, int n_sm, cudaStream_t st) {
    const size_t N = (size_t)nx * ny * nz;
    size_t blocks = (N + 255) / 256;
    if (blocks > (size_t)8 * n_sm) blocks = (size_t)8 * n_sm;   // grid-stride: one wave of 8 CTAs per SM
    if (force == kForceDouble)
        k_force_norms<kForceDouble><<<(unsigned)blocks, 256, 0, st>>>(m, s, r, nx, ny, nz, eps_den, ctl, iter, stop_eps);
    else
        k_force_norms<kForceSingle><<<(unsigned)blocks, 256, 0, st>>>(m, s, r, nx, ny, nz, eps_den, ctl, iter, stop_eps);
}

void launch_stop_reset(StopCtl* ctl, cudaStream_t st) { k_stop_reset<<<1, 1, 0, st>>>(ctl); }
void launch_stop_record(StopCtl* ctl, int level, int n_iters, cudaStream_t st) {
    k_stop_record<<<1, 1, 0, st>>>(ctl, level, n_iters);
}

void launch_warp_kernel(const float* moving, const float* r, float* out, int nx, int ny, int nz, cudaStream_t st) {
    if (nx % 2 == 0 && (reinterpret_cast<uintptr_t>(r) & 7u) == 0 && (reinterpret_cast<uintptr_t>(out) & 7u) == 0) {
        dim3 grid2((nx / 2 + 127) / 128, ny, nz);
        k_warp2<<<grid2, 128, 0, st>>>(moving, r, out, nx, ny, nz);
        return;
    }
    dim3 grid((nx + 255) / 256, ny, nz);
    k_warp<<<grid, 256, 0, st>>>(moving, r, out, nx, ny, nz);
}

bool launch_moments_any(int R, int mode, int ty, const float* vol, const float* aux, float* out0, float* out1, int nx,
                        int ny, int nz, int zchunk, float eps_var, cudaStream_t st) {
    return launch_moments_tu0(R, mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st) ||
           launch_moments_tu1(R, mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st) ||
           launch_moments_tu2(R, mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st) ||
           launch_moments_tu3(R, mode, ty, vol, aux, out0, out1, nx, ny, nz, zchunk, eps_var, st);
}

bool launch_force_gxy_any(int K, int force, int txb, const float* m, const float* s, const float* rin, float* rout,
                          int nx, int ny, int nz, int yseg, float eps_den, const GaussTaps& taps, cudaStream_t st) {
    return launch_force_gxy_tu0(K, force, txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st) ||
           launch_force_gxy_tu1(K, force, txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st) ||
           launch_force_gxy_tu2(K, force, txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st) ||
           launch_force_gxy_tu3(K, force, txb, m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, st);
}

bool launch_gz_warp_any(int K, bool warp, const float* rin, float* rout, const float* moving, float* mout, int nx,
                        int ny, int nz, int zchunk, const GaussTaps& taps, cudaStream_t st) {
    return launch_gz_warp_tu0(K, warp, rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st) ||
           launch_gz_warp_tu1(K, warp, rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st) ||
           launch_gz_warp_tu2(K, warp, rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st) ||
           launch_gz_warp_tu3(K, warp, rin, rout, moving, mout, nx, ny, nz, zchunk, taps, st);
}
#endif

}  // namespace disc
