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

static int pick_chunk(int n, int min_chunk, long long ctas_per_chunk, long long target_ctas) {
    // split an axis of length n into chunks so that the grid reaches ~target_ctas CTAs,
    // but never below min_chunk (each chunk re-reads a halo)
    long long want = target_ctas / ctas_per_chunk;  // round down: prefer one full wave over 1.x waves
    if (want < 1) want = 1;
    int chunk = (int)((n + want - 1) / want);
    if (chunk < min_chunk) chunk = min_chunk;
    if (chunk > n) chunk = n;
    return chunk;
}

template <int K, int FORCE, int TY, bool STOP>
static void launch_fg_t4s(const DevInfo& di, const float* m, const float* s, const float* rin, float* rout, int nx, int ny,
                          int nz, float eps_den, const GaussTaps& taps, IterCtl ctl, StopReq stop, cudaStream_t st) {
    using C = FgT4Cfg<K, TY>;
    static bool configured[kMaxDevices] = {};  // the opt-in is per device (idempotent, so a race is harmless)
    if (!configured[di.dev]) {
        // on failure the flag stays clear and the launch below fails with a shared-memory error that cudaGetLastError
        // in the caller reports
        if (cudaFuncSetAttribute(k_force_gxy_t4<K, FORCE, TY, STOP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)C::smem_bytes) == cudaSuccess)
            configured[di.dev] = true;
    }
    const long long n_tiles = (long long)((nx + C::TX - 1) / C::TX) * ((ny + C::TY - 1) / C::TY) * nz;
    const int grid = (int)(n_tiles < (long long)C::OCC * di.n_sm ? n_tiles : (long long)C::OCC * di.n_sm);   // persistent: OCC CTAs per SM
    k_force_gxy_t4<K, FORCE, TY, STOP><<<grid, C::NT, C::smem_bytes, st>>>(m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop.ctl,
                                                                         stop.iter, stop.eps);
}

template <int K, int FORCE, int TY>
static void launch_fg_t4(const DevInfo& di, const float* m, const float* s, const float* rin, float* rout, int nx, int ny,
                         int nz, float eps_den, const GaussTaps& taps, IterCtl ctl, StopReq stop, cudaStream_t st) {
    if constexpr (FORCE != 0) {
        if (stop.ctl) { launch_fg_t4s<K, FORCE, TY, true>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st); return; }
    }
    launch_fg_t4s<K, FORCE, TY, false>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
}

template <int K, int FORCE>
static void launch_fg(const DevInfo& di, const float* m, const float* s, const float* rin, float* rout, int nx, int ny,
                      int nz, float eps_den, const GaussTaps& taps, IterCtl ctl, StopReq stop, cudaStream_t st) {
    const bool vec_ok = nx % 4 == 0 && aligned16(rin) && aligned16(rout) && (!FORCE || (aligned16(m) && aligned16(s))) &&
                        3ull * nx * ny * nz < 0xffffffffull;   // the tile kernel indexes voxels with 32 bits
    const int n_sm = di.n_sm;
    if (vec_ok && di.dev >= 0 && di.dev < kMaxDevices) {
        // 64 x 32 tiles; 64 x 8 where those would leave CTA slots of the device empty (small levels)
        const long long tiles32 = (long long)((nx + 63) / 64) * ((ny + 31) / 32) * nz;
        if (tiles32 < (long long)FgT4Cfg<K, 32>::OCC * n_sm)
            launch_fg_t4<K, FORCE, 8>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        else
            launch_fg_t4<K, FORCE, 32>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        return;
    }
    // plain-load fallback: the criterion's sums come from their own pass over m, s', r
    if (FORCE != 0 && stop.ctl)
        launch_force_norms(FORCE, m, s, rin, nx, ny, nz, eps_den, stop.ctl, stop.iter, stop.eps, n_sm, st);
    const int txb = nx > 64 ? 128 : (nx > 32 ? 64 : 32);
    const int xt = (nx + txb - 1) / txb;
    const int yseg = pick_chunk(ny, 8 * K > 32 ? 8 * K : 32, (long long)xt * nz, 4LL * n_sm);
    dim3 grid((nx + txb - 1) / txb, (ny + yseg - 1) / yseg, nz);
    if (txb == 128)
        k_force_gxy<K, FORCE, 128><<<grid, 128, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, ctl);
    else if (txb == 64)
        k_force_gxy<K, FORCE, 64><<<grid, 64, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, ctl);
    else
        k_force_gxy<K, FORCE, 32><<<grid, 32, 0, st>>>(m, s, rin, rout, nx, ny, nz, yseg, eps_den, taps, ctl);
}

template <int K, bool WARP, int LZ>
static void launch_gzd(const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                       const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    const size_t plane = (size_t)nx * ny;
    dim3 grid((unsigned)((plane + kGzdThreads - 1) / kGzdThreads), (nz + LZ - 1) / LZ, 1);
    k_gz_warp_d<K, WARP, LZ><<<grid, kGzdThreads, 0, st>>>(rin, rout, moving, mout, nx, ny, nz, taps, ctl);
}

template <int K, bool WARP, int LZ>
static void launch_gzd2(const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                        const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    const size_t pairs = (size_t)nx * ny / 2;
    dim3 grid((unsigned)((pairs + kGzdThreads - 1) / kGzdThreads), (nz + LZ - 1) / LZ, 1);
    k_gz_warp_d2<K, WARP, LZ><<<grid, kGzdThreads, 0, st>>>(rin, rout, moving, mout, nx, ny, nz, taps, ctl);
}

static inline bool aligned8(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 7u) == 0; }

// A thread owns two adjacent columns (one when nx is odd or a field is not 8-byte aligned) and LZ output slices.
// Measured on B200: at the fine levels 4 slices beat 8 (more threads in flight; the 2K halo re-reads come from L2).
// A small level does not fill the device with 4 slices per thread: LZ is halved while the grid stays below a quarter of
// the device's thread slots (the 13 / LZ re-reads per output hit L2, and the level is latency-bound anyway).
template <int K, bool WARP>
static void launch_gz(const DevInfo& di, const float* rin, float* rout, const float* moving, float* mout, int nx, int ny,
                      int nz, const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    const long long want = 512LL * di.n_sm;
    if (nx % 2 == 0 && aligned8(rin) && aligned8(rout) && (!WARP || aligned8(mout))) {
        const long long cols = (long long)nx * ny / 2;
        if (cols * ((nz + 3) / 4) >= want) launch_gzd2<K, WARP, 4>(rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
        else if (cols * ((nz + 1) / 2) >= want) launch_gzd2<K, WARP, 2>(rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
        else launch_gzd2<K, WARP, 1>(rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
    } else {
        launch_gzd<K, WARP, 4>(rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
    }
}

// one Gaussian radius: launches if K lies in this unit's range (the discarded branch is never instantiated)
template <int K>
static bool case_fg(const DevInfo& di, int force, const float* m, const float* s, const float* rin, float* rout, int nx,
                    int ny, int nz, float eps_den, const GaussTaps& taps, IterCtl ctl, StopReq stop, cudaStream_t st) {
    if constexpr (K >= DISC_K_LO && K <= DISC_K_HI) {
        if (force == kForceDouble) launch_fg<K, kForceDouble>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        else if (force == kForceSingle) launch_fg<K, kForceSingle>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        else launch_fg<K, kForceNone>(di, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        return true;
    } else {
        return false;
    }
}

template <int K>
static bool case_gz(const DevInfo& di, bool warp, const float* rin, float* rout, const float* moving, float* mout, int nx, int ny, int nz,
                    const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    if constexpr (K >= DISC_K_LO && K <= DISC_K_HI) {
        if (warp) launch_gz<K, true>(di, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
        else launch_gz<K, false>(di, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
        return true;
    } else {
        return false;
    }
}

#define DISC_FOR_K(X) X(1) X(2) X(3) X(4) X(5) X(6) X(7) X(8) X(9) X(10) X(11) X(12)

bool DISC_CAT(launch_force_gxy_tu, DISC_TU)(const DevInfo& di, int K, int force, const float* m, const float* s,
                                            const float* rin, float* rout, int nx, int ny, int nz, float eps_den,
                                            const GaussTaps& taps, IterCtl ctl, StopReq stop, cudaStream_t st) {
    switch (K) {
#define DISC_CASE(k) \
    case k: return case_fg<k>(di, force, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
        DISC_FOR_K(DISC_CASE)
#undef DISC_CASE
    }
    return false;
}

bool DISC_CAT(launch_gz_warp_tu, DISC_TU)(const DevInfo& di, int K, bool warp, const float* rin, float* rout,
                                          const float* moving, float* mout, int nx, int ny, int nz,
                                          const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    switch (K) {
#define DISC_CASE(k) \
    case k: return case_gz<k>(di, warp, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
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
    if (blocks > (size_t)kStopBlocks) blocks = kStopBlocks;
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

bool launch_moments_any(const DevInfo& di, int rxy, int rz, int mode, const float* vol, const float* aux, float* out0,
                        float* out1, int nx, int ny, int nz, float eps_var, IterCtl ctl, cudaStream_t st) {
    return launch_moments_tu0(di, rxy, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st) ||
           launch_moments_tu1(di, rxy, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st) ||
           launch_moments_tu2(di, rxy, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st) ||
           launch_moments_tu3(di, rxy, rz, mode, vol, aux, out0, out1, nx, ny, nz, eps_var, ctl, st);
}

bool launch_force_gxy_any(const DevInfo& di, int K, int force, const float* m, const float* s, const float* rin,
                          float* rout, int nx, int ny, int nz, float eps_den, const GaussTaps& taps, IterCtl ctl,
                          StopReq stop, cudaStream_t st) {
    return launch_force_gxy_tu0(di, K, force, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st) ||
           launch_force_gxy_tu1(di, K, force, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st) ||
           launch_force_gxy_tu2(di, K, force, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st) ||
           launch_force_gxy_tu3(di, K, force, m, s, rin, rout, nx, ny, nz, eps_den, taps, ctl, stop, st);
}

bool launch_gz_warp_any(const DevInfo& di, int K, bool warp, const float* rin, float* rout, const float* moving,
                        float* mout, int nx, int ny, int nz, const GaussTaps& taps, IterCtl ctl, cudaStream_t st) {
    return launch_gz_warp_tu0(di, K, warp, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st) ||
           launch_gz_warp_tu1(di, K, warp, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st) ||
           launch_gz_warp_tu2(di, K, warp, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st) ||
           launch_gz_warp_tu3(di, K, warp, rin, rout, moving, mout, nx, ny, nz, taps, ctl, st);
}
#endif

}  // namespace disc
