// moments_v3.cuh -- patch moments + intensity correction, step (a): the warp-specialised sm_100a kernel.
//
// What it computes (PAPER.md:95 Eq. 3, :117-119 Eqs. 5-6, :458 A.4; readings A4, A5): over the box of radius
// (RXY, RXY, RZ) truncated to the volume, S1 = sum v and S2 = sum v^2 as separable sliding-window sums in fp64
// (cost independent of the radius; the paper's kernel loops over the whole patch), then
// mu = S1/n, var = S2/n - mu^2 and the mode's output.  RXY is a template parameter, RZ a run-time one
// (the paper's non-cubic patches 3x3x3 ... 25x25x7, all have RX = RY).
//
// A CTA owns a 32 x TY (x,y) tile and marches z through a chunk.  Three roles, handing buffers over through
// mbarriers, each on a different slice at any time:
//   producer  one thread: 3-D TMA tile loads (zero out-of-bounds fill = the truncated patch) NSTG slices ahead;
//   x pass    NXW warps.  Task = one ROW of one slice, lanes <-> rows; the tasks of all slices are numbered
//             consecutively and dealt out 32 at a time, so every warp instruction has 32 live lanes whatever
//             the tile height.  A lane reads its raw row (16-byte loads), converts to fp64 and slides (S1, S2)
//             along x over the whole tile width: one conversion and four fp64 operations per element --
//             d_new^2 - d_old^2 = (d_new - d_old)(d_new + d_old) is exact in fp64 for fp32 inputs;
//   y/z pass  TX*TY/LY threads.  A thread owns column x = lane and LY rows, BOTH sums: slides along y out of the
//             x pass's exchange buffer (16-byte loads, conflict free), moves the z window -- the last 2 RZ + 1
//             xy box sums of its columns, fp64, kept in TENSOR MEMORY as a private ring in the thread's TMEM
//             lane (tcgen05.ld / tcgen05.st, one slot per slice) -- and evaluates its LY voxels.
// Against moments_v2 (r01): one thread per column instead of an S1 thread and an S2 thread that swap sums by
// shuffle, x runs over the whole tile width instead of runs of 8, no per-voxel operand staging by TMA, 32-bit
// shared addresses folded into immediates: 132 -> ~50 thread instructions per voxel (profiles/r02_*).
//
// Requirements (checked by the launcher): nx % 4 == 0, 16-byte aligned volume (tensor-map rules).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "launch.h"
#include "pipeline.cuh"

namespace disc {

constexpr int kMaxWz = 33;   // longest z window any configuration of this kernel supports (WZ_MAX <= 32)

__host__ __device__ constexpr uint32_t pow2_tmem_cols(uint32_t n) { return n <= 32 ? 32 : n <= 64 ? 64 : n <= 128 ? 128 : n <= 256 ? 256 : 512; }

template <int R, int TY>
struct MomV3Cfg {
    static constexpr int W = 2 * R + 1;
    static constexpr int TX = 32, LY = 4;                             // rows per y/z thread (2: 61.8 us, 4: 57.6, 8: 88.8)
    static constexpr int PX = TX + 2 * R, PY = TY + 2 * R;
    static constexpr int NYZ = TX * TY / LY;                          // y/z-pass threads
    static constexpr int NXW = 4;                                      // x-pass warps
    static constexpr int NT = NYZ + 32 * NXW + 32;                     // + the producer warp
    // The innermost TMA coordinate must be a multiple of 4 floats, so the box starts at x0 - RA (RA = R rounded
    // up to 4) and column x0 - R sits at offset OFF of a raw row; the box width is a multiple of 4 floats with
    // an odd number of 16-byte chunks (lanes <-> rows reads are then bank-conflict free).
    static constexpr int RA = (R + 3) / 4 * 4, OFF = RA - R;
    static constexpr int PXB = (((OFF + PX + 3) / 4) | 1) * 4;
    static constexpr int XSP = TX + 1;                                 // exchange-row pitch in (S1,S2) pairs, odd
    static constexpr size_t raw_bytes = sizeof(float) * PY * PXB;      // one stage; multiple of 16
    static constexpr size_t raw_stride = (raw_bytes + 127) / 128 * 128;
    static constexpr size_t xs_bytes = sizeof(double2) * PY * XSP;
    // stages: as many as fit 200 KB, at most 8 raw / 4 exchange
    static constexpr int NXS = (4 * xs_bytes + 6 * raw_stride <= 200 * 1024) ? 4 : 3;
    static constexpr int NSTG_FIT = (int)((200 * 1024 - NXS * xs_bytes) / raw_stride);
    static constexpr int NSTG = NSTG_FIT > 8 ? 8 : NSTG_FIT;
    static constexpr size_t smem_bytes = 128 + NSTG * raw_stride + NXS * xs_bytes;
    static constexpr int RING_WORDS = 4 * LY;                          // one ring slot of one thread: LY x (S1,S2) fp64
    static constexpr int GROUPS = (NYZ / 32 + 3) / 4;                  // warps sharing a TMEM lane quadrant
    static constexpr int WZ_MAX = 512 / (GROUPS * RING_WORDS);         // longest z window tensor memory holds
    static_assert(PY >= 32, "a group of 32 x-pass tasks must not span more than two slices");
    static_assert(NSTG >= 3, "raw ring too short");
    static_assert(LY == 2 || LY == 4 || LY == 8, "the ring slot moves with the .x8 / .x16 / .x32 tcgen05 shapes");
};

#define DISC_R8(v, b) "=r"(v[b]), "=r"(v[b + 1]), "=r"(v[b + 2]), "=r"(v[b + 3]), "=r"(v[b + 4]), "=r"(v[b + 5]), "=r"(v[b + 6]), "=r"(v[b + 7])
#define DISC_I8(v, b) "r"(v[b]), "r"(v[b + 1]), "r"(v[b + 2]), "r"(v[b + 3]), "r"(v[b + 4]), "r"(v[b + 5]), "r"(v[b + 6]), "r"(v[b + 7])
// one ring slot of one thread (N = 8, 16 or 32 words) between its TMEM lane and registers
template <int N>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t (&v)[N]) {
    static_assert(N == 8 || N == 16 || N == 32, "tcgen05.ld shapes .x8 / .x16 / .x32");
    if constexpr (N == 8) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                     : DISC_R8(v, 0) : "r"(taddr) : "memory");
    } else if constexpr (N == 16) {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                     : DISC_R8(v, 0), DISC_R8(v, 8) : "r"(taddr) : "memory");
    } else {
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                     "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                     : DISC_R8(v, 0), DISC_R8(v, 8), DISC_R8(v, 16), DISC_R8(v, 24) : "r"(taddr) : "memory");
    }
}
template <int N>
__device__ __forceinline__ void tmem_st(uint32_t taddr, const uint32_t (&v)[N]) {
    static_assert(N == 8 || N == 16 || N == 32, "tcgen05.st shapes .x8 / .x16 / .x32");
    if constexpr (N == 8) {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                     :: "r"(taddr), DISC_I8(v, 0) : "memory");
    } else if constexpr (N == 16) {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
                     :: "r"(taddr), DISC_I8(v, 0), DISC_I8(v, 8) : "memory");
    } else {
        asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
                     "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
                     :: "r"(taddr), DISC_I8(v, 0), DISC_I8(v, 8), DISC_I8(v, 16), DISC_I8(v, 24) : "memory");
    }
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// sum of n fp64 values as a balanced tree (short dependency chains); overwrites t
template <int N>
__device__ __forceinline__ double tree_sum(double (&t)[N]) {
#pragma unroll
    for (int n = N; n > 1; n = (n + 1) / 2)
#pragma unroll
        for (int i = 0; i < n / 2; ++i) t[i] = t[i] + t[n - 1 - i];
    return t[0];
}

// sigma from the fp32 variance: var * rsqrt(var) with one Newton step on the reciprocal square root (the
// approximation's 2 ulp would otherwise be the largest term of the correction's error)
__device__ __forceinline__ float rsqrt_nr(float v) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(v));
    return y * fmaf(-0.5f * v * y, y, 1.5f);
}

template <int R, int TY, int MODE>
__global__ void __launch_bounds__(MomV3Cfg<R, TY>::NT, 1)
k_moments_v3(const __grid_constant__ CUtensorMap tmap, const float* __restrict__ pv, float* __restrict__ out0,
             float* __restrict__ out1, int nx, int ny, int nz, int rz, int zchunk, float eps_var, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    using C = MomV3Cfg<R, TY>;
    constexpr int W = C::W, PY = C::PY, PXB = C::PXB, LY = C::LY, XSP = C::XSP, TX = C::TX;
    constexpr int NYZ = C::NYZ, NXW = C::NXW, NSTG = C::NSTG, NXS = C::NXS;
    constexpr int RAWS = (int)(C::raw_stride / sizeof(float));
    constexpr int XSS = PY * XSP;                                    // one exchange buffer in double2
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* raw = reinterpret_cast<float*>(smem_raw);                                            // [NSTG][PY][PXB]
    double2* xs = reinterpret_cast<double2*>(smem_raw + (size_t)NSTG * C::raw_stride);           // [NXS][PY][XSP]
    __shared__ uint64_t raw_full[NSTG], raw_empty[NSTG], xs_full[NXS], xs_empty[NXS];
    __shared__ uint32_t tmem_base_s;
    __shared__ double inv_cnt_z[kMaxWz + 1];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const uint32_t zero = rt_zero(nx);
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, nz);
    const int wz = 2 * rz + 1;
    const int zfirst = max(z0 - rz, 0), zlast = min(z1 - 1 + rz, nz - 1);   // slices that exist; the others are zero
    const int T = zlast - zfirst + 1;
    const uint32_t tmem_cols = pow2_tmem_cols((uint32_t)(C::GROUPS * C::RING_WORDS * wz));

    // The producer thread sets up its own barriers and has the first NSTG slices on their way before the CTA-wide
    // sync: the first load's latency (tensor-map fetch + DRAM) then overlaps the tensor-memory allocation, the zeroing
    // of the ring and the fp64 divisions of the set-up instead of following them.
    const int n_first = min(NSTG, T);
    if (tid == NYZ + 32 * NXW) {
        for (int i = 0; i < NSTG; ++i) { mbar_init(&raw_full[i], 1); mbar_init(&raw_empty[i], PY); }
        mbar_fence_init();
        for (int t = 0; t < n_first; ++t) {
            mbar_expect_tx(&raw_full[t], (uint32_t)C::raw_bytes);
            tma_load_3d(raw + t * RAWS, &tmap, x0 - C::RA, y0 - R, zfirst + t, &raw_full[t]);
        }
    }
    if (tid == 0) {
        for (int i = 0; i < NXS; ++i) { mbar_init(&xs_full[i], PY); mbar_init(&xs_empty[i], NYZ); }
        mbar_fence_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                     "r"(tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid <= wz) inv_cnt_z[tid] = tid > 0 ? 1.0 / (double)tid : 0.0;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = tmem_base_s;

    if (warp < NYZ / 32) {
        // ------------------------------------------------------------------ y pass, z window, evaluation
        const int yb = warp * LY;
        const int gx = x0 + lane;
        // this thread's ring: its own lane of the warp's TMEM quadrant, RING_WORDS words per slice
        const uint32_t ring0 = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(warp >> 2) * (uint32_t)(C::RING_WORDS * wz);
        {
            uint32_t zero[C::RING_WORDS];
#pragma unroll
            for (int i = 0; i < C::RING_WORDS; ++i) zero[i] = 0u;
            for (int j = 0; j < wz; ++j) tmem_st<C::RING_WORDS>(ring0 + j * C::RING_WORDS, zero);
        }
        double Z1[LY], Z2[LY], cxy[LY];
        const int cx = min(gx + R, nx - 1) - max(gx - R, 0) + 1;
        bool live[LY];
        int ro[LY];       // row offsets of the thread's voxels (rows outside the volume alias row 0: loads stay legal)
#pragma unroll
        for (int o = 0; o < LY; ++o) {
            Z1[o] = 0.0; Z2[o] = 0.0;
            const int gy = y0 + yb + o;
            const int cy = min(gy + R, ny - 1) - max(gy - R, 0) + 1;
            live[o] = gx < nx && gy < ny;
            cxy[o] = live[o] ? 1.0 / ((double)cx * (double)cy) : 0.0;
            ro[o] = live[o] ? o * nx : 0;
        }
        double inv_n_full[LY];      // 1/n of a voxel whose z window lies wholly inside the volume
        float inv_nf_full[LY];
#pragma unroll
        for (int o = 0; o < LY; ++o) { inv_n_full[o] = cxy[o] * (1.0 / (double)wz); inv_nf_full[o] = (float)inv_n_full[o]; }
        // the thread's first voxel at slice z0 (clamped into the volume); the pointers advance one slice per emit
        const size_t plane = (size_t)nx * ny;
        const size_t off = (size_t)z0 * plane + (size_t)min(y0 + yb, ny - 1) * nx + min(gx, nx - 1);
        const float* pp = pv + off;
        float* po0 = out0 + off;
        float* po1 = MODE == kModeMoments ? out1 + off : nullptr;
        const double2* xq = xs + yb * XSP + lane;
        uint32_t slot = ring0;
        const uint32_t ring_end = ring0 + (uint32_t)(C::RING_WORDS * wz);
        int tv = 0;
        for (int zz = z0 - rz; zz < z1 + rz; ++zz) {
            const bool valid = zz >= 0 && zz < nz;   // uniform
            const int zo = zz - rz;
            const bool emit = zo >= z0;              // uniform
            uint32_t old[C::RING_WORDS];
            tmem_wait_st();                          // the slot written wz slices ago has landed
            tmem_ld<C::RING_WORDS>(slot, old);
            float pre[LY];
            if (MODE != kModeMoments && emit) {
#pragma unroll
                for (int o = 0; o < LY; ++o) pre[o] = __ldg(pp + ro[o]);
                pp += plane;
            }
            uint32_t nw[C::RING_WORDS];
            if (valid) {
                const int buf = tv % NXS;
                mbar_wait(&xs_full[buf], (tv / NXS) & 1);
                const double2* ip = xq + buf * XSS;
                double2 v[LY + 2 * R];
#pragma unroll
                for (int i = 0; i < LY + 2 * R; ++i) v[i] = ip[i * XSP];
                double t1[W], t2[W], b1[LY], b2[LY];
#pragma unroll
                for (int i = 0; i < W; ++i) { t1[i] = v[i].x; t2[i] = v[i].y; }
                b1[0] = tree_sum(t1); b2[0] = tree_sum(t2);
#pragma unroll
                for (int o = 1; o < LY; ++o) {
                    b1[o] = b1[o - 1] + (v[o + 2 * R].x - v[o - 1].x);
                    b2[o] = b2[o - 1] + (v[o + 2 * R].y - v[o - 1].y);
                }
                // release the buffer only after the last use of what was loaded from it (the arrive carries a
                // register dependency on the sums: a load still in flight when the x pass overwrites is a race)
                mbar_arrive_after(&xs_empty[buf], ((uint32_t)__double2loint(b1[LY - 1]) ^ (uint32_t)__double2loint(b2[LY - 1])) & zero);
                ++tv;
                tmem_wait_ld();
#pragma unroll
                for (int o = 0; o < LY; ++o) {
                    Z1[o] += b1[o] - __hiloint2double((int)old[4 * o + 1], (int)old[4 * o]);
                    Z2[o] += b2[o] - __hiloint2double((int)old[4 * o + 3], (int)old[4 * o + 2]);
                    nw[4 * o] = (uint32_t)__double2loint(b1[o]); nw[4 * o + 1] = (uint32_t)__double2hiint(b1[o]);
                    nw[4 * o + 2] = (uint32_t)__double2loint(b2[o]); nw[4 * o + 3] = (uint32_t)__double2hiint(b2[o]);
                }
            } else {   // a slice beyond the volume: its box sums are zero
                tmem_wait_ld();
#pragma unroll
                for (int o = 0; o < LY; ++o) {
                    Z1[o] -= __hiloint2double((int)old[4 * o + 1], (int)old[4 * o]);
                    Z2[o] -= __hiloint2double((int)old[4 * o + 3], (int)old[4 * o + 2]);
                }
#pragma unroll
                for (int i = 0; i < C::RING_WORDS; ++i) nw[i] = 0u;
            }
            tmem_st<C::RING_WORDS>(slot, nw);
            slot += C::RING_WORDS;
            if (slot == ring_end) slot = ring0;
            if (emit) {   // uniform
                // the in-volume count n = cx cy cz; away from the z faces cz = 2 rz + 1 and 1/n is the thread's constant
                const int cz = min(zo + rz, nz - 1) - max(zo - rz, 0) + 1;
                double inv_n[LY];
                float inv_nf[LY];
                if (cz == wz) {   // uniform
#pragma unroll
                    for (int o = 0; o < LY; ++o) { inv_n[o] = inv_n_full[o]; inv_nf[o] = inv_nf_full[o]; }
                } else {
                    const double inv_cz = inv_cnt_z[cz];
#pragma unroll
                    for (int o = 0; o < LY; ++o) { inv_n[o] = cxy[o] * inv_cz; inv_nf[o] = (float)inv_n[o]; }
                }
#pragma unroll
                for (int o = 0; o < LY; ++o) {
                    // mu = S1/n, var = (S2 - S1 mu)/n: the cancellation in fp64, the division by n in fp32
                    const double mu = Z1[o] * inv_n[o];
                    const double nvar = fma(-Z1[o], mu, Z2[o]);
                    const float varf = fmaxf((float)nvar * inv_nf[o], 0.f);
                    float r0;
                    if (MODE == kModeMoments) {
                        r0 = (float)mu;
                    } else if (MODE == kModeZscore) {
                        const float dv = (float)((double)pre[o] - mu);
                        // reading A5: the threshold decision is taken on the fp64 variance
                        r0 = nvar * inv_n[o] > (double)eps_var ? dv * rsqrt_nr(varf) : 0.f;
                    } else {
                        // sigma_m: one MUFU; its 2^-23 relative error is 1e-5 HU on the corrected intensity, and 0 -> 0
                        r0 = fmaf(sqrt_approx(varf), pre[o], (float)mu);
                    }
                    if (live[o]) {
                        po0[ro[o]] = r0;
                        if (MODE == kModeMoments) po1[ro[o]] = varf;
                    }
                }
                po0 += plane;
                if (MODE == kModeMoments) po1 += plane;
            }
        }
        tmem_wait_st();
    } else if (warp < NYZ / 32 + NXW) {
        // ------------------------------------------------------------------ x pass
        const int xw = warp - NYZ / 32;
        const int n_tasks = T * PY;
        constexpr int O4 = C::OFF & ~3, O1 = C::OFF & 3;
        constexpr int NV = (O1 + C::PX + 3) / 4;
        for (int g = xw; g * 32 < n_tasks; g += NXW) {
            const int id = g * 32 + lane;
            const bool has = id < n_tasks;
            const int idc = has ? id : n_tasks - 1;
            const int t = idc / PY, r = idc - t * PY;
            const int t_lo = (g * 32) / PY, t_hi = min(g * 32 + 31, n_tasks - 1) / PY;   // uniform
            mbar_wait(&raw_full[t_lo % NSTG], (t_lo / NSTG) & 1);
            if (t_hi != t_lo) mbar_wait(&raw_full[t_hi % NSTG], (t_hi / NSTG) & 1);
            float rv[NV * 4];
            {
                const float4* rp = reinterpret_cast<const float4*>(raw + (t % NSTG) * RAWS + r * PXB + O4);
#pragma unroll
                for (int i = 0; i < NV; ++i) {
                    const float4 f = rp[i];
                    rv[4 * i] = f.x; rv[4 * i + 1] = f.y; rv[4 * i + 2] = f.z; rv[4 * i + 3] = f.w;
                }
            }
            if (t_lo >= NXS) mbar_wait(&xs_empty[t_lo % NXS], ((t_lo / NXS) - 1) & 1);
            if (t_hi != t_lo && t_hi >= NXS) mbar_wait(&xs_empty[t_hi % NXS], ((t_hi / NXS) - 1) & 1);
            // first window as balanced trees, then TX - 1 slides with the window's elements in a register ring
            double win[W], t1[W], t2[W];
#pragma unroll
            for (int i = 0; i < W; ++i) { win[i] = (double)rv[O1 + i]; t1[i] = win[i]; t2[i] = win[i] * win[i]; }
            double s1 = tree_sum(t1), s2 = tree_sum(t2);
            double2* op = xs + (t % NXS) * XSS + r * XSP;
            if (has) op[0] = make_double2(s1, s2);
#pragma unroll
            for (int o = 1; o < TX; ++o) {
                const double dn = (double)rv[O1 + o + 2 * R], dl = win[(o - 1) % W];
                const double e = dn - dl, f = dn + dl;
                s1 += e;
                s2 = fma(e, f, s2);
                win[(o - 1) % W] = dn;
                if (has) op[o] = make_double2(s1, s2);
            }
            if (has) {
                // the raw stage is released only after the last use of what was loaded from it (see the y/z pass)
                mbar_arrive_after(&raw_empty[t % NSTG], (uint32_t)__double2loint(s2) & zero);
                mbar_arrive(&xs_full[t % NXS]);
            }
        }
    } else if (tid == NYZ + 32 * NXW) {
        // ------------------------------------------------------------------ producer
        for (int t = n_first; t < T; ++t) {
            const int st = t % NSTG;
            mbar_wait(&raw_empty[st], ((t / NSTG) - 1) & 1);
            mbar_expect_tx(&raw_full[st], (uint32_t)C::raw_bytes);
            tma_load_3d(raw + st * RAWS, &tmap, x0 - C::RA, y0 - R, zfirst + t, &raw_full[st]);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
}

}  // namespace disc
