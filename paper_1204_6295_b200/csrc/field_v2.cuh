// field_v2.cuh -- the two field kernels of the iteration, second generation (same arithmetic as field.cuh /
// field_tma.cuh, same results up to fp32 rounding order):
//   k_gz_warp_v2<K, WARP>     Gaussian z pass of the scratch field -> r, [then m = ct(x + r(x))]
//   k_force_gxy_v2<K, FORCE>  [r += force(m, s')], Gaussian x pass, Gaussian y pass -> scratch field
//
// What changed against the first generation, and why (profiles/r01a_*): those kernels ran 7-11 warps per SM,
// replicated their whole loop body 2K+1 times (instruction-cache misses) and consumed the warp's eight
// gathered loads in the instruction right after issuing them.  Here
//   * only the register-ring part (ring push + the 2K+1 packed FMAs per component) is specialised per ring
//     phase, through a uniform `switch`; everything else exists once;
//   * the trilinear gather is software-pipelined: the loads of slice z are issued, the z pass of slice z+1
//     runs, then the loads are consumed -- their latency is hidden inside the thread;
//   * CTAs are small (64 threads x 2 columns) so that one wave of CTAs fills every SM evenly.
// Input slices / rows still arrive by 1-D bulk TMA copies (cp.async.bulk -> UBLKCP) behind mbarriers.
#pragma once
#include "common.cuh"
#include "field.cuh"
#include "pipeline.cuh"

namespace disc {

__device__ __forceinline__ float wfma(float w, float a, float acc) { return fmaf(w, a, acc); }
__device__ __forceinline__ float2 wfma(float w, float2 a, float2 acc) { return ffma2(make_float2(w, w), a, acc); }
__device__ __forceinline__ void vzero(float& a) { a = 0.f; }
__device__ __forceinline__ void vzero(float2& a) { a = make_float2(0.f, 0.f); }

// ring[c][J] <- v[c]; if OUT, r[c] = sum_k w[k] * ring[c][(J + 1 + k) % W]   (all ring indices are compile-time)
// T = float2: two adjacent columns per thread, packed FFMA2; T = float: one column per thread.
template <int K, int J, typename T>
__device__ __forceinline__ void ring_push_conv(T (&ring)[3][2 * K + 1], const T (&v)[3], const GaussTaps& gw, bool out,
                                               T (&r)[3]) {
    constexpr int W = 2 * K + 1;
#pragma unroll
    for (int c = 0; c < 3; ++c) ring[c][J] = v[c];
    if (out) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            T acc;
            vzero(acc);
#pragma unroll
            for (int k = 0; k < W; ++k) acc = wfma(gw.w[k], ring[c][(J + 1 + k) % W], acc);
            r[c] = acc;
        }
    }
}

template <int K, typename T>
__device__ __forceinline__ void ring_step(int j, T (&ring)[3][2 * K + 1], const T (&v)[3], const GaussTaps& gw, bool out,
                                          T (&r)[3]) {
    static_assert(K <= 12, "ring_step enumerates 25 phases");
    switch (j) {   // uniform over the CTA
#define DISC_RS(J) \
    case J:        \
        if constexpr (J < 2 * K + 1) ring_push_conv<K, (J < 2 * K + 1 ? J : 0), T>(ring, v, gw, out, r); \
        break;
        DISC_RS(0) DISC_RS(1) DISC_RS(2) DISC_RS(3) DISC_RS(4) DISC_RS(5) DISC_RS(6) DISC_RS(7) DISC_RS(8)
        DISC_RS(9) DISC_RS(10) DISC_RS(11) DISC_RS(12) DISC_RS(13) DISC_RS(14) DISC_RS(15) DISC_RS(16)
        DISC_RS(17) DISC_RS(18) DISC_RS(19) DISC_RS(20) DISC_RS(21) DISC_RS(22) DISC_RS(23) DISC_RS(24)
#undef DISC_RS
        default: break;
    }
}

// The eight neighbours and three weights of one trilinear sample (reading A11), split in two halves so that the
// loads can be issued long before they are used.
struct TriSample {
    float a[8];
    float tx, ty, tz;
};

// FAST: every axis has at least two voxels (checked once per kernel, uniform), so the neighbour offsets are the
// constants +1, +nx, +plane and the eight addresses share four row pointers.
template <bool FAST>
__device__ __forceinline__ void tri_issue(const float* __restrict__ I, int nx, int ny, int nz, float px, float py,
                                          float pz, TriSample& s) {
    px = fminf(fmaxf(px, 0.f), (float)(nx - 1));
    py = fminf(fmaxf(py, 0.f), (float)(ny - 1));
    pz = fminf(fmaxf(pz, 0.f), (float)(nz - 1));
    if (FAST) {
        const int x0 = min((int)px, nx - 2), y0 = min((int)py, ny - 2), z0 = min((int)pz, nz - 2);
        s.tx = px - (float)x0; s.ty = py - (float)y0; s.tz = pz - (float)z0;
        const float* p00 = I + ((size_t)(unsigned)((z0 * ny + y0) * nx + x0));
        const float* p10 = p00 + nx;
        const float* p01 = p00 + (size_t)nx * ny;
        const float* p11 = p01 + nx;
        s.a[0] = __ldg(p00); s.a[1] = __ldg(p00 + 1);
        s.a[2] = __ldg(p10); s.a[3] = __ldg(p10 + 1);
        s.a[4] = __ldg(p01); s.a[5] = __ldg(p01 + 1);
        s.a[6] = __ldg(p11); s.a[7] = __ldg(p11 + 1);
    } else {
        const int x0 = max(min((int)px, nx - 2), 0), y0 = max(min((int)py, ny - 2), 0), z0 = max(min((int)pz, nz - 2), 0);
        const int dx = nx > 1 ? 1 : 0;
        const int dy = ny > 1 ? nx : 0;
        const size_t dz = nz > 1 ? (size_t)nx * ny : 0;
        s.tx = px - (float)x0; s.ty = py - (float)y0; s.tz = pz - (float)z0;
        const float* p = I + ((size_t)z0 * ny + y0) * nx + x0;
        s.a[0] = __ldg(p); s.a[1] = __ldg(p + dx);
        s.a[2] = __ldg(p + dy); s.a[3] = __ldg(p + dy + dx);
        s.a[4] = __ldg(p + dz); s.a[5] = __ldg(p + dz + dx);
        s.a[6] = __ldg(p + dz + dy); s.a[7] = __ldg(p + dz + dy + dx);
    }
}

__device__ __forceinline__ float tri_finish(const TriSample& s) {
    // (1-t)*a + t*b: exact at t = 0 and t = 1, so a zero field reproduces the input bit for bit
    const float ux = 1.f - s.tx, uy = 1.f - s.ty, uz = 1.f - s.tz;
    const float c00 = fmaf(s.tx, s.a[1], ux * s.a[0]);
    const float c10 = fmaf(s.tx, s.a[3], ux * s.a[2]);
    const float c01 = fmaf(s.tx, s.a[5], ux * s.a[4]);
    const float c11 = fmaf(s.tx, s.a[7], ux * s.a[6]);
    const float c0 = fmaf(s.ty, c10, uy * c00);
    const float c1 = fmaf(s.ty, c11, uy * c01);
    return fmaf(s.tz, c1, uz * c0);
}

// ---------------------------------------------------------------------------------------------------------
// Gaussian z pass (+ warp).  CTA = 64 threads x 2 columns = 128 consecutive (x,y) columns, one z chunk.
// Stage = one slice of the three components (3 x 128 floats).
// ---------------------------------------------------------------------------------------------------------
constexpr int kGz2Threads = 64, kGz2Cols = 2 * kGz2Threads, kGz2Stages = 8;
constexpr int kWarpPrefetch = 3;   // the warp's moving-image lines are prefetched this many slices ahead

// 4-byte asynchronous copy global -> shared (LDGSTS), used as a register-free prefetch through L1
__device__ __forceinline__ void cp_async4(void* dst_smem, const void* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}

template <int K, bool WARP>
__global__ void __launch_bounds__(kGz2Threads, 8)
k_gz_warp_v2(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
             float* __restrict__ mout, int nx, int ny, int nz, int zchunk, GaussTaps gw) {
    constexpr int W = 2 * K + 1, NS = kGz2Stages, TC = kGz2Cols, NWARP = kGz2Threads / 32;
    __shared__ __align__(128) float stage[NS][3][TC];
    __shared__ uint64_t full[NS], empty[NS];
    __shared__ float pf_sink[2 * kGz2Threads];   // landing zone of the prefetch copies, never read

    const int tid = threadIdx.x;
    const size_t plane = (size_t)nx * ny, N = plane * nz;
    const size_t col0 = (size_t)blockIdx.x * TC;
    const int ncol = (int)min((size_t)TC, plane - col0);  // multiple of 4
    const int z0 = blockIdx.y * zchunk, z1 = min(z0 + zchunk, nz);
    const int T = (z1 - z0) + 2 * K;  // streamed slices: z0-K .. z1-1+K (clamped)

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARP); }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int t) {  // thread 0 only
        const int s = t % NS;
        if (t >= NS) mbar_wait(&empty[s], ((t / NS) - 1) & 1);
        const int zz = clampi(z0 - K + t, 0, nz - 1);
        const uint32_t bytes = (uint32_t)ncol * 4u;
        mbar_expect_tx(&full[s], 3 * bytes);
        const float* src = rin + (size_t)zz * plane + col0;
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_load_1d(&stage[s][c][0], src + c * N, bytes, &full[s]);
    };
    if (tid == 0)
        for (int t = 0; t < min(NS - 1, T); ++t) issue(t);

    // threads beyond the plane's last column work on the last pair and store nothing
    const bool live = 2 * tid < ncol;
    const int tcol = live ? 2 * tid : max(ncol - 2, 0);
    const size_t col = col0 + tcol;
    const int y = (int)(col / nx), x = (int)(col - (size_t)y * nx);  // both columns share y (nx is even)
    const float fx0 = (float)x, fx1 = (float)(x + 1), fy = (float)y;
    // 32-bit voxel indices in the fast gather path
    const bool fast = nx > 1 && ny > 1 && nz > 1 && N < (size_t)0x7fffffff;

    float2 ring[3][W];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < W; ++j) ring[c][j] = make_float2(0.f, 0.f);

    int j = 0;
    for (int t = 0; t < T; ++t) {
        if (tid == 0 && t + NS - 1 < T) issue(t + NS - 1);
        const int s = t % NS;
        mbar_wait(&full[s], (t / NS) & 1);
        float2 v[3], r[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = *reinterpret_cast<const float2*>(&stage[s][c][tcol]);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        const bool out = t >= 2 * K;
        ring_step<K, float2>(j, ring, v, gw, out, r);
        j = j + 1 == W ? 0 : j + 1;
        if (out) {
            const int z = z0 + t - 2 * K;
            const size_t o = (size_t)z * plane + col;
            if (live) {
#pragma unroll
                for (int c = 0; c < 3; ++c) *reinterpret_cast<float2*>(rout + c * N + o) = r[c];
            }
            if (WARP) {
                TriSample g0, g1;
                if (fast) {
                    // The field is smooth along z: the sample of slice z + kWarpPrefetch will land close to this
                    // one, kWarpPrefetch planes further.  Pull the two rows of the plane it newly touches towards
                    // L1 now (asynchronous 4-byte copies into a sink), so that those gathers do not wait for HBM.
                    const int xq = clampi((int)(fx0 + r[0].x), 0, nx - 1);
                    const int yq = clampi((int)(fy + r[1].x), 0, ny - 2);
                    const int zq = clampi((int)((float)z + r[2].x) + 1 + kWarpPrefetch, 0, nz - 1);
                    const float* q = moving + (size_t)(unsigned)((zq * ny + yq) * nx + xq);
                    cp_async4(&pf_sink[2 * tid], q);
                    cp_async4(&pf_sink[2 * tid + 1], q + nx);
                    tri_issue<true>(moving, nx, ny, nz, fx0 + r[0].x, fy + r[1].x, (float)z + r[2].x, g0);
                    tri_issue<true>(moving, nx, ny, nz, fx1 + r[0].y, fy + r[1].y, (float)z + r[2].y, g1);
                } else {
                    tri_issue<false>(moving, nx, ny, nz, fx0 + r[0].x, fy + r[1].x, (float)z + r[2].x, g0);
                    tri_issue<false>(moving, nx, ny, nz, fx1 + r[0].y, fy + r[1].y, (float)z + r[2].y, g1);
                }
                const float2 mv = make_float2(tri_finish(g0), tri_finish(g1));
                if (live) *reinterpret_cast<float2*>(mout + o) = mv;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// One column per thread: a 39-register ring instead of 78, so 28 warps per SM instead of 16.  The z pass + warp is
// bound by the latency of the warp's gathers (profiles/r01b), which only resident warps can hide; the extra
// scalar FMAs are free in that regime.  CTA = 128 threads = 128 consecutive (x,y) columns, one z chunk.
// ---------------------------------------------------------------------------------------------------------
constexpr int kGz1Threads = 128, kGz1Stages = 8;

template <int K, bool WARP>
__global__ void __launch_bounds__(kGz1Threads, 7)
k_gz_warp_c1(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
             float* __restrict__ mout, int nx, int ny, int nz, int zchunk, GaussTaps gw) {
    constexpr int W = 2 * K + 1, NS = kGz1Stages, TC = kGz1Threads, NWARP = kGz1Threads / 32;
    __shared__ __align__(128) float stage[NS][3][TC];
    __shared__ uint64_t full[NS], empty[NS];

    const int tid = threadIdx.x;
    const size_t plane = (size_t)nx * ny, N = plane * nz;
    const size_t col0 = (size_t)blockIdx.x * TC;
    const int ncol = (int)min((size_t)TC, plane - col0);  // multiple of 4
    const int z0 = blockIdx.y * zchunk, z1 = min(z0 + zchunk, nz);
    const int T = (z1 - z0) + 2 * K;  // streamed slices: z0-K .. z1-1+K (clamped)

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARP); }
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int t) {  // thread 0 only
        const int s = t % NS;
        if (t >= NS) mbar_wait(&empty[s], ((t / NS) - 1) & 1);
        const int zz = clampi(z0 - K + t, 0, nz - 1);
        const uint32_t bytes = (uint32_t)ncol * 4u;
        mbar_expect_tx(&full[s], 3 * bytes);
        const float* src = rin + (size_t)zz * plane + col0;
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_load_1d(&stage[s][c][0], src + c * N, bytes, &full[s]);
    };
    if (tid == 0)
        for (int t = 0; t < min(NS - 1, T); ++t) issue(t);

    const bool live = tid < ncol;
    const int tcol = live ? tid : max(ncol - 1, 0);
    const size_t col = col0 + tcol;
    const int y = (int)(col / nx), x = (int)(col - (size_t)y * nx);
    const float fx = (float)x, fy = (float)y;
    const bool fast = nx > 1 && ny > 1 && nz > 1 && N < (size_t)0x7fffffff;

    float ring[3][W];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < W; ++j) ring[c][j] = 0.f;

    int j = 0;
    for (int t = 0; t < T; ++t) {
        if (tid == 0 && t + NS - 1 < T) issue(t + NS - 1);
        const int s = t % NS;
        mbar_wait(&full[s], (t / NS) & 1);
        float v[3], r[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = stage[s][c][tcol];
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        const bool out = t >= 2 * K;
        ring_step<K, float>(j, ring, v, gw, out, r);
        j = j + 1 == W ? 0 : j + 1;
        if (out) {
            const int z = z0 + t - 2 * K;
            const size_t o = (size_t)z * plane + col;
            if (live) {
#pragma unroll
                for (int c = 0; c < 3; ++c) rout[c * N + o] = r[c];
            }
            if (WARP) {
                TriSample g;
                if (fast) tri_issue<true>(moving, nx, ny, nz, fx + r[0], fy + r[1], (float)z + r[2], g);
                else tri_issue<false>(moving, nx, ny, nz, fx + r[0], fy + r[1], (float)z + r[2], g);
                const float mv = tri_finish(g);
                if (live) mout[o] = mv;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// [force + update] + Gaussian x + Gaussian y as a TILE kernel: no marching, no ring, every CTA independent.
//
// CTA = 256 threads, one 64 x 32 (x,y) tile of one slice z.
//   phase 1  u = r [+ force] at the (64+2K) x (32+2K) points around the tile, coordinates clamped to the volume
//            (that IS the replicate border of the Gaussian, reading A10); one point per thread and step, rows
//            coalesced; -> shared memory U[3][32+2K][64+2K]
//   phase 2  x pass: task = (component, row, run of 8 outputs), lanes <-> rows: 5 LDS.128, 8x(2K+1) FMAs
//            -> shared memory X[3][32+2K][64]
//   phase 3  y pass: task = (component, 4 adjacent columns, run of 8 rows), lanes <-> columns: 8+2K LDS.128,
//            packed FMAs on column pairs, 8 coalesced float4 stores
// Halo work (force and x pass on 2K extra rows) is recomputed per tile; in exchange the grid has thousands of
// independent CTAs at every pyramid level and no serial row-by-row latency chain.
// Requirements (launcher): nx % 4 == 0, 16-byte aligned rout.
// ---------------------------------------------------------------------------------------------------------
template <int K>
struct FgTileCfg {
    static constexpr int TX = 64, TY = 32, NT = 256, LX = 8, LY = 8;
    static constexpr int W = 2 * K + 1;
    static constexpr int PX = TX + 2 * K, PY = TY + 2 * K;
    static constexpr int UP = (((PX + 3) / 4) | 1) * 4;          // U row pitch: multiple of 4 floats, odd number of 16-byte chunks
    static constexpr int XP = TX + 4;                            // X row pitch: 17 chunks (odd)
    static constexpr int P2_TASKS = 3 * PY * (TX / LX);
    static constexpr int P3_TASKS = 3 * (TX / 4) * (TY / LY);
    static constexpr size_t smem_bytes = sizeof(float) * 3 * PY * (UP + XP);
    static constexpr int NV = (LX + 2 * K + 3) / 4;              // float4 chunks of one x-pass run (the last may overhang
                                                                 // into the row's padding: g*LX + 4*NV <= UP)
    static_assert(2 * K <= 24 && (TX - LX) + 4 * NV <= UP, "x-pass run must stay inside the padded U row");
};

template <int K, bool FORCE>
__global__ void __launch_bounds__(FgTileCfg<K>::NT, 2)
k_force_gxy_tile(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ rin,
                 float* __restrict__ rout, int nx, int ny, int nz, float eps_den, GaussTaps gw) {
    using C = FgTileCfg<K>;
    constexpr int W = C::W, TX = C::TX, TY = C::TY, NT = C::NT, LX = C::LX, LY = C::LY, PX = C::PX, PY = C::PY;
    constexpr int UP = C::UP, XP = C::XP;
    extern __shared__ __align__(16) float smem_f[];
    float* U = smem_f;                       // [3][PY][UP]
    float* X = smem_f + 3 * PY * UP;         // [3][PY][XP]

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z = blockIdx.z;
    const size_t N = (size_t)nx * ny * nz;

    // ---- phase 1: updated field at the tile + halo, replicate border through clamped coordinates
    for (int p = tid; p < PY * PX; p += NT) {
        const int r = p / PX, c = p - r * PX;
        const int gx = clampi(x0 - K + c, 0, nx - 1), gy = clampi(y0 - K + r, 0, ny - 1);
        float u[3];
        updated_field<FORCE>(m, s, rin, nx, ny, nz, N, gx, gy, z, eps_den, u);
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) U[(cc * PY + r) * UP + c] = u[cc];
    }
    __syncthreads();

    // ---- phase 2: x pass, lanes <-> rows
    for (int t = tid; t < C::P2_TASKS; t += NT) {
        const int r = t % PY, q = t / PY, g = q % (TX / LX), cc = q / (TX / LX);
        const float4* up = reinterpret_cast<const float4*>(U + (cc * PY + r) * UP + g * LX);
        float v[4 * C::NV];
#pragma unroll
        for (int i = 0; i < C::NV; ++i) {
            const float4 f = up[i];
            v[4 * i] = f.x; v[4 * i + 1] = f.y; v[4 * i + 2] = f.z; v[4 * i + 3] = f.w;
        }
        float o[LX];
#pragma unroll
        for (int j = 0; j < LX; ++j) {
            float acc = 0.f;
#pragma unroll
            for (int k = 0; k < W; ++k) acc = fmaf(gw.w[k], v[j + k], acc);
            o[j] = acc;
        }
        float4* xp = reinterpret_cast<float4*>(X + (cc * PY + r) * XP + g * LX);
        xp[0] = make_float4(o[0], o[1], o[2], o[3]);
        xp[1] = make_float4(o[4], o[5], o[6], o[7]);
    }
    __syncthreads();

    // ---- phase 3: y pass, lanes <-> column groups
    for (int t = tid; t < C::P3_TASKS; t += NT) {
        const int cg = t % (TX / 4), q = t / (TX / 4), h = q % (TY / LY), cc = q / (TY / LY);
        const float4* xp = reinterpret_cast<const float4*>(X + (cc * PY + h * LY) * XP + cg * 4);
        float2 a0[LY], a1[LY];
#pragma unroll
        for (int j = 0; j < LY; ++j) { a0[j] = make_float2(0.f, 0.f); a1[j] = make_float2(0.f, 0.f); }
#pragma unroll
        for (int i = 0; i < LY + 2 * K; ++i) {
            const float4 f = xp[i * (XP / 4)];
            const float2 lo = make_float2(f.x, f.y), hi = make_float2(f.z, f.w);
#pragma unroll
            for (int j = 0; j < LY; ++j) {
                const int k = i - j;          // input row i contributes to output row j with tap k
                if (k >= 0 && k < W) {
                    const float2 w2 = make_float2(gw.w[k], gw.w[k]);
                    a0[j] = ffma2(w2, lo, a0[j]);
                    a1[j] = ffma2(w2, hi, a1[j]);
                }
            }
        }
        const int gx = x0 + cg * 4;
        if (gx < nx) {
            float* op = rout + cc * N + ((size_t)z * ny + (y0 + h * LY)) * nx + gx;
#pragma unroll
            for (int j = 0; j < LY; ++j)
                if (y0 + h * LY + j < ny)
                    *reinterpret_cast<float4*>(op + (size_t)j * nx) = make_float4(a0[j].x, a0[j].y, a1[j].x, a1[j].y);
        }
    }
}

}  // namespace disc
