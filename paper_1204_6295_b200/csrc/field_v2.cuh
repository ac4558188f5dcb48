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
#include "pipeline.cuh"

namespace disc {

// ring[c][J] <- v[c]; if OUT, r[c] = sum_k w[k] * ring[c][(J + 1 + k) % W]   (all ring indices are compile-time)
template <int K, int J>
__device__ __forceinline__ void ring_push_conv(float2 (&ring)[3][2 * K + 1], const float2 (&v)[3], const GaussTaps& gw,
                                               bool out, float2 (&r)[3]) {
    constexpr int W = 2 * K + 1;
#pragma unroll
    for (int c = 0; c < 3; ++c) ring[c][J] = v[c];
    if (out) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int k = 0; k < W; ++k) acc = ffma2(make_float2(gw.w[k], gw.w[k]), ring[c][(J + 1 + k) % W], acc);
            r[c] = acc;
        }
    }
}

template <int K>
__device__ __forceinline__ void ring_step(int j, float2 (&ring)[3][2 * K + 1], const float2 (&v)[3], const GaussTaps& gw,
                                          bool out, float2 (&r)[3]) {
    static_assert(K <= 12, "ring_step enumerates 25 phases");
    switch (j) {   // uniform over the CTA
#define DISC_RS(J) \
    case J:        \
        if constexpr (J < 2 * K + 1) ring_push_conv<K, (J < 2 * K + 1 ? J : 0)>(ring, v, gw, out, r); \
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

__device__ __forceinline__ void tri_issue(const float* __restrict__ I, int nx, int ny, int nz, float px, float py,
                                          float pz, TriSample& s) {
    px = fminf(fmaxf(px, 0.f), (float)(nx - 1));
    py = fminf(fmaxf(py, 0.f), (float)(ny - 1));
    pz = fminf(fmaxf(pz, 0.f), (float)(nz - 1));
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

template <int K, bool WARP>
__global__ void __launch_bounds__(kGz2Threads, 7)
k_gz_warp_v2(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
             float* __restrict__ mout, int nx, int ny, int nz, int zchunk, GaussTaps gw) {
    constexpr int W = 2 * K + 1, NS = kGz2Stages, TC = kGz2Cols, NWARP = kGz2Threads / 32;
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

    const size_t col = col0 + 2 * tid;
    const bool live = 2 * tid < ncol;
    const int y = (int)(col / nx), x = (int)(col - (size_t)y * nx);  // both columns share y (nx is even)

    float2 ring[3][W];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < W; ++j) ring[c][j] = make_float2(0.f, 0.f);

    TriSample pend0, pend1;      // the gather in flight: columns x, x+1 of the previous output slice
    bool pending = false;
    size_t pend_o = 0;
    int j = 0;
    for (int t = 0; t < T; ++t) {
        if (tid == 0 && t + NS - 1 < T) issue(t + NS - 1);
        const int s = t % NS;
        mbar_wait(&full[s], (t / NS) & 1);
        float2 v[3], r[3];
#pragma unroll
        for (int c = 0; c < 3; ++c) v[c] = *reinterpret_cast<const float2*>(&stage[s][c][2 * tid]);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(&empty[s]);
        const bool out = t >= 2 * K;
        ring_step<K>(j, ring, v, gw, out, r);
        j = j + 1 == W ? 0 : j + 1;
        if (out && live) {
            const int z = z0 + t - 2 * K;
            const size_t o = (size_t)z * plane + col;
#pragma unroll
            for (int c = 0; c < 3; ++c) *reinterpret_cast<float2*>(rout + c * N + o) = r[c];
            if (WARP) {
                if (pending) *reinterpret_cast<float2*>(mout + pend_o) = make_float2(tri_finish(pend0), tri_finish(pend1));
                tri_issue(moving, nx, ny, nz, (float)x + r[0].x, (float)y + r[1].x, (float)z + r[2].x, pend0);
                tri_issue(moving, nx, ny, nz, (float)(x + 1) + r[0].y, (float)y + r[1].y, (float)z + r[2].y, pend1);
                pending = true;
                pend_o = o;
            }
        }
    }
    if (WARP && pending) *reinterpret_cast<float2*>(mout + pend_o) = make_float2(tri_finish(pend0), tri_finish(pend1));
}

}  // namespace disc
