// field_tma.cuh -- TMA-fed versions of the two field kernels of field.cuh (same arithmetic, same results up to
// fp32 rounding order): input rows / slices are streamed into a shared-memory ring by 1-D bulk copies
// (cp.async.bulk -> UBLKCP) behind mbarriers, NS stages deep, so the bytes in flight per SM do not depend on
// registers or occupancy.  Each thread owns TWO adjacent columns: global stores are float2, the Gaussian taps
// are packed fp32x2 FMAs (FFMA2).  Requirements (checked by the launcher, which otherwise falls back to the
// plain-load kernels of field.cuh): nx % 4 == 0 and 16-byte aligned base pointers.
#pragma once
#include "common.cuh"
#include "pipeline.cuh"

namespace disc {

// ---------------------------------------------------------------------------------------------------------
// Gaussian z pass (+ warp).  CTA = 128 threads x 2 columns = 256 consecutive (x,y) columns, one z chunk.
// Stage = one slice of the three components (3 x 256 floats).
// ---------------------------------------------------------------------------------------------------------
constexpr int kGzCols = 256, kGzStages = 8;

template <int K, bool WARP>
__global__ void __launch_bounds__(128)
k_gz_warp_tma(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
              float* __restrict__ mout, int nx, int ny, int nz, int zchunk, GaussTaps gw) {
    constexpr int W = 2 * K + 1, NS = kGzStages, TC = kGzCols;
    __shared__ __align__(128) float stage[NS][3][TC];
    __shared__ uint64_t full[NS], empty[NS];

    const int tid = threadIdx.x;
    const size_t plane = (size_t)nx * ny, N = plane * nz;
    const size_t col0 = (size_t)blockIdx.x * TC;
    const int ncol = (int)min((size_t)TC, plane - col0);  // multiple of 4
    const int z0 = blockIdx.y * zchunk, z1 = min(z0 + zchunk, nz);
    const int T = (z1 - z0) + 2 * K;  // streamed slices: z0-K .. z1-1+K (clamped)

    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 4); }
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

    for (int tb = 0; tb < T; tb += W) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int t = tb + j;  // streamed slice t lives in ring slot j
            if (t >= T) break;
            if (tid == 0 && t + NS - 1 < T) issue(t + NS - 1);
            const int s = t % NS;
            mbar_wait(&full[s], (t / NS) & 1);
#pragma unroll
            for (int c = 0; c < 3; ++c) ring[c][j] = *reinterpret_cast<const float2*>(&stage[s][c][2 * tid]);
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(&empty[s]);
            if (t >= 2 * K && live) {
                // output slice z = z0 + t - 2K uses streamed slices t-2K .. t = slots (j+1+k) % W, k = 0..2K
                const int z = z0 + t - 2 * K;
                float2 r[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < W; ++k)
                        acc = ffma2(make_float2(gw.w[k], gw.w[k]), ring[c][(j + 1 + k) % W], acc);
                    r[c] = acc;
                }
                const size_t o = (size_t)z * plane + col;
#pragma unroll
                for (int c = 0; c < 3; ++c) *reinterpret_cast<float2*>(rout + c * N + o) = r[c];
                if (WARP) {
                    float2 mv;
                    mv.x = trilinear_clamped(moving, nx, ny, nz, (float)x + r[0].x, (float)y + r[1].x, (float)z + r[2].x);
                    mv.y = trilinear_clamped(moving, nx, ny, nz, (float)(x + 1) + r[0].y, (float)y + r[1].y, (float)z + r[2].y);
                    *reinterpret_cast<float2*>(mout + o) = mv;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// [force + update] + Gaussian x + Gaussian y.  CTA = NT threads x 2 columns = TX = 2*NT columns of one slice z,
// one y segment.  Stage = one input row of {r0, r1, r2, m, s(z), s(z-1), s(z+1)} over the aligned window
// [a0, a1) that covers the tile, the Gaussian halo K and the gradient halo 1.  The force at row y needs s rows
// y-1, y, y+1: they are three consecutive stages of the ring.
// ---------------------------------------------------------------------------------------------------------
constexpr int kFgStages = 6;

template <int K, bool FORCE, int NT>
struct FgCfg {
    static constexpr int TX = 2 * NT;
    static constexpr int SP = TX + ((2 * K + 8 + 3) & ~3);  // stage row pitch (floats), multiple of 4 (16-byte rows)
    static constexpr int NARR = FORCE ? 7 : 3;
    static constexpr int E = K & 1;                     // one pad element on the left keeps own pairs 8-byte aligned
    static constexpr int XP = TX + 2 * K + 2;           // x-pass row: [E pad][K halo][TX own][K halo][pad], even
    static constexpr size_t smem_bytes = sizeof(float) * ((size_t)kFgStages * NARR * SP + 2 * 3 * XP);
};

template <int K, bool FORCE, int NT>
__global__ void __launch_bounds__(NT)
k_force_gxy_tma(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ rin,
                float* __restrict__ rout, int nx, int ny, int nz, int yseg, float eps_den, GaussTaps gw) {
    using C = FgCfg<K, FORCE, NT>;
    constexpr int W = 2 * K + 1, NS = kFgStages, TX = C::TX, SP = C::SP, NARR = C::NARR, XP = C::XP, E = C::E;
    constexpr int NWARP = NT / 32;
    static_assert(2 * K <= NT, "halo duty needs 2K threads");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* stage = reinterpret_cast<float*>(smem_raw);                 // [NS][NARR][SP]
    float* xrow = stage + (size_t)NS * NARR * SP;                      // [2][3][XP]
    __shared__ uint64_t full[NS], empty[NS];

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TX;
    const int z = blockIdx.z;
    const int y0 = blockIdx.y * yseg, y1 = min(y0 + yseg, ny);
    const size_t plane = (size_t)nx * ny, N = plane * nz;
    // aligned window of columns held by a stage
    const int a0 = max(x0 - K - 1, 0) & ~3;
    const int a1 = min((min(x0 + TX + K + 1, nx) + 3) & ~3, nx);
    const uint32_t row_bytes = (uint32_t)(a1 - a0) * 4u;
    // centre rows yc0..yc1 are x-smoothed; the stream has one more row on each side for the y gradient
    const int yc0 = max(y0 - K, 0), yc1 = min(y1 - 1 + K, ny - 1);
    const int ya = FORCE ? max(yc0 - 1, 0) : yc0;
    const int yb = FORCE ? min(yc1 + 1, ny - 1) : yc1;
    const int T = yb - ya + 1;
    const int zm = max(z - 1, 0), zp = min(z + 1, nz - 1);

    if (tid == 0) {
        for (int i = 0; i < NS; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NWARP); }
        mbar_fence_init();
    }
    for (int i = tid; i < 2 * 3 * XP; i += NT) xrow[i] = 0.f;   // pad elements meet zero taps: keep them finite
    __syncthreads();

    auto issue = [&](int t) {  // thread 0 only: stream row t (= volume row ya + t) -> stage t % NS
        const int st = t % NS;
        if (t >= NS) mbar_wait(&empty[st], ((t / NS) - 1) & 1);
        const int yy = ya + t;
        float* dst = stage + (size_t)st * NARR * SP;
        mbar_expect_tx(&full[st], NARR * row_bytes);
        const size_t o = (size_t)z * plane + (size_t)yy * nx + a0;
#pragma unroll
        for (int c = 0; c < 3; ++c) tma_load_1d(dst + c * SP, rin + c * N + o, row_bytes, &full[st]);
        if (FORCE) {
            tma_load_1d(dst + 3 * SP, m + o, row_bytes, &full[st]);
            tma_load_1d(dst + 4 * SP, s + o, row_bytes, &full[st]);
            tma_load_1d(dst + 5 * SP, s + (size_t)zm * plane + (size_t)yy * nx + a0, row_bytes, &full[st]);
            tma_load_1d(dst + 6 * SP, s + (size_t)zp * plane + (size_t)yy * nx + a0, row_bytes, &full[st]);
        }
    };
    int issued = 0;   // thread 0: stream rows [0, issued) have been requested
    int waited = 0;   // every thread: stream rows [0, waited) are known to have landed
    if (tid == 0)
        for (; issued < min(NS - 1, T); ++issued) issue(issued);

    // this thread's two columns and its halo duty, window-relative and clamped to the volume
    const int xa = x0 + 2 * tid;
    const int xl0 = min(xa, nx - 1) - a0, xl1 = min(xa + 1, nx - 1) - a0;
    const bool halo = tid < 2 * K;
    const int hx = clampi(tid < K ? x0 - K + tid : x0 + TX + (tid - K), 0, nx - 1) - a0;
    const int hslot = E + (tid < K ? tid : TX + tid);    // position in the x-pass row
    const int xmax = nx - 1 - a0;                        // window-relative index of the last column

    // updated field at window-relative column xl; c/u/d = stages of rows y, clamp(y-1), clamp(y+1)
    auto updated = [&](const float* c, const float* u, const float* d, int xl, float out[3]) {
        out[0] = c[0 * SP + xl]; out[1] = c[1 * SP + xl]; out[2] = c[2 * SP + xl];
        if (FORCE) {
            const float* sc = c + 4 * SP;
            const float gx = 0.5f * (sc[min(xl + 1, xmax)] - sc[max(xl - 1, 0)]);
            const float gy = 0.5f * (d[4 * SP + xl] - u[4 * SP + xl]);
            const float gz = 0.5f * (c[6 * SP + xl] - c[5 * SP + xl]);
            const float dd = sc[xl] - c[3 * SP + xl];
            const float den = fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, fmaf(dd, dd, eps_den))));
            const float q = __fdividef(dd, den);
            out[0] = fmaf(q, gx, out[0]); out[1] = fmaf(q, gy, out[1]); out[2] = fmaf(q, gz, out[2]);
        }
    };

    auto tap = [&](int i) { return (i >= 0 && i < W) ? gw.w[min(max(i, 0), W - 1)] : 0.f; };  // i is compile-time after unrolling
    float2 ring[3][W];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < W; ++j) ring[c][j] = make_float2(0.f, 0.f);
    float2 xs[3] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
    int last_row = -1, buf = 0;

    const int yend = y1 + K;
    for (int yb0 = y0 - K; yb0 < yend; yb0 += W) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int yy = yb0 + j;  // ring push event: row yy (replicated outside the volume) -> slot j
            if (yy >= yend) break;
            const int yr = clampi(yy, 0, ny - 1);
            if (yr != last_row) {    // uniform over the CTA: a new centre row has to be x-smoothed
                last_row = yr;
                const int tc = yr - ya;                                  // stream index of the centre row
                const int need = FORCE ? min(tc + 1, T - 1) : tc;        // last stream row this centre row reads
                if (tid == 0)
                    for (; issued < T && issued <= need + NS - 3; ++issued) issue(issued);
                for (; waited <= need; ++waited) mbar_wait(&full[waited % NS], (waited / NS) & 1);
                const float* c = stage + (size_t)(tc % NS) * NARR * SP;
                const float* u = stage + (size_t)(max(tc - 1, 0) % NS) * NARR * SP;
                const float* d = stage + (size_t)(min(tc + 1, T - 1) % NS) * NARR * SP;
                float* xr = xrow + (size_t)buf * 3 * XP;
                float v0[3], v1[3];
                updated(c, u, d, xl0, v0);
                updated(c, u, d, xl1, v1);
#pragma unroll
                for (int cc = 0; cc < 3; ++cc)
                    *reinterpret_cast<float2*>(&xr[cc * XP + E + K + 2 * tid]) = make_float2(v0[cc], v1[cc]);
                if (halo) {
                    float h[3];
                    updated(c, u, d, hx, h);
#pragma unroll
                    for (int cc = 0; cc < 3; ++cc) xr[cc * XP + hslot] = h[cc];
                }
                __syncthreads();   // x-pass row complete; every thread is also done reading stream row tc-1
                if ((tid & 31) == 0) {
                    if (FORCE) { if (tc >= 1) mbar_arrive(&empty[(tc - 1) % NS]); }
                    else mbar_arrive(&empty[tc % NS]);
                }
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) {
                    // row index i <-> column x0 - K - E + i; output 0 (column 2*tid) uses i = 2*tid + E + k,
                    // output 1 uses i = 2*tid + E + 1 + k, k = 0..2K.  With aligned pairs P_q = (v[2q], v[2q+1]):
                    // out0 = sum_q (w(2q-E), w(2q+1-E)) . P_q,  out1 = sum_q (w(2q-E-1), w(2q-E)) . P_q
                    const float2* p = reinterpret_cast<const float2*>(&xr[cc * XP + 2 * tid]);
                    float2 acc0 = make_float2(0.f, 0.f), acc1 = make_float2(0.f, 0.f);
#pragma unroll
                    for (int q = 0; q <= K + E; ++q) {
                        const float2 P = p[q];
                        const int i0 = 2 * q - E;
                        const float wm = tap(i0 - 1), wa = tap(i0), wb = tap(i0 + 1);
                        acc0 = ffma2(make_float2(wa, wb), P, acc0);
                        acc1 = ffma2(make_float2(wm, wa), P, acc1);
                    }
                    xs[cc] = make_float2(acc0.x + acc0.y, acc1.x + acc1.y);
                }
                buf ^= 1;
            }
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) ring[cc][j] = xs[cc];
            const int yo = yy - K;
            if (yo >= y0 && xa < nx) {
                const size_t o = (size_t)z * plane + (size_t)yo * nx + xa;
#pragma unroll
                for (int cc = 0; cc < 3; ++cc) {
                    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < W; ++k)
                        acc = ffma2(make_float2(gw.w[k], gw.w[k]), ring[cc][(j + 1 + k) % W], acc);
                    *reinterpret_cast<float2*>(rout + cc * N + o) = acc;
                }
            }
        }
    }
}

}  // namespace disc
