// field.cuh -- the displacement-field kernels: force + update, Gaussian regularisation, warp.
//
// Steps (c) and (d) of an iteration plus the warp (b) that opens the next one:
//   k_force_gxy<K, FORCE> : [r += force(m, s')]  then the x and y Gaussian passes   -> scratch field
//   (the z Gaussian pass of the scratch field -> r, [then m = ct(x + r(x))] lives in field_v3.cuh)
// Fusing the force into the x/y passes and the warp into the z pass removes one read of r (12 B/voxel)
// and one read + one write of the un-smoothed field per iteration; the stand-alone variants
// (FORCE = false, WARP = false) serve disc_smooth_field.
//
// Force (Eq. 1, first term, with the corrected CBCT s'; readings A1, A2, A7, A8):
//   g = central difference of s' with clamped indices, d = s' - m, r_c += d g_c / (|g|^2 + d^2 + eps).
// Gaussian (reading A10): taps w[-K..K], replicate border, passes x, y, z.
// Both marching passes keep their (2K+1)-deep window in REGISTERS, statically indexed through a loop
// unrolled 2K+1 times; threads map to x so every global access is a coalesced row segment.
#pragma once
#include "common.cuh"

namespace disc {

// Force modes: none (plain field), the Thirion / passive force of north_star (c), and the double force = both terms
// of Eq. (1), which adds d grad(m) / (|grad m|^2 + d^2 + eps).
enum ForceMode { kForceNone = 0, kForceSingle = 1, kForceDouble = 2 };

// r_c(x,y,z) after the force update (or just r_c when MODE = kForceNone); x,y,z must be in range.
template <int MODE>
__device__ __forceinline__ void updated_field(const float* __restrict__ m, const float* __restrict__ s,
                                              const float* __restrict__ rin, int nx, int ny, int nz, size_t N,
                                              int x, int y, int z, float eps_den, float out[3]) {
    const size_t plane = (size_t)nx * ny;
    const size_t i = (size_t)z * plane + (size_t)y * nx + x;
    out[0] = __ldg(rin + i);
    out[1] = __ldg(rin + N + i);
    out[2] = __ldg(rin + 2 * N + i);
    if (MODE != kForceNone) {
        const size_t xp = i + (x < nx - 1 ? 1 : 0), xm = i - (x > 0 ? 1 : 0);
        const size_t yp = i + (y < ny - 1 ? (size_t)nx : 0), ym = i - (y > 0 ? (size_t)nx : 0);
        const size_t zp = i + (z < nz - 1 ? plane : 0), zm = i - (z > 0 ? plane : 0);
        const float gx = 0.5f * (__ldg(s + xp) - __ldg(s + xm));
        const float gy = 0.5f * (__ldg(s + yp) - __ldg(s + ym));
        const float gz = 0.5f * (__ldg(s + zp) - __ldg(s + zm));
        const float d = __ldg(s + i) - __ldg(m + i);
        const float dd = fmaf(d, d, eps_den);
        const float q = __fdividef(d, fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, dd))));
        out[0] = fmaf(q, gx, out[0]);
        out[1] = fmaf(q, gy, out[1]);
        out[2] = fmaf(q, gz, out[2]);
        if (MODE == kForceDouble) {
            const float hx = 0.5f * (__ldg(m + xp) - __ldg(m + xm));
            const float hy = 0.5f * (__ldg(m + yp) - __ldg(m + ym));
            const float hz = 0.5f * (__ldg(m + zp) - __ldg(m + zm));
            const float p = __fdividef(d, fmaf(hx, hx, fmaf(hy, hy, fmaf(hz, hz, dd))));
            out[0] = fmaf(p, hx, out[0]);
            out[1] = fmaf(p, hy, out[1]);
            out[2] = fmaf(p, hz, out[2]);
        }
    }
}

// The increment alone (no field): dr_c = d g_c / (|g|^2 + d^2 + eps) [+ d h_c / (|h|^2 + d^2 + eps)].
template <int MODE>
__device__ __forceinline__ void force_increment(const float* __restrict__ m, const float* __restrict__ s, int nx, int ny,
                                                int nz, int x, int y, int z, float eps_den, float dr[3]) {
    const size_t plane = (size_t)nx * ny;
    const size_t i = (size_t)z * plane + (size_t)y * nx + x;
    const size_t xp = i + (x < nx - 1 ? 1 : 0), xm = i - (x > 0 ? 1 : 0);
    const size_t yp = i + (y < ny - 1 ? (size_t)nx : 0), ym = i - (y > 0 ? (size_t)nx : 0);
    const size_t zp = i + (z < nz - 1 ? plane : 0), zm = i - (z > 0 ? plane : 0);
    const float gx = 0.5f * (__ldg(s + xp) - __ldg(s + xm));
    const float gy = 0.5f * (__ldg(s + yp) - __ldg(s + ym));
    const float gz = 0.5f * (__ldg(s + zp) - __ldg(s + zm));
    const float d = __ldg(s + i) - __ldg(m + i);
    const float dd = fmaf(d, d, eps_den);
    const float q = __fdividef(d, fmaf(gx, gx, fmaf(gy, gy, fmaf(gz, gz, dd))));
    dr[0] = q * gx; dr[1] = q * gy; dr[2] = q * gz;
    if (MODE == kForceDouble) {
        const float hx = 0.5f * (__ldg(m + xp) - __ldg(m + xm));
        const float hy = 0.5f * (__ldg(m + yp) - __ldg(m + ym));
        const float hz = 0.5f * (__ldg(m + zp) - __ldg(m + zm));
        const float p = __fdividef(d, fmaf(hx, hx, fmaf(hy, hy, fmaf(hz, hz, dd))));
        dr[0] = fmaf(p, hx, dr[0]); dr[1] = fmaf(p, hy, dr[1]); dr[2] = fmaf(p, hz, dr[2]);
    }
}

// NEXT-3, the paper's "comparison kernel": sum_x |dr(x)| and sum_x |r(x)| (Euclidean norm per
// voxel, reading A16) of iteration `iter`, per-thread fp32 norms accumulated in fp64.  Every block writes its two
// partial sums to its own slot; the last block to finish adds them in a fixed association (so l, and with it the iteration the
// level stops at, is the same from run to run), forms l = sum|dr| / sum|r| (+inf while the field is zero), files it in
// the 16-slot history and, from iteration 10 on, sets stop_iter = iter when l(iter-10) - l(iter) <= stop_eps.  Kernels
// of later iterations then fall through.
template <int MODE>
__global__ void __launch_bounds__(256)
k_force_norms(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ r, int nx, int ny,
              int nz, float eps_den, StopCtl* ctl, int iter, float stop_eps) {
    if (iter > *reinterpret_cast<volatile int*>(&ctl->stop_iter)) return;
    const size_t N = (size_t)nx * ny * nz;
    double a = 0.0, b = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const int x = (int)(i % nx), y = (int)((i / nx) % ny), z = (int)(i / ((size_t)nx * ny));
        float dr[3];
        force_increment<MODE>(m, s, nx, ny, nz, x, y, z, eps_den, dr);
        const float rx = __ldg(r + i), ry = __ldg(r + N + i), rz = __ldg(r + 2 * N + i);
        a += (double)sqrtf(fmaf(dr[0], dr[0], fmaf(dr[1], dr[1], dr[2] * dr[2])));
        b += (double)sqrtf(fmaf(rx, rx, fmaf(ry, ry, rz * rz)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    __shared__ double sh[2][8];
    __shared__ bool last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][warp] = a; sh[1][warp] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0.0, tb = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { ta += sh[0][w]; tb += sh[1][w]; }
        ctl->partial[2 * blockIdx.x] = ta; ctl->partial[2 * blockIdx.x + 1] = tb;
        __threadfence();
        last = atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last) {
        // the last block adds the partials in a FIXED association (thread i takes blocks i, i + 256, ... in rising order,
        // then a fixed tree over the 256 threads), so l -- and the iteration a level stops at -- is the same from run
        // to run, without one thread walking up to 2048 partials through L2 one after the other
        __threadfence();
        double sdr = 0.0, sr = 0.0;
        for (unsigned k = threadIdx.x; k < gridDim.x; k += blockDim.x) { sdr += ctl->partial[2 * k]; sr += ctl->partial[2 * k + 1]; }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sdr += __shfl_xor_sync(0xffffffffu, sdr, o);
            sr += __shfl_xor_sync(0xffffffffu, sr, o);
        }
        __syncthreads();                      // sh[] of the first reduction has been read by thread 0
        if (lane == 0) { sh[0][warp] = sdr; sh[1][warp] = sr; }
        __syncthreads();
        if (threadIdx.x == 0) {
            sdr = 0.0; sr = 0.0;
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { sdr += sh[0][w]; sr += sh[1][w]; }
            const double l = sr > 0.0 ? sdr / sr : (double)INFINITY;
            ctl->hist[iter & 15] = l;
            if (iter >= 10 && ctl->hist[(iter - 10) & 15] - l <= (double)stop_eps) ctl->stop_iter = iter;
            ctl->ticket = 0u;
            __threadfence();
        }
    }
}

static __global__ void k_stop_reset(StopCtl* ctl) {
    ctl->ticket = 0u; ctl->stop_iter = 0x7fffffff;
}
static __global__ void k_stop_record(StopCtl* ctl, int level, int n_iters) {
    ctl->runs[level] = ctl->stop_iter == 0x7fffffff ? n_iters : ctl->stop_iter + 1;
}

// Step (c) alone, in place (disc_force_update).
template <int MODE>
__global__ void __launch_bounds__(256)
k_force_update(const float* __restrict__ m, const float* __restrict__ s, float* __restrict__ r, int nx, int ny,
               int nz, float eps_den) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const size_t N = (size_t)nx * ny * nz;
    float u[3];
    updated_field<MODE>(m, s, r, nx, ny, nz, N, x, y, z, eps_den, u);
    const size_t i = ((size_t)z * ny + y) * nx + x;
    r[i] = u[0]; r[N + i] = u[1]; r[2 * N + i] = u[2];
}

// [force + update] + Gaussian x + Gaussian y.  Grid (x tiles, y segments, z); TXB threads <-> x.
template <int K, int FORCE, int TXB>
__global__ void __launch_bounds__(TXB)
k_force_gxy(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ rin,
            float* __restrict__ rout, int nx, int ny, int nz, int yseg, float eps_den, GaussTaps gw, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    constexpr int W = 2 * K + 1;
    __shared__ float row[2][3][TXB + 2 * K];
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TXB;
    const int x = x0 + tid;
    const int xc = min(x, nx - 1);
    const int z = blockIdx.z;
    const int y0 = blockIdx.y * yseg, y1 = min(y0 + yseg, ny);
    const size_t N = (size_t)nx * ny * nz;
    const size_t plane = (size_t)nx * ny;
    // halo duty: threads 0..K-1 take the left halo, K..2K-1 the right halo
    const bool halo = tid < 2 * K;
    const int hx = clampi(tid < K ? x0 - K + tid : x0 + TXB + (tid - K), 0, nx - 1);
    const int hslot = tid < K ? tid : TXB + tid;  // tid>=K: K + TXB + (tid-K)

    float ring[3][W];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int j = 0; j < W; ++j) ring[c][j] = 0.f;

    // rows yy = y0-K .. y1-1+K enter in order; row (yy) lives in ring slot (yy - (y0-K)) % W
    const int yend = y1 + K;
    int buf = 0;
    for (int yb = y0 - K; yb < yend; yb += W) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int yy = yb + j;
            if (yy >= yend) break;
            const int yr = clampi(yy, 0, ny - 1);  // replicate border in y
            float u[3];
            updated_field<FORCE>(m, s, rin, nx, ny, nz, N, xc, yr, z, eps_den, u);
#pragma unroll
            for (int c = 0; c < 3; ++c) row[buf][c][K + tid] = u[c];
            if (halo) {
                float h[3];
                updated_field<FORCE>(m, s, rin, nx, ny, nz, N, hx, yr, z, eps_den, h);
#pragma unroll
                for (int c = 0; c < 3; ++c) row[buf][c][hslot] = h[c];
            }
            __syncthreads();
            // x pass: replicate border in x is already in the row (positions were clamped)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float acc = 0.f;
#pragma unroll
                for (int k = 0; k < W; ++k) acc = fmaf(gw.w[k], row[buf][c][tid + k], acc);
                ring[c][j] = acc;
            }
            buf ^= 1;  // the other buffer was last read before the previous barrier
            // y pass: output row yo = yy - K uses rows yo-K..yo+K = slots (j+1+k) % W, k = 0..2K
            const int yo = yy - K;
            if (yo >= y0 && x < nx) {
                const size_t o = (size_t)z * plane + (size_t)yo * nx + x;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    float acc = 0.f;
#pragma unroll
                    for (int k = 0; k < W; ++k) acc = fmaf(gw.w[k], ring[c][(j + 1 + k) % W], acc);
                    rout[c * N + o] = acc;
                }
            }
        }
    }
}

// Step (b) alone (disc_warp).
static __global__ void __launch_bounds__(256)
k_warp(const float* __restrict__ moving, const float* __restrict__ r, float* __restrict__ out, int nx, int ny,
       int nz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const size_t N = (size_t)nx * ny * nz;
    const size_t i = ((size_t)z * ny + y) * nx + x;
    out[i] = trilinear_at_voxel(moving, nx, ny, nz, x, y, z, __ldg(r + i), __ldg(r + N + i), __ldg(r + 2 * N + i));
}

}  // namespace disc
