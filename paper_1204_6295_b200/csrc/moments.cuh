// moments.cuh -- patch first/second moments as separable sliding-window box sums (step (a)).
//
// What it computes (PAPER.md:95 Eq. 3, :458 A.4; readings A4, A5): for every voxel, over the cube of
// radius R truncated to the volume, mu = S1/n and var = S2/n - mu^2 with S1 = sum v, S2 = sum v^2.
// Box sums are zero-padded and divided by the analytic in-volume count n = cx*cy*cz.
//
// How (differs from the paper's one-thread-loops-over-the-patch kernel): cost is
// independent of R.  A CTA owns a 32x16 (x,y) tile and marches z through a chunk.  Per incoming slice:
//   L   the zero-padded (32+2R)x(16+2R) raw tile goes to shared memory;
//   P1  x pass: one task per (row, run of 8 outputs) slides S1,S2 along x in fp64 -> xs;
//   P2  y pass: one task per (column, run of 4 outputs) slides along y -> bs (the slice's xy box sums);
//   P3  z pass: the thread that owns an output column keeps a ring of the last 2R+1 xy box sums in
//       REGISTERS (statically indexed through a loop unrolled 2R+1 times) and a running sum
//       Z += B_new - B_leaving; then evaluates mu, var and the mode's output for slice z-R.
// All sums are fp64: E(x^2) - mu^2 in fp32 is unusable (a constant 343-voxel patch at 1234.567 HU gives
// var = 9 HU^2); squares of fp32 values are exact in fp64 and DADD runs at half the fp32 rate on B200.
#pragma once
#include "common.cuh"

#include "launch.h"

namespace disc {

// tile constants kMomTX, kMomTY live in launch.h

template <int R>
struct MomCfg {
    static constexpr int NT = (R <= 6) ? 256 : 512;        // threads per CTA
    static constexpr int COLS = kMomTX * kMomTY / NT;      // output columns owned per thread
    static constexpr int W = 2 * R + 1;
    static constexpr int PX = kMomTX + 2 * R, PY = kMomTY + 2 * R;
    static constexpr int PXP = PX | 1;                     // odd pitch: lanes <-> rows is conflict free
    static constexpr int LX = 8, LY = 4;
    static constexpr int XSP = kMomTX + 1;                 // pitch of xs in doubles (odd)
    static constexpr int P1_TASKS = PY * (kMomTX / LX);
    static constexpr int P2_TASKS = kMomTX * (kMomTY / LY);
};

template <int R, int MODE>
__global__ void __launch_bounds__(MomCfg<R>::NT, (R <= 6) ? 2 : 1)
k_moments(const float* __restrict__ vol, const float* __restrict__ aux, float* __restrict__ out0,
          float* __restrict__ out1, int nx, int ny, int nz, int zchunk, float eps_var, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    using C = MomCfg<R>;
    constexpr int W = C::W, PX = C::PX, PY = C::PY, PXP = C::PXP, LX = C::LX, LY = C::LY, XSP = C::XSP;
    constexpr int NT = C::NT, COLS = C::COLS;
    static_assert(C::P1_TASKS <= NT && C::P2_TASKS <= NT, "task counts must fit the CTA");

    __shared__ float raw[PY * PXP];
    __shared__ double xs[2][PY * XSP];
    __shared__ double bs[2][kMomTY * kMomTX];
    __shared__ double inv_cnt_z[W + 1];

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * kMomTX, y0 = blockIdx.y * kMomTY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, nz);
    const size_t plane = (size_t)nx * ny;

    if (tid <= W) inv_cnt_z[tid] = tid > 0 ? 1.0 / (double)tid : 0.0;

    // the columns this thread owns, and 1/(cx*cy) for them
    const int tx = tid & 31;
    int ty[COLS];
    double inv_nxy[COLS];
    bool live[COLS];
#pragma unroll
    for (int k = 0; k < COLS; ++k) {
        ty[k] = (tid >> 5) + k * (NT / 32);
        const int gx = x0 + tx, gy = y0 + ty[k];
        live[k] = gx < nx && gy < ny;
        const int cx = min(gx + R, nx - 1) - max(gx - R, 0) + 1;
        const int cy = min(gy + R, ny - 1) - max(gy - R, 0) + 1;
        inv_nxy[k] = live[k] ? 1.0 / ((double)cx * (double)cy) : 0.0;
    }

    double ring1[COLS][W], ring2[COLS][W], Z1[COLS], Z2[COLS];
#pragma unroll
    for (int k = 0; k < COLS; ++k) {
        Z1[k] = 0.0; Z2[k] = 0.0;
#pragma unroll
        for (int j = 0; j < W; ++j) { ring1[k][j] = 0.0; ring2[k][j] = 0.0; }
    }

    const int zend = z1 + R;  // last incoming slice is z1-1+R
    for (int zb = z0 - R; zb < zend; zb += W) {
#pragma unroll
        for (int j = 0; j < W; ++j) {
            const int zz = zb + j;  // incoming slice; it replaces slice zz-W, which lives in ring slot j
            if (zz >= zend) break;
            const bool valid = zz >= 0 && zz < nz;  // uniform over the CTA
            if (valid) {
                // L: zero-padded raw tile
                const float* src = vol + (size_t)zz * plane;
                for (int e = tid; e < PY * PX; e += NT) {
                    const int r = e / PX, c = e - r * PX;
                    const int gx = x0 - R + c, gy = y0 - R + r;
                    float v = 0.f;
                    if (gx >= 0 && gx < nx && gy >= 0 && gy < ny) v = __ldg(src + (size_t)gy * nx + gx);
                    raw[r * PXP + c] = v;
                }
                __syncthreads();
                // P1: x pass, lanes <-> rows
                if (tid < C::P1_TASKS) {
                    const int g = tid / PY, r = tid - g * PY;
                    const float* rp = raw + r * PXP + g * LX;
                    double d[LX + 2 * R];
#pragma unroll
                    for (int i = 0; i < LX + 2 * R; ++i) d[i] = (double)rp[i];
                    double s1 = 0.0, s2 = 0.0;
#pragma unroll
                    for (int i = 0; i < W; ++i) { s1 += d[i]; s2 = fma(d[i], d[i], s2); }
                    double* o1 = &xs[0][r * XSP + g * LX];
                    double* o2 = &xs[1][r * XSP + g * LX];
                    o1[0] = s1; o2[0] = s2;
#pragma unroll
                    for (int o = 1; o < LX; ++o) {
                        s1 += d[o + 2 * R] - d[o - 1];
                        s2 = fma(d[o + 2 * R], d[o + 2 * R], s2);
                        s2 = fma(-d[o - 1], d[o - 1], s2);
                        o1[o] = s1; o2[o] = s2;
                    }
                }
                __syncthreads();
                // P2: y pass, lanes <-> x
                if (tid < C::P2_TASKS) {
                    const int x = tid & 31, h = tid >> 5;
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const double* ip = &xs[q][(h * LY) * XSP + x];
                        double v[LY + 2 * R];
#pragma unroll
                        for (int i = 0; i < LY + 2 * R; ++i) v[i] = ip[i * XSP];
                        double s = 0.0;
#pragma unroll
                        for (int i = 0; i < W; ++i) s += v[i];
                        double* op = &bs[q][(h * LY) * kMomTX + x];
                        op[0] = s;
#pragma unroll
                        for (int o = 1; o < LY; ++o) {
                            s += v[o + 2 * R] - v[o - 1];
                            op[o * kMomTX] = s;
                        }
                    }
                }
                __syncthreads();
            }
            // P3: z pass (ring in registers) + evaluation of output slice zo = zz - R
            const int zo = zz - R;
            const bool emit = zo >= z0 && zo < z1;
            double inv_cz = 0.0;
            if (emit) {
                const int cz = min(zo + R, nz - 1) - max(zo - R, 0) + 1;
                inv_cz = inv_cnt_z[cz];
            }
#pragma unroll
            for (int k = 0; k < COLS; ++k) {
                double b1 = 0.0, b2 = 0.0;
                if (valid) { b1 = bs[0][ty[k] * kMomTX + tx]; b2 = bs[1][ty[k] * kMomTX + tx]; }
                Z1[k] += b1 - ring1[k][j]; ring1[k][j] = b1;
                Z2[k] += b2 - ring2[k][j]; ring2[k][j] = b2;
                if (emit && live[k]) {
                    const double inv_n = inv_nxy[k] * inv_cz;
                    const double mu = Z1[k] * inv_n;
                    const double var = fmax(fma(-mu, mu, Z2[k] * inv_n), 0.0);
                    const size_t idx = (size_t)zo * plane + (size_t)(y0 + ty[k]) * nx + (x0 + tx);
                    if (MODE == kModeMoments) {
                        out0[idx] = (float)mu;
                        out1[idx] = (float)var;
                    } else if (MODE == kModeZscore) {
                        const float varf = (float)var;
                        const float dv = (float)((double)__ldg(vol + idx) - mu);
                        out0[idx] = var > (double)eps_var ? dv * rsqrtf(varf) : 0.f;
                    } else {
                        out0[idx] = fmaf(sqrtf((float)var), __ldg(aux + idx), (float)mu);
                    }
                }
            }
            // bs is rewritten only after the next slice's two barriers; raw/xs are safe as well
        }
    }
}

// The plain definition, one thread per voxel looping over its whole patch (as the paper's own kernel does,
// PAPER.md:410), for what the sliding-window kernels do not cover: a non-cubic patch
// on a volume the TMA kernel cannot take (nx % 4 != 0, unaligned base) or with a z radius beyond its tensor-memory
// ring.  fp64 sums over the truncated box (reading A4), cost proportional to the patch: a fallback, not a fast path.
template <int MODE>
__global__ void __launch_bounds__(128)
k_moments_direct(const float* __restrict__ vol, const float* __restrict__ aux, float* __restrict__ out0,
                 float* __restrict__ out1, int nx, int ny, int nz, int rx, int ry, int rz, float eps_var, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const int xa = max(x - rx, 0), xb = min(x + rx, nx - 1);
    const int ya = max(y - ry, 0), yb = min(y + ry, ny - 1);
    const int za = max(z - rz, 0), zb = min(z + rz, nz - 1);
    double s1 = 0.0, s2 = 0.0;
    for (int c = za; c <= zb; ++c)
        for (int b = ya; b <= yb; ++b) {
            const float* row = vol + ((size_t)c * ny + b) * nx;
            for (int a = xa; a <= xb; ++a) {
                const double v = (double)__ldg(row + a);
                s1 += v;
                s2 = fma(v, v, s2);
            }
        }
    const double inv_n = 1.0 / ((double)(xb - xa + 1) * (double)(yb - ya + 1) * (double)(zb - za + 1));
    const double mu = s1 * inv_n;
    const double var = fmax(fma(-mu, mu, s2 * inv_n), 0.0);
    const size_t idx = ((size_t)z * ny + y) * nx + x;
    if (MODE == kModeMoments) {
        out0[idx] = (float)mu;
        out1[idx] = (float)var;
    } else if (MODE == kModeZscore) {
        const float varf = (float)var;
        const float dv = (float)((double)__ldg(vol + idx) - mu);
        out0[idx] = var > (double)eps_var ? dv * rsqrtf(varf) : 0.f;
    } else {
        out0[idx] = fmaf(sqrtf((float)var), __ldg(aux + idx), (float)mu);
    }
}

}  // namespace disc
