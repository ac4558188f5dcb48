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
#include <cuda.h>

#include "launch.h"
#include "pipeline.cuh"

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
          float* __restrict__ out1, int nx, int ny, int nz, int zchunk, float eps_var) {
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

// =========================================================================================================
// TMA version (the one the hot path uses when nx % 4 == 0 and the volume is 16-byte aligned).
//
// Same sums, different plumbing:
//   * the zero-padded raw tile of every incoming slice is fetched by ONE 3-D TMA tile load
//     (cp.async.bulk.tensor.3d, out-of-bounds elements zero-filled = the zero padding of the truncated
//     patch, reading A4), NSTG slices ahead, behind an mbarrier;
//   * the z window lives in SHARED memory (ring of the last 2R+1 xy box sums, fp64), which frees the registers
//     and lets the y pass own 4 (or 2) consecutive rows per thread and finish the voxel itself:
//       P1  x pass   task = (row, run of 8 outputs), lanes <-> rows, LDS.128 on an odd-chunk pitch
//       P2  y pass + z ring update + evaluation + store, task = (column, run of LY rows), lanes <-> x
//     two CTA barriers per slice, no third exchange buffer.
// =========================================================================================================
template <int R>
struct MomTmaCfg {
    static constexpr int W = 2 * R + 1;
    static constexpr int NT = (R <= 5) ? 128 : 256;
    static constexpr int LX = 8;
    static constexpr int LY = kMomTX * kMomTY / NT;                    // rows per P2 task: 4 or 2
    static constexpr int PX = kMomTX + 2 * R, PY = kMomTY + 2 * R;
    // The innermost TMA coordinate must be a multiple of 4 floats (16 bytes; an unaligned start raises an
    // illegal-instruction fault on sm_100a, measured), so the box starts at x0 - RA with RA = R rounded up to 4 and
    // column x0 - R sits at offset OFF in a raw row.
    static constexpr int RA = (R + 3) / 4 * 4, OFF = RA - R;
    static constexpr int PXB = (((OFF + PX + 3) / 4) | 1) * 4;         // TMA box width: multiple of 4 floats, odd number of 16-byte chunks
    static constexpr int XSP = kMomTX + 1;
    static constexpr int NSTG = (R <= 4) ? 3 : 2;                      // raw stages in flight
    static constexpr int P1_TASKS = PY * (kMomTX / LX);
    static constexpr size_t raw_bytes = sizeof(float) * PY * PXB;      // one stage (multiple of 16)
    static constexpr size_t ring_bytes = sizeof(double) * 2 * W * kMomTX * kMomTY;
    static constexpr size_t xs_bytes = sizeof(double) * 2 * PY * XSP;
    static constexpr size_t smem_bytes = 128 + NSTG * ((raw_bytes + 127) / 128 * 128) + ring_bytes + xs_bytes;
};

template <int R, int MODE>
__global__ void __launch_bounds__(MomTmaCfg<R>::NT)
k_moments_tma(const __grid_constant__ CUtensorMap tmap, const float* __restrict__ vol, const float* __restrict__ aux,
              float* __restrict__ out0, float* __restrict__ out1, int nx, int ny, int nz, int zchunk, float eps_var) {
    using C = MomTmaCfg<R>;
    constexpr int W = C::W, PY = C::PY, PXB = C::PXB, LX = C::LX, LY = C::LY, XSP = C::XSP, NT = C::NT, NSTG = C::NSTG;
    constexpr int RAWS = (int)((C::raw_bytes + 127) / 128 * 128 / sizeof(float));   // stage stride in floats
    static_assert(C::P1_TASKS <= NT, "x-pass tasks must fit the CTA");
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* raw = reinterpret_cast<float*>(smem_raw);                                   // [NSTG][PY][PXB]
    double* ring = reinterpret_cast<double*>(smem_raw + (size_t)NSTG * RAWS * sizeof(float));   // [W][2][TY][TX]
    double* xs = ring + (size_t)2 * W * kMomTX * kMomTY;                               // [2][PY][XSP]
    __shared__ uint64_t full[NSTG];
    __shared__ double inv_cnt_z[W + 1];

    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * kMomTX, y0 = blockIdx.y * kMomTY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, nz);
    const size_t plane = (size_t)nx * ny;
    const int zfirst = max(z0 - R, 0), zlast = min(z1 - 1 + R, nz - 1);   // slices that exist; the others are zero
    const int T = zlast - zfirst + 1;

    if (tid == 0) {
        for (int i = 0; i < NSTG; ++i) mbar_init(&full[i], 1);
        mbar_fence_init();
    }
    if (tid <= W) inv_cnt_z[tid] = tid > 0 ? 1.0 / (double)tid : 0.0;
    for (int i = tid; i < 2 * W * kMomTX * kMomTY; i += NT) ring[i] = 0.0;
    __syncthreads();

    auto issue = [&](int t) {   // thread 0: existing slice zfirst + t -> stage t % NSTG (its previous reader passed a CTA barrier)
        const int st = t % NSTG;
        mbar_expect_tx(&full[st], (uint32_t)C::raw_bytes);
        tma_load_3d(raw + (size_t)st * RAWS, &tmap, x0 - C::RA, y0 - R, zfirst + t, &full[st]);
    };
    if (tid == 0)
        for (int t = 0; t < min(NSTG, T); ++t) issue(t);

    // P2 ownership: column x = tid & 31, rows yb .. yb + LY - 1
    const int px = tid & 31, yb = (tid >> 5) * LY;
    const int gx = x0 + px;
    double Z1[LY], Z2[LY], inv_nxy[LY];
#pragma unroll
    for (int o = 0; o < LY; ++o) {
        Z1[o] = 0.0; Z2[o] = 0.0;
        const int gy = y0 + yb + o;
        const int cx = min(gx + R, nx - 1) - max(gx - R, 0) + 1;
        const int cy = min(gy + R, ny - 1) - max(gy - R, 0) + 1;
        inv_nxy[o] = (gx < nx && gy < ny) ? 1.0 / ((double)cx * (double)cy) : 0.0;
    }
    // P1 task: lanes <-> rows
    const int p1g = tid / PY, p1r = tid - p1g * PY;

    int slot = 0;  // ring slot of the incoming slice = (zz - (z0 - R)) % W
    for (int zz = z0 - R; zz < z1 + R; ++zz) {
        const bool valid = zz >= 0 && zz < nz;   // uniform
        const int zo = zz - R;
        const bool emit = zo >= z0;
        // prefetch what the evaluation needs from global memory before the passes
        float pre[LY];
        if (emit && MODE != kModeMoments) {
            const float* src = (MODE == kModeZscore) ? vol : aux;
#pragma unroll
            for (int o = 0; o < LY; ++o) {
                const int gy = y0 + yb + o;
                pre[o] = (gx < nx && gy < ny) ? __ldg(src + (size_t)zo * plane + (size_t)gy * nx + gx) : 0.f;
            }
        }
        if (valid) {
            const int t = zz - zfirst, st = t % NSTG;
            mbar_wait(&full[st], (t / NSTG) & 1);
            if (tid < C::P1_TASKS) {
                // the run starts at float OFF + g*LX of the row: read from the aligned chunk below it
                constexpr int O4 = C::OFF & ~3, O1 = C::OFF & 3;
                const float4* rp = reinterpret_cast<const float4*>(raw + (size_t)st * RAWS + p1r * PXB + p1g * LX + O4);
                constexpr int NV = (O1 + LX + 2 * R + 3) / 4;
                double dd[NV * 4];
#pragma unroll
                for (int i = 0; i < NV; ++i) {
                    const float4 f = rp[i];
                    dd[4 * i] = (double)f.x; dd[4 * i + 1] = (double)f.y; dd[4 * i + 2] = (double)f.z; dd[4 * i + 3] = (double)f.w;
                }
                const double* d = dd + O1;
                double s1 = 0.0, s2 = 0.0;
#pragma unroll
                for (int i = 0; i < W; ++i) { s1 += d[i]; s2 = fma(d[i], d[i], s2); }
                double* o1 = xs + p1r * XSP + p1g * LX;
                double* o2 = o1 + PY * XSP;
                o1[0] = s1; o2[0] = s2;
#pragma unroll
                for (int o = 1; o < LX; ++o) {
                    s1 += d[o + 2 * R] - d[o - 1];
                    s2 = fma(d[o + 2 * R], d[o + 2 * R], s2);
                    s2 = fma(-d[o - 1], d[o - 1], s2);
                    o1[o] = s1; o2[o] = s2;
                }
            }
            __syncthreads();   // xs complete; raw stage st is free again
            if (tid == 0 && t + NSTG < T) issue(t + NSTG);
        }
        // P2: y pass, z ring update, evaluation
        double b1[LY], b2[LY];
        if (valid) {
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const double* ip = xs + q * PY * XSP + yb * XSP + px;
                double v[LY + 2 * R];
#pragma unroll
                for (int i = 0; i < LY + 2 * R; ++i) v[i] = ip[i * XSP];
                double s = 0.0;
#pragma unroll
                for (int i = 0; i < W; ++i) s += v[i];
                if (q == 0) b1[0] = s; else b2[0] = s;
#pragma unroll
                for (int o = 1; o < LY; ++o) {
                    s += v[o + 2 * R] - v[o - 1];
                    if (q == 0) b1[o] = s; else b2[o] = s;
                }
            }
        } else {
#pragma unroll
            for (int o = 0; o < LY; ++o) { b1[o] = 0.0; b2[o] = 0.0; }
        }
        double inv_cz = 0.0;
        if (emit) inv_cz = inv_cnt_z[min(zo + R, nz - 1) - max(zo - R, 0) + 1];
        double* rg = ring + (size_t)slot * 2 * kMomTX * kMomTY + yb * kMomTX + px;
#pragma unroll
        for (int o = 0; o < LY; ++o) {
            double* r1 = rg + o * kMomTX;
            double* r2 = r1 + kMomTX * kMomTY;
            Z1[o] += b1[o] - *r1; *r1 = b1[o];
            Z2[o] += b2[o] - *r2; *r2 = b2[o];
            const int gy = y0 + yb + o;
            if (emit && gx < nx && gy < ny) {
                const double inv_n = inv_nxy[o] * inv_cz;
                const double mu = Z1[o] * inv_n;
                const double var = fma(-mu, mu, Z2[o] * inv_n);
                const float varf = fmaxf((float)var, 0.f);
                const size_t idx = (size_t)zo * plane + (size_t)gy * nx + gx;
                if (MODE == kModeMoments) {
                    out0[idx] = (float)mu;
                    out1[idx] = varf;
                } else if (MODE == kModeZscore) {
                    const float dv = (float)((double)pre[o] - mu);
                    out0[idx] = var > (double)eps_var ? dv * rsqrtf(varf) : 0.f;
                } else {
                    out0[idx] = fmaf(sqrtf(varf), pre[o], (float)mu);
                }
            }
        }
        slot = slot + 1 == W ? 0 : slot + 1;
        if (valid) __syncthreads();   // xs may be overwritten by the next slice's x pass
    }
}

}  // namespace disc
