// common.cuh -- small device helpers shared by the DISC kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace disc {

constexpr int kMaxGaussTaps = 2 * 12 + 1;

// Gaussian taps travel as a kernel parameter (constant bank): FFMA reads them as immediates-from-bank.
struct GaussTaps {
    float w[kMaxGaussTaps];
};

struct Dims {
    int nx, ny, nz;
};

// Stopping criterion: device-side state of one context.  Every kernel of iteration
// `iter` gets an IterCtl by value and returns at once when iter > *stop_iter, so an early stop needs no host
// synchronisation: the remaining launches of the level fall through.  stop_iter == nullptr: criterion off.
constexpr int kStopBlocks = 2048;   // most blocks k_force_norms is launched with
struct StopCtl {
    double partial[2 * kStopBlocks];   // per-block (sum|dr|, sum|r|) of the running iteration, added in block order
    double hist[16];           // l^(k) of the last 16 iterations, slot k & 15
    unsigned ticket;           // blocks of k_force_norms finished
    int stop_iter;             // last iteration of the level (INT_MAX while running)
    int runs[8];               // iterations run per level (DISC_MAX_LEVELS)
};
struct IterCtl {
    const int* stop_iter;
    int iter;
};
__device__ __forceinline__ bool iter_skipped(const IterCtl& c) {
    return c.stop_iter != nullptr && c.iter > *reinterpret_cast<const volatile int*>(c.stop_iter);
}

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return min(max(v, lo), hi); }

// one MUFU: relative error 2^-23, 0 -> 0
__device__ __forceinline__ float sqrt_approx(float v) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(v));
    return y;
}

// Trilinear sample of I at (px,py,pz), position clamped to the volume (reading A11):
// p = clamp(p, 0, n-1), i0 = min(floor(p), n-2), t = p - i0; an axis of length 1 has weight 0.
__device__ __forceinline__ float trilinear_clamped(const float* __restrict__ I, int nx, int ny, int nz, float px,
                                                   float py, float pz) {
    px = fminf(fmaxf(px, 0.f), (float)(nx - 1));
    py = fminf(fmaxf(py, 0.f), (float)(ny - 1));
    pz = fminf(fmaxf(pz, 0.f), (float)(nz - 1));
    const int x0 = max(min((int)px, nx - 2), 0), y0 = max(min((int)py, ny - 2), 0), z0 = max(min((int)pz, nz - 2), 0);
    const int dx = nx > 1 ? 1 : 0;
    const size_t dy = ny > 1 ? (size_t)nx : 0, dz = nz > 1 ? (size_t)nx * ny : 0;
    const float tx = px - (float)x0, ty = py - (float)y0, tz = pz - (float)z0;
    const float* p = I + ((size_t)z0 * ny + y0) * nx + x0;
    const float a000 = __ldg(p), a100 = __ldg(p + dx);
    const float a010 = __ldg(p + dy), a110 = __ldg(p + dy + dx);
    const float a001 = __ldg(p + dz), a101 = __ldg(p + dz + dx);
    const float a011 = __ldg(p + dz + dy), a111 = __ldg(p + dz + dy + dx);
    // (1-t)*a + t*b: exact at t = 0 and t = 1, so a zero field reproduces the input bit for bit
    const float ux = 1.f - tx, uy = 1.f - ty, uz = 1.f - tz;
    const float c00 = fmaf(tx, a100, ux * a000);
    const float c10 = fmaf(tx, a110, ux * a010);
    const float c01 = fmaf(tx, a101, ux * a001);
    const float c11 = fmaf(tx, a111, ux * a011);
    const float c0 = fmaf(ty, c10, uy * c00);
    const float c1 = fmaf(ty, c11, uy * c01);
    return fmaf(tz, c1, uz * c0);
}

// The warp's sample m(x) = I(x + r(x)) with the cell and weight formed from the voxel's integer coordinate and its
// displacement separately (floor(i + r) = i + floor(r) and r - floor(r) are exact in fp32, fl(i + r) is not) and the
// lerp written a + t (b - a), b the neighbour at +1 inside the volume and at -1 for a sample clamped to the far face:
// a zero field, an integer shift, a clamped sample and a flat region are all reproduced bit for bit (field_v3.cuh).
__device__ __forceinline__ float trilinear_at_voxel(const float* __restrict__ I, int nx, int ny, int nz, int x, int y,
                                                    int z, float rx, float ry, float rz) {
    int c0[3] = {0, 0, 0}, st[3] = {0, 0, 0};
    float t[3] = {0.f, 0.f, 0.f};
    const int n[3] = {nx, ny, nz}, i[3] = {x, y, z};
    const float r[3] = {rx, ry, rz};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (n[a] > 1) {
            const float fl = floorf(r[a]);
            const int j = i[a] + (int)fl;
            const bool lo = j < 0, hi = j > n[a] - 2;
            c0[a] = lo ? 0 : (hi ? n[a] - 1 : j);
            t[a] = (lo || hi) ? 0.f : r[a] - fl;
            st[a] = hi ? -1 : 1;
        }
    }
    const ptrdiff_t dx = st[0], dy = (ptrdiff_t)st[1] * nx, dz = (ptrdiff_t)st[2] * nx * ny;
    const float* p = I + ((size_t)c0[2] * ny + c0[1]) * nx + c0[0];
    const float a000 = __ldg(p), a100 = __ldg(p + dx);
    const float a010 = __ldg(p + dy), a110 = __ldg(p + dy + dx);
    const float a001 = __ldg(p + dz), a101 = __ldg(p + dz + dx);
    const float a011 = __ldg(p + dz + dy), a111 = __ldg(p + dz + dy + dx);
    const float c00 = fmaf(t[0], a100 - a000, a000);
    const float c10 = fmaf(t[0], a110 - a010, a010);
    const float c01 = fmaf(t[0], a101 - a001, a001);
    const float c11 = fmaf(t[0], a111 - a011, a011);
    const float e0 = fmaf(t[1], c10 - c00, c00);
    const float e1 = fmaf(t[1], c11 - c01, c01);
    return fmaf(t[2], e1 - e0, e0);
}

}  // namespace disc
