// pyramid.cuh -- coarse-to-fine operators (reading A9) with a per-axis factor of 1 or 2
// (the paper's own preprocessing halves only the transverse plane).
#pragma once
#include "common.cuh"

namespace disc {

// Block mean over fx x fy x fz fine voxels: in [fz*mz][fy*my][fx*mx] -> out [mz][my][mx].  Threads <-> coarse x.
// VEC: fx == 2 and `in` 8-byte aligned -> the two x neighbours come as one 8-byte load.
template <bool VEC>
__global__ void __launch_bounds__(128)
k_downsample(const float* __restrict__ in, float* __restrict__ out, int mx, int my, int mz, int fx, int fy, int fz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= mx) return;
    const int nx = fx * mx, ny = fy * my;
    const size_t plane = (size_t)nx * ny;
    const float* p = in + ((size_t)(fz * z) * ny + fy * y) * nx + fx * x;
    float acc = 0.f;
    // fixed summation order: ((x0 + x1) + (next row ...)) per slice, slices added last
    for (int c = 0; c < fz; ++c) {
        float sl = 0.f;
        for (int b = 0; b < fy; ++b) {
            const float* q = p + (size_t)c * plane + (size_t)b * nx;
            float row;
            if (VEC) { const float2 v = __ldg(reinterpret_cast<const float2*>(q)); row = v.x + v.y; }
            else { row = __ldg(q); if (fx == 2) row += __ldg(q + 1); }
            sl = b == 0 ? row : sl + row;
        }
        acc = c == 0 ? sl : acc + sl;
    }
    out[((size_t)z * my + y) * mx + x] = acc * (1.f / (float)(fx * fy * fz));
}

// Field up-sampling: along an axis with factor 2 the cell-centre-aligned coordinate i/2 - 1/4 (clamped) and
// component value x2, along an axis with factor 1 the coordinate i and value x1 (component c is in voxel units of
// axis c).  gridDim.z = 3 * nz_fine.
__global__ void __launch_bounds__(128)
k_upsample_field(const float* __restrict__ coarse, float* __restrict__ fine, int cx, int cy, int cz, int fx, int fy,
                 int fz) {
    const int nx = fx * cx, ny = fy * cy, nz = fz * cz;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y;
    const int comp = blockIdx.z / nz, z = blockIdx.z - comp * nz;
    if (x >= nx) return;
    const float* src = coarse + (size_t)comp * cx * cy * cz;
    const float px = fx == 2 ? 0.5f * (float)x - 0.25f : (float)x;
    const float py = fy == 2 ? 0.5f * (float)y - 0.25f : (float)y;
    const float pz = fz == 2 ? 0.5f * (float)z - 0.25f : (float)z;
    const float v = trilinear_clamped(src, cx, cy, cz, px, py, pz);
    const float scale = (float)(comp == 0 ? fx : (comp == 1 ? fy : fz));
    fine[(size_t)comp * nx * ny * nz + ((size_t)z * ny + y) * nx + x] = scale * v;
}

// The same operator for the all-axes factor 2, eight fine voxels per thread: a thread owns coarse cell (i, j, k), loads
// its clamped 3x3x3 neighbourhood once (27 loads for 8 outputs instead of 64) and forms the 2x2x2 fine voxels with the
// lerps of trilinear_clamped in the same order (x, then y, then z), with the same (cell, weight) per axis and fine
// index -- so every output is bit-identical to k_upsample_field's.  gridDim.z = 3 * cz.
struct UpsAxis {
    int k[2];       // which of the two neighbour pairs (v[0],v[1]) / (v[1],v[2]) fine voxel 2i + a interpolates
    float t[2];
};
__device__ __forceinline__ UpsAxis ups_axis(int i, int n) {
    UpsAxis r;
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        float p = 0.5f * (float)(2 * i + a) - 0.25f;
        p = fminf(fmaxf(p, 0.f), (float)(n - 1));
        const int i0 = max(min((int)p, n - 2), 0);
        r.t[a] = p - (float)i0;
        r.k[a] = i0 - max(i - 1, 0) + (i == 0 ? 1 : 0);      // v[0] = c[max(i-1,0)], v[1] = c[i], v[2] = c[min(i+1,n-1)]
        if (n == 1) { r.k[a] = 1; r.t[a] = 0.f; }
    }
    return r;
}
__global__ void __launch_bounds__(128)
k_upsample_field_222(const float* __restrict__ coarse, float* __restrict__ fine, int cx, int cy, int cz) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y;
    const int comp = blockIdx.z / cz, k = blockIdx.z - comp * cz;
    if (i >= cx) return;
    const float* src = coarse + (size_t)comp * cx * cy * cz;
    const int xi[3] = {max(i - 1, 0), i, min(i + 1, cx - 1)};
    const int yj[3] = {max(j - 1, 0), j, min(j + 1, cy - 1)};
    const int zk[3] = {max(k - 1, 0), k, min(k + 1, cz - 1)};
    float v[3][3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const float* row = src + ((size_t)zk[c] * cy + yj[b]) * cx;
#pragma unroll
            for (int a = 0; a < 3; ++a) v[c][b][a] = __ldg(row + xi[a]);
        }
    const UpsAxis ax = ups_axis(i, cx), ay = ups_axis(j, cy), az = ups_axis(k, cz);
    // x lerps of all nine (y, z) lines for both fine x, exactly as trilinear_clamped: fmaf(t, hi, (1 - t) * lo)
    float lx[3][3][2];
#pragma unroll
    for (int a = 0; a < 2; ++a) {
        const float t = ax.t[a], u = 1.f - t;
        const bool hi = ax.k[a] != 0;
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b) lx[c][b][a] = fmaf(t, hi ? v[c][b][2] : v[c][b][1], u * (hi ? v[c][b][1] : v[c][b][0]));
    }
    const int nx = 2 * cx, ny = 2 * cy, nz = 2 * cz;
    float* dst = fine + (size_t)comp * nx * ny * nz;
#pragma unroll
    for (int c2 = 0; c2 < 2; ++c2) {
        const float tz = az.t[c2], uz = 1.f - tz;
        const bool hz = az.k[c2] != 0;
#pragma unroll
        for (int b2 = 0; b2 < 2; ++b2) {
            const float ty = ay.t[b2], uy = 1.f - ty;
            const bool hy = ay.k[b2] != 0;
            float o[2];
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                // y lerps of the two z planes involved, then the z lerp
                const float lo0 = hy ? lx[hz ? 1 : 0][1][a] : lx[hz ? 1 : 0][0][a], hi0 = hy ? lx[hz ? 1 : 0][2][a] : lx[hz ? 1 : 0][1][a];
                const float lo1 = hy ? lx[hz ? 2 : 1][1][a] : lx[hz ? 2 : 1][0][a], hi1 = hy ? lx[hz ? 2 : 1][2][a] : lx[hz ? 2 : 1][1][a];
                const float c0 = fmaf(ty, hi0, uy * lo0), c1 = fmaf(ty, hi1, uy * lo1);
                o[a] = 2.f * fmaf(tz, c1, uz * c0);
            }
            *reinterpret_cast<float2*>(dst + ((size_t)(2 * k + c2) * ny + (2 * j + b2)) * nx + 2 * i) = make_float2(o[0], o[1]);
        }
    }
}

}  // namespace disc
