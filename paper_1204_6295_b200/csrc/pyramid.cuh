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

}  // namespace disc
