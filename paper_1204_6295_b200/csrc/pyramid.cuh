// pyramid.cuh -- coarse-to-fine operators (reading A9).
#pragma once
#include "common.cuh"

namespace disc {

// 2x2x2 block mean: in [2*mz][2*my][2*mx] -> out [mz][my][mx].  Threads <-> coarse x.
__global__ void __launch_bounds__(128)
k_downsample(const float* __restrict__ in, float* __restrict__ out, int mx, int my, int mz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= mx) return;
    const int nx = 2 * mx, ny = 2 * my;
    const float* p = in + ((size_t)(2 * z) * ny + 2 * y) * nx + 2 * x;
    const size_t plane = (size_t)nx * ny;
    const float2 a = __ldg(reinterpret_cast<const float2*>(p));
    const float2 b = __ldg(reinterpret_cast<const float2*>(p + nx));
    const float2 c = __ldg(reinterpret_cast<const float2*>(p + plane));
    const float2 d = __ldg(reinterpret_cast<const float2*>(p + plane + nx));
    out[((size_t)z * my + y) * mx + x] = 0.125f * (((a.x + a.y) + (b.x + b.y)) + ((c.x + c.y) + (d.x + d.y)));
}

// Field up-sampling x2: fine(i) = 2 * trilinear(coarse, clamp(i/2 - 1/4)); gridDim.z = 3*nz_fine.
__global__ void __launch_bounds__(128)
k_upsample_field(const float* __restrict__ coarse, float* __restrict__ fine, int cx, int cy, int cz) {
    const int nx = 2 * cx, ny = 2 * cy, nz = 2 * cz;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y;
    const int comp = blockIdx.z / nz, z = blockIdx.z - comp * nz;
    if (x >= nx) return;
    const float* src = coarse + (size_t)comp * cx * cy * cz;
    const float v = trilinear_clamped(src, cx, cy, cz, 0.5f * (float)x - 0.25f, 0.5f * (float)y - 0.25f,
                                      0.5f * (float)z - 0.25f);
    fine[(size_t)comp * nx * ny * nz + ((size_t)z * ny + y) * nx + x] = 2.f * v;
}

}  // namespace disc
