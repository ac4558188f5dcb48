// moments_blk.cuh -- patch moments + intensity correction, step (a), for SMALL volumes (the coarse pyramid levels).
//
// Same arithmetic as moments_v3.cuh (PAPER.md:95 Eq. 3, :117-119 Eqs. 5-6; readings A4, A5): zero-padded box sums of
// v and v^2 in fp64 as separable sliding windows, divided by the analytic in-volume count.  What differs is the
// decomposition.  The marching kernel gives one CTA a 32x32 column of the volume and walks it slice by slice; on a
// 64x64x32 level that is 4 columns, so even with one-slice chunks a CTA walks 2 rz + 1 slices one after the other and
// the launch lasts ~10 us for 0.13 M voxels (profiles/r02a).  Here a CTA owns a small BLOCK of 32 x BY x BZ outputs,
// takes the block + halo with ONE 3-D TMA load (zero out-of-bounds fill = the truncated patch) and runs the three
// passes one after the other out of shared memory, every pass over all slices of the block at once:
//   x pass  one task per raw row (lanes <-> rows): convert, slide (S1, S2) along x over the 32 outputs;
//   y pass  one task per (slice, x): slide along y IN PLACE (output row o overwrites input row o after it was read);
//   z pass  one task per (y, x): slide along z, evaluate mu, var and the mode's output, coalesced stores.
// The halo is recomputed per block ((BY + 2R)(BZ + 2 rz) / (BY BZ) rows per output row) -- irrelevant at these
// sizes: the launch is bound by its dependent chains, not by throughput, and the whole level lives in L2.
//
// Requirements (checked by the launcher): nx % 4 == 0, 16-byte aligned volume (tensor-map rules).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "launch.h"
#include "moments_v3.cuh"   // tree_sum, rsqrt_nr, kMaxWz
#include "pipeline.cuh"

namespace disc {

template <int R>
struct MomBlkCfg {
    static constexpr int W = 2 * R + 1, TX = 32, PX = TX + 2 * R;
    static constexpr int RA = (R + 3) / 4 * 4, OFF = RA - R;                 // the TMA box starts at x0 - RA (16-byte rule)
    static constexpr int PXB = (((OFF + PX + 3) / 4) | 1) * 4;               // raw row pitch: odd number of 16-byte chunks
    static constexpr int XSP = TX + 1;                                       // pair-row pitch in double2, odd
    static constexpr int NT = 256;
    static __host__ __device__ size_t raw_bytes(int py, int pz) { return sizeof(float) * (size_t)PXB * py * pz; }
    static __host__ __device__ size_t raw_stride(int py, int pz) { return (raw_bytes(py, pz) + 127) / 128 * 128; }
    static __host__ __device__ size_t smem_bytes(int py, int pz) { return raw_stride(py, pz) + sizeof(double2) * (size_t)XSP * py * pz; }
};

template <int R, int MODE>
__global__ void __launch_bounds__(MomBlkCfg<R>::NT, 1)
k_moments_blk(const __grid_constant__ CUtensorMap tmap, const float* __restrict__ pv, float* __restrict__ out0,
              float* __restrict__ out1, int nx, int ny, int nz, int rz, int by, int bz, float eps_var, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    using C = MomBlkCfg<R>;
    constexpr int W = C::W, TX = C::TX, PXB = C::PXB, XSP = C::XSP, NT = C::NT;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ uint64_t full;
    __shared__ double inv_cnt_z[kMaxWz + 1];

    const int tid = threadIdx.x, lane = tid & 31;
    const int py = by + 2 * R, wz = 2 * rz + 1, pz = bz + 2 * rz;
    float* raw = reinterpret_cast<float*>(smem_raw);                                        // [pz][py][PXB]
    double2* xs = reinterpret_cast<double2*>(smem_raw + C::raw_stride(py, pz));             // [pz][py][XSP]
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * by, z0 = blockIdx.z * bz;

    if (tid == 0) {
        mbar_init(&full, 1);
        mbar_fence_init();
        mbar_expect_tx(&full, (uint32_t)C::raw_bytes(py, pz));
        tma_load_3d(raw, &tmap, x0 - C::RA, y0 - R, z0 - rz, &full);
    }
    if (tid <= wz) inv_cnt_z[tid] = tid > 0 ? 1.0 / (double)tid : 0.0;
    __syncthreads();
    mbar_wait(&full, 0);

    // ------------------------------------------------------------------ x pass: raw rows -> (S1, S2) pairs
    {
        constexpr int O4 = C::OFF & ~3, O1 = C::OFF & 3;
        constexpr int NV = (O1 + C::PX + 3) / 4;
        const int rows = py * pz;
        for (int r = tid; r < rows; r += NT) {
            float rv[NV * 4];
            const float4* rp = reinterpret_cast<const float4*>(raw + r * PXB + O4);
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                const float4 f = rp[i];
                rv[4 * i] = f.x; rv[4 * i + 1] = f.y; rv[4 * i + 2] = f.z; rv[4 * i + 3] = f.w;
            }
            double win[W], t1[W], t2[W];
#pragma unroll
            for (int i = 0; i < W; ++i) { win[i] = (double)rv[O1 + i]; t1[i] = win[i]; t2[i] = win[i] * win[i]; }
            double s1 = tree_sum(t1), s2 = tree_sum(t2);
            double2* op = xs + r * XSP;
            op[0] = make_double2(s1, s2);
#pragma unroll
            for (int o = 1; o < TX; ++o) {
                // d_new^2 - d_old^2 = (d_new - d_old)(d_new + d_old): exact factors in fp64 for fp32 inputs
                const double dn = (double)rv[O1 + o + 2 * R], dl = win[(o - 1) % W];
                const double e = dn - dl, f = dn + dl;
                s1 += e;
                s2 = fma(e, f, s2);
                win[(o - 1) % W] = dn;
                op[o] = make_double2(s1, s2);
            }
        }
    }
    __syncthreads();

    // ------------------------------------------------------------------ y pass, in place: rows 0 .. by-1 of every slice
    for (int t = tid; t < pz * TX; t += NT) {
        const int zz = t >> 5;
        double2* col = xs + (zz * py) * XSP + lane;
        double t1[W], t2[W];
#pragma unroll
        for (int i = 0; i < W; ++i) { const double2 v = col[i * XSP]; t1[i] = v.x; t2[i] = v.y; }
        double s1 = tree_sum(t1), s2 = tree_sum(t2);
        for (int o = 0; o < by; ++o) {
            double2* p = col + o * XSP;
            const double2 lo = p[0];
            p[0] = make_double2(s1, s2);            // row o is no input of any later output
            if (o + 1 < by) {
                const double2 hi = p[W * XSP];
                s1 += hi.x - lo.x;
                s2 += hi.y - lo.y;
            }
        }
    }
    __syncthreads();

    // ------------------------------------------------------------------ z pass + evaluation
    const size_t plane = (size_t)nx * ny;
    for (int t = tid; t < by * TX; t += NT) {
        const int yy = t >> 5;
        const int gx = x0 + lane, gy = y0 + yy;
        if (gx >= nx || gy >= ny) continue;
        const int cx = min(gx + R, nx - 1) - max(gx - R, 0) + 1;
        const int cy = min(gy + R, ny - 1) - max(gy - R, 0) + 1;
        const double cxy = 1.0 / ((double)cx * (double)cy);
        const double2* col = xs + yy * XSP + lane;
        const int sstride = py * XSP;
        double Z1 = 0.0, Z2 = 0.0;
        for (int i = 0; i < wz; ++i) { const double2 v = col[i * sstride]; Z1 += v.x; Z2 += v.y; }
        const size_t idx0 = (size_t)z0 * plane + (size_t)gy * nx + gx;
        const int nout = min(bz, nz - z0);
        float pre = 0.f;
        if (MODE != kModeMoments) pre = __ldg(pv + idx0);
        for (int o = 0; o < nout; ++o) {
            const int zo = z0 + o;
            const size_t idx = idx0 + (size_t)o * plane;
            float nxt = 0.f;
            if (MODE != kModeMoments && o + 1 < nout) nxt = __ldg(pv + idx + plane);
            const int cz = min(zo + rz, nz - 1) - max(zo - rz, 0) + 1;
            // mu = S1/n, var = (S2 - S1 mu)/n: the cancellation in fp64, the division by n in fp32 (as moments_v3.cuh)
            const double inv_n = cxy * inv_cnt_z[cz];
            const double mu = Z1 * inv_n;
            const double nvar = fma(-Z1, mu, Z2);
            const float varf = fmaxf((float)nvar * (float)inv_n, 0.f);
            float r0;
            if (MODE == kModeMoments) {
                r0 = (float)mu;
                out1[idx] = varf;
            } else if (MODE == kModeZscore) {
                const float dv = (float)((double)pre - mu);
                r0 = nvar * inv_n > (double)eps_var ? dv * rsqrt_nr(varf) : 0.f;   // reading A5: decided on the fp64 variance
            } else {
                const float sd = varf * rsqrt_nr(fmaxf(varf, 1e-30f));
                r0 = fmaf(sd, pre, (float)mu);
            }
            out0[idx] = r0;
            pre = nxt;
            if (o + 1 < nout) {
                const double2 hi = col[(o + wz) * sstride], lo = col[o * sstride];
                Z1 += hi.x - lo.x;
                Z2 += hi.y - lo.y;
            }
        }
    }
}

}  // namespace disc
