// field_v3.cuh -- the two field kernels of the iteration (same arithmetic as the plain kernels of field.cuh, same
// results up to fp32 rounding order):
//   k_force_gxy_t4<K, FORCE>      [r += force(m, s')], Gaussian x pass, Gaussian y pass -> scratch field
//   k_gz_warp_d / _d2<K, WARP, LZ> Gaussian z pass of the scratch field -> r, [then m = ct(x + r(x))]
//
// History (profiles/r01a, r01b): the marching ring kernels of the first two generations were bound by their
// INSTRUCTION COUNT (280-290 thread instructions per voxel, a quarter of them pipeline bookkeeping and 64-bit
// address arithmetic) and by the exposed latency of their loads, not by HBM.  Hence
//   * z pass + warp: no ring, no shared memory, no barriers.  A thread owns one (or two adjacent) (x,y) columns
//     and LZ consecutive output slices; per component it issues all LZ + 2K input loads at once (coalesced
//     across the warp, latency overlapped LZ + 2K deep), forms the LZ outputs from statically indexed registers,
//     then runs the warp's trilinear gathers in batches (16-32 independent loads in flight).  The input is
//     re-read (LZ + 2K)/LZ times, but only from L2: neighbouring z blocks run at the same time on other SMs.
//   * force + x + y passes: a persistent tile kernel whose phase 1 works on groups of four x-adjacent points
//     with 16-byte loads (see below).
#pragma once
#include "common.cuh"
#include "field.cuh"
#include "pipeline.cuh"

namespace disc {

// The eight neighbours and three weights of one trilinear sample (reading A11), split in two halves so that the
// loads can be issued long before they are used.
struct TriSample {
    float a[8];
    float tx, ty, tz;
};

// Cell, weight and neighbour direction of one axis of the sample position p = clamp(i + r, 0, n - 1) (reading A11),
// WITHOUT forming i + r: floor(i + r) = i + floor(r) and the weight r - floor(r) are exact in fp32, whereas fl(i + r)
// loses up to ulp(i)/2 = 3e-5 voxel at i ~ 500.  The lerp is a + t (b - a) with a = I[i0], b = I[i0 + step]:
//   inside      i0 = i + floor(r), t = r - floor(r), step = +1
//   p <= 0      i0 = 0,     t = 0, step = +1
//   p >= n - 1  i0 = n - 1, t = 0, step = -1   (the neighbour is never out of the volume; n >= 2)
// so a zero field, an integer shift and a clamped sample reproduce a voxel bit for bit (t = 0), and a flat region
// stays flat bit for bit (b - a = 0): with (1 - t) a + t b a constant CT came out +-1 ulp noisy, which the patch
// variance of step (a) turns into a spurious sigma_m and the demons force of a flat region amplifies.
__device__ __forceinline__ void tri_axis(int i, float r, int n, int& i0, float& t, int& step) {
    const float fl = floorf(r);
    i0 = i + (int)fl;
    t = r - fl;
    const bool lo = i0 < 0, hi = i0 > n - 2;
    i0 = lo ? 0 : (hi ? n - 1 : i0);
    t = (lo || hi) ? 0.f : t;
    step = hi ? -1 : 1;
}

// (x, y, z): the voxel, (rx, ry, rz): its displacement.  FAST: every axis has at least two voxels and the voxel
// indices fit 32 bits (checked once per kernel, uniform).
template <bool FAST>
__device__ __forceinline__ void tri_issue(const float* __restrict__ I, int nx, int ny, int nz, int x, int y, int z,
                                          float rx, float ry, float rz, TriSample& s) {
    int x0 = 0, y0 = 0, z0 = 0, sx = 0, sy = 0, sz = 0;
    s.tx = 0.f; s.ty = 0.f; s.tz = 0.f;                // an axis of length 1 has weight 0 and no neighbour
    if (FAST || nx > 1) tri_axis(x, rx, nx, x0, s.tx, sx);
    if (FAST || ny > 1) tri_axis(y, ry, ny, y0, s.ty, sy);
    if (FAST || nz > 1) tri_axis(z, rz, nz, z0, s.tz, sz);
    if (FAST) {
        const int dy = sy * nx, dz = sz * nx * ny;
        const float* p00 = I + ((z0 * ny + y0) * nx + x0);
        const float* p10 = p00 + dy;
        const float* p01 = p00 + dz;
        const float* p11 = p01 + dy;
        s.a[0] = __ldg(p00); s.a[1] = __ldg(p00 + sx);
        s.a[2] = __ldg(p10); s.a[3] = __ldg(p10 + sx);
        s.a[4] = __ldg(p01); s.a[5] = __ldg(p01 + sx);
        s.a[6] = __ldg(p11); s.a[7] = __ldg(p11 + sx);
    } else {
        const ptrdiff_t dx = sx, dy = (ptrdiff_t)sy * nx, dz = (ptrdiff_t)sz * nx * ny;
        const float* p = I + ((size_t)z0 * ny + y0) * nx + x0;
        s.a[0] = __ldg(p); s.a[1] = __ldg(p + dx);
        s.a[2] = __ldg(p + dy); s.a[3] = __ldg(p + dy + dx);
        s.a[4] = __ldg(p + dz); s.a[5] = __ldg(p + dz + dx);
        s.a[6] = __ldg(p + dz + dy); s.a[7] = __ldg(p + dz + dy + dx);
    }
}

__device__ __forceinline__ float tri_finish(const TriSample& s) {
    // a + t (b - a): exact at t = 0 and wherever the two neighbours are equal
    const float c00 = fmaf(s.tx, s.a[1] - s.a[0], s.a[0]);
    const float c10 = fmaf(s.tx, s.a[3] - s.a[2], s.a[2]);
    const float c01 = fmaf(s.tx, s.a[5] - s.a[4], s.a[4]);
    const float c11 = fmaf(s.tx, s.a[7] - s.a[6], s.a[6]);
    const float c0 = fmaf(s.ty, c10 - c00, c00);
    const float c1 = fmaf(s.ty, c11 - c01, c01);
    return fmaf(s.tz, c1 - c0, c0);
}

// Step (b) alone (disc_warp) with two x-adjacent voxels per thread: 8-byte field loads and stores, both samples'
// sixteen gathered loads issued before either is interpolated.  Needs nx even and 8-byte aligned r, out.
static __global__ void __launch_bounds__(128)
k_warp2(const float* __restrict__ moving, const float* __restrict__ r, float* __restrict__ out, int nx, int ny, int nz) {
    const int x = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int y = blockIdx.y, z = blockIdx.z;
    if (x >= nx) return;
    const size_t N = (size_t)nx * ny * nz;
    const size_t i = ((size_t)z * ny + y) * nx + x;
    const float2 rx = __ldg(reinterpret_cast<const float2*>(r + i));
    const float2 ry = __ldg(reinterpret_cast<const float2*>(r + N + i));
    const float2 rz = __ldg(reinterpret_cast<const float2*>(r + 2 * N + i));
    const bool fast = nx > 1 && ny > 1 && nz > 1 && N < (size_t)0x7fffffff;   // 32-bit voxel indices
    TriSample g0, g1;
    if (fast) {
        tri_issue<true>(moving, nx, ny, nz, x, y, z, rx.x, ry.x, rz.x, g0);
        tri_issue<true>(moving, nx, ny, nz, x + 1, y, z, rx.y, ry.y, rz.y, g1);
    } else {
        tri_issue<false>(moving, nx, ny, nz, x, y, z, rx.x, ry.x, rz.x, g0);
        tri_issue<false>(moving, nx, ny, nz, x + 1, y, z, rx.y, ry.y, rz.y, g1);
    }
    *reinterpret_cast<float2*>(out + i) = make_float2(tri_finish(g0), tri_finish(g1));
}

constexpr int kGzdThreads = 128;

template <int K, bool WARP, int LZ>
__global__ void __launch_bounds__(kGzdThreads)
k_gz_warp_d(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
            float* __restrict__ mout, int nx, int ny, int nz, GaussTaps gw, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    constexpr int W = 2 * K + 1, NV = LZ + 2 * K;
    const unsigned plane = (unsigned)nx * (unsigned)ny;
    const unsigned col = blockIdx.x * kGzdThreads + threadIdx.x;
    if (col >= plane) return;
    const size_t N = (size_t)plane * nz;
    const int z0 = blockIdx.y * LZ;
    const bool interior = z0 - K >= 0 && z0 + LZ + K <= nz;   // uniform over the CTA

    float res[3][LZ];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* src = rin + c * N + col;
        float v[NV];
        if (interior) {
            const float* p = src + (size_t)(z0 - K) * plane;
#pragma unroll
            for (int i = 0; i < NV; ++i) v[i] = __ldg(p + (size_t)i * plane);
        } else {
#pragma unroll
            for (int i = 0; i < NV; ++i) v[i] = __ldg(src + (size_t)clampi(z0 - K + i, 0, nz - 1) * plane);   // replicate border
        }
#pragma unroll
        for (int j = 0; j < LZ; ++j) {
            float acc = 0.f;
#pragma unroll
            for (int k = 0; k < W; ++k) acc = fmaf(gw.w[k], v[j + k], acc);
            res[c][j] = acc;
        }
        float* dst = rout + c * N + (size_t)z0 * plane + col;
        if (interior) {
#pragma unroll
            for (int j = 0; j < LZ; ++j) dst[(size_t)j * plane] = res[c][j];
        } else {
#pragma unroll
            for (int j = 0; j < LZ; ++j)
                if (z0 + j < nz) dst[(size_t)j * plane] = res[c][j];
        }
    }
    if (WARP) {
        const int y = (int)(col / (unsigned)nx), x = (int)(col - (unsigned)y * (unsigned)nx);
        const bool fast = nx > 1 && ny > 1 && nz > 1 && N < (size_t)0x7fffffff;   // 32-bit voxel indices
        float* mp = mout + (size_t)z0 * plane + col;
        constexpr int B = 4;
        static_assert(LZ % B == 0, "gather batches");
#pragma unroll
        for (int j0 = 0; j0 < LZ; j0 += B) {
            TriSample g[B];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int j = j0 + b;
                if (fast) tri_issue<true>(moving, nx, ny, nz, x, y, z0 + j, res[0][j], res[1][j], res[2][j], g[b]);
                else tri_issue<false>(moving, nx, ny, nz, x, y, z0 + j, res[0][j], res[1][j], res[2][j], g[b]);
            }
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int j = j0 + b;
                const float mv = tri_finish(g[b]);
                if (interior || z0 + j < nz) mp[(size_t)j * plane] = mv;
            }
        }
    }
}

// Two adjacent columns per thread (nx even, 8-byte aligned fields): 8-byte loads and stores, packed FFMA2 taps --
// half the load / store / FMA instructions and half the address arithmetic per voxel.
template <int K, bool WARP, int LZ>
__global__ void __launch_bounds__(kGzdThreads, 8)   // 64 registers: eight CTAs per SM keep the gathers' latency covered
k_gz_warp_d2(const float* __restrict__ rin, float* __restrict__ rout, const float* __restrict__ moving,
             float* __restrict__ mout, int nx, int ny, int nz, GaussTaps gw, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    constexpr int W = 2 * K + 1, NV = LZ + 2 * K;
    const unsigned plane = (unsigned)nx * (unsigned)ny;
    const unsigned col = 2u * (blockIdx.x * kGzdThreads + threadIdx.x);
    if (col >= plane) return;
    const size_t N = (size_t)plane * nz;
    const int z0 = blockIdx.y * LZ;
    const bool interior = z0 - K >= 0 && z0 + LZ + K <= nz;   // uniform over the CTA

    float2 res[3][LZ];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* src = rin + c * N + col;
        float2 v[NV];
        if (interior) {
            const float* p = src + (size_t)(z0 - K) * plane;
#pragma unroll
            for (int i = 0; i < NV; ++i) { v[i] = __ldg(reinterpret_cast<const float2*>(p)); p += plane; }
        } else {
#pragma unroll
            for (int i = 0; i < NV; ++i)
                v[i] = __ldg(reinterpret_cast<const float2*>(src + (size_t)clampi(z0 - K + i, 0, nz - 1) * plane));   // replicate border
        }
#pragma unroll
        for (int j = 0; j < LZ; ++j) {
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int k = 0; k < W; ++k) acc = ffma2(make_float2(gw.w[k], gw.w[k]), v[j + k], acc);
            res[c][j] = acc;
        }
        float* dst = rout + c * N + (size_t)z0 * plane + col;
#pragma unroll
        for (int j = 0; j < LZ; ++j) {
            if (interior || z0 + j < nz) *reinterpret_cast<float2*>(dst) = res[c][j];
            dst += plane;
        }
    }
    if (WARP) {
        const int y = (int)(col / (unsigned)nx), x = (int)(col - (unsigned)y * (unsigned)nx);   // both columns share y (nx even)
        const bool fast = nx > 1 && ny > 1 && nz > 1 && N < (size_t)0x7fffffff;   // 32-bit voxel indices
        float* mp = mout + (size_t)z0 * plane + col;
        constexpr int B = 1;   // gather batches of one slice (two voxels, 16 loads in flight) measured best
        static_assert(LZ % B == 0, "gather batches");
#pragma unroll
        for (int j0 = 0; j0 < LZ; j0 += B) {
            TriSample g[B][2];
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int j = j0 + b;
                if (fast) {
                    tri_issue<true>(moving, nx, ny, nz, x, y, z0 + j, res[0][j].x, res[1][j].x, res[2][j].x, g[b][0]);
                    tri_issue<true>(moving, nx, ny, nz, x + 1, y, z0 + j, res[0][j].y, res[1][j].y, res[2][j].y, g[b][1]);
                } else {
                    tri_issue<false>(moving, nx, ny, nz, x, y, z0 + j, res[0][j].x, res[1][j].x, res[2][j].x, g[b][0]);
                    tri_issue<false>(moving, nx, ny, nz, x + 1, y, z0 + j, res[0][j].y, res[1][j].y, res[2][j].y, g[b][1]);
                }
            }
#pragma unroll
            for (int b = 0; b < B; ++b) {
                const int j = j0 + b;
                const float2 mv = make_float2(tri_finish(g[b][0]), tri_finish(g[b][1]));
                if (interior || z0 + j < nz) *reinterpret_cast<float2*>(mp) = mv;
                mp += plane;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// [force + update] + Gaussian x + Gaussian y, tile kernel with a VECTORISED phase 1.
//
// Same three phases as k_force_gxy_tile (field_v2.cuh), but phase 1 -- which held 70 % of that kernel's
// instructions (profiles/r01b: 128 per point, 11 scalar loads each with its own 64-bit address) -- now works on
// groups of four x-adjacent points: nine 16-byte loads and two scalar ones per group, one address computation per
// load, one 16-byte store per component.  For that the tile's x halo is rounded out to a multiple of four
// (KA = K rounded up), so every group is either wholly inside the volume or wholly outside it; outside groups are
// the replicate border: the clamped point's value, broadcast.
// Requirements (launcher): nx % 4 == 0, 16-byte aligned m, s, rin, rout.
// ---------------------------------------------------------------------------------------------------------
#ifndef DISC_FG_LX
#define DISC_FG_LX 8
#endif
#ifndef DISC_FG_NT
#define DISC_FG_NT 256
#endif
#ifndef DISC_FG_OCC
#define DISC_FG_OCC 2
#endif
template <int K, int TY_>
struct FgT4Cfg {
    static constexpr int TX = 64, TY = TY_, NT = DISC_FG_NT, OCC = DISC_FG_OCC, LX = DISC_FG_LX, LY = 8;
    static constexpr int W = 2 * K + 1;
    static constexpr int KA = (K + 3) / 4 * 4, OFF = KA - K;
    static constexpr int PXA = TX + 2 * KA, PY = TY + 2 * K, NG = PXA / 4;
    static constexpr int UP = ((PXA / 4) | 1) * 4;               // U row pitch: odd number of 16-byte chunks
    static constexpr int XP = TX + 4;                            // X row pitch: 17 chunks (odd)
    static constexpr int NV = (OFF + LX + 2 * K + 3) / 4;        // 16-byte chunks of one x-pass run
    static constexpr int P2_TASKS = 3 * PY * (TX / LX);
    static constexpr int P3_TASKS = 3 * (TX / 4) * (TY / LY);
    static constexpr size_t smem_bytes = sizeof(float) * 3 * PY * (UP + XP);
    static_assert((TX - LX) + 4 * NV <= UP, "x-pass run must stay inside the U row");
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// updated field of one group of four x-adjacent points (gx % 4 == 0), loads first, arithmetic after.
// Voxel indices are 32-bit here (the launcher checks 3 N < 2^32): one IMAD.WIDE per load instead of a 64-bit add.
// The force is evaluated with the raw central differences D = 2 g and t = 2 d:
//   d g_c / (|g|^2 + d^2 + eps) = (t / (|D|^2 + t^2 + 4 eps)) * D_c
// -- the same real number (every scaling is by a power of two, so the fused chains round identically) without the
// twelve multiplications by 1/2; the quotient is t * rcp.approx(den), den >= 4 eps > 0.
template <int FORCE>
struct FgGroup {
    float4 u[3], sc, mm, syp, sym, szp, szm;
    float sl, sr;
    float4 myp, mym, mzp, mzm;   // double force only: the moving image's neighbours
    float ml, mr;
    __device__ __forceinline__ void load(const float* __restrict__ m, const float* __restrict__ s,
                                         const float* __restrict__ rin, int nx, int ny, int nz, unsigned plane, unsigned N,
                                         int gx, int gy, int z) {
        const unsigned i = (unsigned)z * plane + (unsigned)gy * (unsigned)nx + (unsigned)gx;
#pragma unroll
        for (int c = 0; c < 3; ++c) u[c] = ldg4(rin + (i + (unsigned)c * N));
        if (FORCE) {
            const unsigned il = i - (gx > 0 ? 1u : 0u), ir = i + 3u + (gx + 4 < nx ? 1u : 0u);
            const unsigned iyp = i + (gy < ny - 1 ? (unsigned)nx : 0u), iym = i - (gy > 0 ? (unsigned)nx : 0u);
            const unsigned izp = i + (z < nz - 1 ? plane : 0u), izm = i - (z > 0 ? plane : 0u);
            sc = ldg4(s + i); mm = ldg4(m + i);
            sl = __ldg(s + il); sr = __ldg(s + ir);
            syp = ldg4(s + iyp); sym = ldg4(s + iym);
            szp = ldg4(s + izp); szm = ldg4(s + izm);
            if (FORCE == kForceDouble) {
                ml = __ldg(m + il); mr = __ldg(m + ir);
                myp = ldg4(m + iyp); mym = ldg4(m + iym);
                mzp = ldg4(m + izp); mzm = ldg4(m + izm);
            }
        }
    }
    __device__ __forceinline__ void finish(float eps_den) {
        if (FORCE) {
            const float ce[6] = {sl, sc.x, sc.y, sc.z, sc.w, sr};
            const float me[4] = {mm.x, mm.y, mm.z, mm.w};
            const float yp[4] = {syp.x, syp.y, syp.z, syp.w}, ym[4] = {sym.x, sym.y, sym.z, sym.w};
            const float zp[4] = {szp.x, szp.y, szp.z, szp.w}, zm[4] = {szm.x, szm.y, szm.z, szm.w};
            float ux[4] = {u[0].x, u[0].y, u[0].z, u[0].w}, uy[4] = {u[1].x, u[1].y, u[1].z, u[1].w};
            float uz[4] = {u[2].x, u[2].y, u[2].z, u[2].w};
            const float he[6] = {ml, mm.x, mm.y, mm.z, mm.w, mr};
            const float hyp[4] = {myp.x, myp.y, myp.z, myp.w}, hym[4] = {mym.x, mym.y, mym.z, mym.w};
            const float hzp[4] = {mzp.x, mzp.y, mzp.z, mzp.w}, hzm[4] = {mzm.x, mzm.y, mzm.z, mzm.w};
            const float eps4 = 4.f * eps_den;
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const float Dx = ce[e + 2] - ce[e], Dy = yp[e] - ym[e], Dz = zp[e] - zm[e];
                const float d = ce[e + 1] - me[e];
                const float t = d + d;
                const float tt = fmaf(t, t, eps4);
                const float q = t * rcp_approx(fmaf(Dx, Dx, fmaf(Dy, Dy, fmaf(Dz, Dz, tt))));
                ux[e] = fmaf(q, Dx, ux[e]);
                uy[e] = fmaf(q, Dy, uy[e]);
                uz[e] = fmaf(q, Dz, uz[e]);
                if (FORCE == kForceDouble) {
                    const float Hx = he[e + 2] - he[e], Hy = hyp[e] - hym[e], Hz = hzp[e] - hzm[e];
                    const float p = t * rcp_approx(fmaf(Hx, Hx, fmaf(Hy, Hy, fmaf(Hz, Hz, tt))));
                    ux[e] = fmaf(p, Hx, ux[e]);
                    uy[e] = fmaf(p, Hy, uy[e]);
                    uz[e] = fmaf(p, Hz, uz[e]);
                }
            }
            u[0] = make_float4(ux[0], ux[1], ux[2], ux[3]);
            u[1] = make_float4(uy[0], uy[1], uy[2], uy[3]);
            u[2] = make_float4(uz[0], uz[1], uz[2], uz[3]);
        }
    }
};

// The tile is 64 x TY_: 32 rows at the fine levels; 8 rows where a level has fewer 64 x 32 tiles than the device has
// CTA slots (64 x 64 x 32: 64 tiles) -- four times the CTAs, each with a quarter of the serial work per phase.
// PERSISTENT: the grid is two CTAs per SM; a CTA walks tiles t = blockIdx.x, += gridDim.x (x fastest, so the CTAs
// running at the same time work on neighbouring tiles and share their halos in L2).  Phase 3 of tile t-1 and
// phase 1 of tile t share one barrier interval -- the y pass (pure FMA work out of shared memory) runs on some
// warps while others wait for phase 1's global loads.
template <int K, int FORCE, int TY_>
__global__ void __launch_bounds__(FgT4Cfg<K, TY_>::NT, FgT4Cfg<K, TY_>::OCC)
k_force_gxy_t4(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ rin,
               float* __restrict__ rout, int nx, int ny, int nz, float eps_den, GaussTaps gw, IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    using C = FgT4Cfg<K, TY_>;
    constexpr int W = C::W, TX = C::TX, TY = C::TY, NT = C::NT, LX = C::LX, LY = C::LY, PY = C::PY, NG = C::NG;
    constexpr int UP = C::UP, XP = C::XP, KA = C::KA, OFF = C::OFF, NV = C::NV;
    extern __shared__ __align__(16) float smem_f[];
    float* U = smem_f;                       // [3][PY][UP]
    float* X = smem_f + 3 * PY * UP;         // [3][PY][XP]

    const int tid = threadIdx.x;
    const size_t plane = (size_t)nx * ny;
    const size_t N = plane * nz;
    const int ntx = (nx + TX - 1) / TX, nty = (ny + TY - 1) / TY;
    const int n_tiles = ntx * nty * nz;

    int px0 = 0, py0 = 0, pz = 0;   // the previous tile (whose y pass is still due)
    bool have_prev = false;
    for (int t = blockIdx.x;; t += gridDim.x) {
        const bool have = t < n_tiles;
        const int z = t / (ntx * nty), txy = t - z * (ntx * nty);
        const int y0 = (txy / ntx) * TY, x0 = (txy - (txy / ntx) * ntx) * TX;

        // ---- phase 1 of tile t: updated field at the tile + halo, four x-adjacent points at a time.  Two groups per
        // thread and round, both groups' loads issued before either is evaluated: phase 1 is bound by the latency of
        // its loads (profiles/r02a: 55 % of the kernel's stall samples on 36 % of its instructions), and twice the
        // loads in flight halves the number of exposed round trips per tile.
        if (have) {
            auto issue = [&](FgGroup<FORCE>& G, int p, int& r, int& g, int& gx) {
                r = p / NG; g = p - r * NG;
                const int gy = clampi(y0 - K + r, 0, ny - 1);
                gx = x0 - KA + 4 * g;
                G.load(m, s, rin, nx, ny, nz, (unsigned)plane, (unsigned)N, clampi(gx, 0, nx - 4), gy, z);
            };
            auto retire = [&](FgGroup<FORCE>& G, int r, int g, int gx) {
                G.finish(eps_den);
                // a group wholly outside the volume is the replicate border: the edge group's outermost value
                if (gx < 0 || gx >= nx) {   // only in the tiles at the volume's x border
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const float e = gx < 0 ? G.u[c].x : G.u[c].w;
                        G.u[c] = make_float4(e, e, e, e);
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) *reinterpret_cast<float4*>(U + (c * PY + r) * UP + 4 * g) = G.u[c];
            };
            for (int p = tid; p < PY * NG; p += 2 * NT) {
                FgGroup<FORCE> G0, G1;
                int r0, g0, gx0, r1 = 0, g1 = 0, gx1 = 0;
                const bool two = p + NT < PY * NG;
                issue(G0, p, r0, g0, gx0);
                if (two) issue(G1, p + NT, r1, g1, gx1);
                retire(G0, r0, g0, gx0);
                if (two) retire(G1, r1, g1, gx1);
            }
        }
        // ---- phase 3 of tile t-1: y pass, lanes <-> column groups
        if (have_prev) {
            for (int tk = tid; tk < C::P3_TASKS; tk += NT) {
                const int cg = tk % (TX / 4), q = tk / (TX / 4), h = q % (TY / LY), cc = q / (TY / LY);
                const float4* xp = reinterpret_cast<const float4*>(X + (cc * PY + h * LY) * XP + cg * 4);
                float2 a0[LY], a1[LY];
#pragma unroll
                for (int j = 0; j < LY; ++j) { a0[j] = make_float2(0.f, 0.f); a1[j] = make_float2(0.f, 0.f); }
#pragma unroll
                for (int i = 0; i < LY + 2 * K; ++i) {
                    const float4 f = xp[i * (XP / 4)];
                    const float2 lo = make_float2(f.x, f.y), hi = make_float2(f.z, f.w);
#pragma unroll
                    for (int j = 0; j < LY; ++j) {
                        const int k = i - j;          // input row i contributes to output row j with tap k
                        if (k >= 0 && k < W) {
                            const float2 w2 = make_float2(gw.w[k], gw.w[k]);
                            a0[j] = ffma2(w2, lo, a0[j]);
                            a1[j] = ffma2(w2, hi, a1[j]);
                        }
                    }
                }
                const int gx = px0 + cg * 4;
                if (gx < nx) {
                    float* op = rout + cc * N + ((size_t)pz * ny + (py0 + h * LY)) * nx + gx;
                    if (py0 + h * LY + LY <= ny) {   // whole run inside the volume: no per-row test
#pragma unroll
                        for (int j = 0; j < LY; ++j) {
                            *reinterpret_cast<float4*>(op) = make_float4(a0[j].x, a0[j].y, a1[j].x, a1[j].y);
                            op += nx;
                        }
                    } else {
#pragma unroll
                        for (int j = 0; j < LY; ++j)
                            if (py0 + h * LY + j < ny)
                                *reinterpret_cast<float4*>(op + (size_t)j * nx) = make_float4(a0[j].x, a0[j].y, a1[j].x, a1[j].y);
                    }
                }
            }
        }
        if (!have) break;
        __syncthreads();

        // ---- phase 2 of tile t: x pass, lanes <-> rows; output x0 + g*LX + j reads U columns OFF + g*LX + j + k
        for (int tk = tid; tk < C::P2_TASKS; tk += NT) {
            const int r = tk % PY, q = tk / PY, g = q % (TX / LX), cc = q / (TX / LX);
            const float4* up = reinterpret_cast<const float4*>(U + (cc * PY + r) * UP + g * LX);
            float v[4 * NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) {
                const float4 f = up[i];
                v[4 * i] = f.x; v[4 * i + 1] = f.y; v[4 * i + 2] = f.z; v[4 * i + 3] = f.w;
            }
            float o[LX];
#pragma unroll
            for (int j = 0; j < LX; ++j) {
                float acc = 0.f;
#pragma unroll
                for (int k = 0; k < W; ++k) acc = fmaf(gw.w[k], v[OFF + j + k], acc);
                o[j] = acc;
            }
            float4* xp = reinterpret_cast<float4*>(X + (cc * PY + r) * XP + g * LX);
#pragma unroll
            for (int q4 = 0; q4 < LX / 4; ++q4) xp[q4] = make_float4(o[4 * q4], o[4 * q4 + 1], o[4 * q4 + 2], o[4 * q4 + 3]);
        }
        __syncthreads();
        px0 = x0; py0 = y0; pz = z; have_prev = true;
    }
}

}  // namespace disc
