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
// Shared-memory layouts (tile 64 x TY, halo K in y, KA = K rounded up to 4 in x; PY = TY + 2K rows, always even):
//   U  updated field at the tile + halo, ROW-PAIR INTERLEAVED: U[c][rp][x][2] holds rows 2rp and 2rp+1 of column x
//      side by side, so that the x pass finds (row 2rp, row 2rp+1) of every column in one aligned 64-bit register
//      pair and runs as packed FFMA2 over two rows at once -- whatever the tap, the pair is aligned (pairs ALONG x
//      would be misaligned for every odd tap);
//   X  x-smoothed field, plain rows grouped in pairs: row R at (R >> 1) * XPP + (R & 1) * XP, XPP an odd number of
//      16-byte chunks (lanes <-> row pairs store conflict free), read by the y pass with lanes <-> column groups.
template <int K, int TY_>
struct FgT4Cfg {
    // 224 threads, two CTAs per SM: at K = 6 the 440 / 528 / 192 tasks of the three phases fill whole rounds of 224 better
    // than of 256 (measured 87.7 against 89.1 us); 8 outputs per x-pass task and row, 8 rows per y-pass task
    static constexpr int TX = 64, TY = TY_, NT = 224, OCC = 2, LX = 8, LY = 8;
    static constexpr int W = 2 * K + 1;
    static constexpr int KA = (K + 3) / 4 * 4, OFF = KA - K;
    static constexpr int PXA = TX + 2 * KA, PY = TY + 2 * K, NG = PXA / 4, NRP = PY / 2;
    static constexpr int UPP = ((2 * PXA / 4) | 1) * 4;          // U row-pair pitch in floats: odd number of 16-byte chunks
    static constexpr int XP = TX + 4;                            // X row pitch
    static constexpr int XPP = ((2 * XP / 4) | 1) * 4;           // X row-pair pitch: odd number of 16-byte chunks
    static constexpr int O4 = (2 * OFF) / 4, O2 = (2 * OFF) % 4; // first chunk / float of an x-pass run inside its segment
    static constexpr int NV = (O2 + 2 * (LX + 2 * K) + 3) / 4;   // 16-byte chunks of one x-pass run (two rows)
    static constexpr int P1_TASKS = NRP * NG;
    static constexpr int P2_TASKS = 3 * NRP * (TX / LX);
    static constexpr int P3_TASKS = 3 * (TX / 4) * (TY / LY);
    static constexpr size_t smem_bytes = sizeof(float) * 3 * NRP * (UPP + XPP);
    static_assert(PY % 2 == 0 && TY % LY == 0 && TX % LX == 0 && LX % 4 == 0, "tile shape");
    static_assert(2 * (TX - LX) + 4 * (O4 + NV) <= UPP, "x-pass run must stay inside the U row pair");
};

__device__ __forceinline__ float4 ldg4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

__device__ __forceinline__ float rcp_approx(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// packed fp32x2 add / subtract / multiply (Blackwell): both halves round exactly like the scalar instruction
__device__ __forceinline__ float2 fadd2(float2 a, float2 b) {
    unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a), rb = *reinterpret_cast<unsigned long long*>(&b), rd;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2*>(&rd);
}
__device__ __forceinline__ float2 fsub2(float2 a, float2 b) {
    unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a), rb = *reinterpret_cast<unsigned long long*>(&b), rd;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2*>(&rd);
}
__device__ __forceinline__ float2 fmul2(float2 a, float2 b) {
    unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a), rb = *reinterpret_cast<unsigned long long*>(&b), rd;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(rd) : "l"(ra), "l"(rb));
    return *reinterpret_cast<float2*>(&rd);
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
    // The group's own row and its z neighbours; the y neighbours (sym, syp, [mym, myp]) and the x neighbours
    // (sl, sr, [ml, mr]) are filled in by the caller, which shares them between the two rows of a pair and between
    // the lanes of a warp.
    __device__ __forceinline__ void load(const float* __restrict__ m, const float* __restrict__ s,
                                         const float* __restrict__ rin, int nz, unsigned plane, unsigned N, unsigned i,
                                         int z) {
#pragma unroll
        for (int c = 0; c < 3; ++c) u[c] = ldg4(rin + (i + (unsigned)c * N));
        if (FORCE) {
            const unsigned izp = i + (z < nz - 1 ? plane : 0u), izm = i - (z > 0 ? plane : 0u);
            sc = ldg4(s + i); mm = ldg4(m + i);
            szp = ldg4(s + izp); szm = ldg4(s + izm);
            if (FORCE == kForceDouble) { mzp = ldg4(m + izp); mzm = ldg4(m + izm); }
        }
    }
    // Two points at a time (x-adjacent halves of the 16-byte loads) with packed fp32x2 arithmetic: the same operations
    // in the same order as the scalar form, so every half rounds identically; only the x differences, whose operands
    // straddle the halves, and the two reciprocals are scalar.
    // NORMS (stopping criterion; reading A16): also the sums over the four points of |dr| (the increment
    // about to be added, Euclidean norm) and |r| (the field before the update), as k_force_norms forms them.
    template <bool NORMS>
    __device__ __forceinline__ void finish(float eps_den, float& sum_dr, float& sum_r) {
        if (FORCE) {
            const float2 eps4 = make_float2(4.f * eps_den, 4.f * eps_den);
            const float2 scp[2] = {make_float2(sc.x, sc.y), make_float2(sc.z, sc.w)};
            const float2 mmp[2] = {make_float2(mm.x, mm.y), make_float2(mm.z, mm.w)};
            const float2 ypp[2] = {make_float2(syp.x, syp.y), make_float2(syp.z, syp.w)};
            const float2 ymp[2] = {make_float2(sym.x, sym.y), make_float2(sym.z, sym.w)};
            const float2 zpp[2] = {make_float2(szp.x, szp.y), make_float2(szp.z, szp.w)};
            const float2 zmp[2] = {make_float2(szm.x, szm.y), make_float2(szm.z, szm.w)};
            const float2 Dxp[2] = {make_float2(sc.y - sl, sc.z - sc.x), make_float2(sc.w - sc.y, sr - sc.z)};
            float2 up[3][2] = {{make_float2(u[0].x, u[0].y), make_float2(u[0].z, u[0].w)},
                               {make_float2(u[1].x, u[1].y), make_float2(u[1].z, u[1].w)},
                               {make_float2(u[2].x, u[2].y), make_float2(u[2].z, u[2].w)}};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const float2 Dx = Dxp[h], Dy = fsub2(ypp[h], ymp[h]), Dz = fsub2(zpp[h], zmp[h]);
                const float2 d = fsub2(scp[h], mmp[h]);
                const float2 t = fadd2(d, d);
                const float2 tt = ffma2(t, t, eps4);
                const float2 den = ffma2(Dx, Dx, ffma2(Dy, Dy, ffma2(Dz, Dz, tt)));
                const float2 q = fmul2(t, make_float2(rcp_approx(den.x), rcp_approx(den.y)));
                float2 ax, ay, az;      // the increment itself, for its norm
                if (NORMS) {
                    const float2 r2 = ffma2(up[0][h], up[0][h], ffma2(up[1][h], up[1][h], fmul2(up[2][h], up[2][h])));
                    sum_r += sqrt_approx(r2.x) + sqrt_approx(r2.y);
                    ax = fmul2(q, Dx); ay = fmul2(q, Dy); az = fmul2(q, Dz);
                }
                up[0][h] = ffma2(q, Dx, up[0][h]);
                up[1][h] = ffma2(q, Dy, up[1][h]);
                up[2][h] = ffma2(q, Dz, up[2][h]);
                if (FORCE == kForceDouble) {
                    const float2 Hx = h == 0 ? make_float2(mm.y - ml, mm.z - mm.x) : make_float2(mm.w - mm.y, mr - mm.z);
                    const float2 Hy = h == 0 ? fsub2(make_float2(myp.x, myp.y), make_float2(mym.x, mym.y))
                                             : fsub2(make_float2(myp.z, myp.w), make_float2(mym.z, mym.w));
                    const float2 Hz = h == 0 ? fsub2(make_float2(mzp.x, mzp.y), make_float2(mzm.x, mzm.y))
                                             : fsub2(make_float2(mzp.z, mzp.w), make_float2(mzm.z, mzm.w));
                    const float2 dh = ffma2(Hx, Hx, ffma2(Hy, Hy, ffma2(Hz, Hz, tt)));
                    const float2 p = fmul2(t, make_float2(rcp_approx(dh.x), rcp_approx(dh.y)));
                    if (NORMS) { ax = ffma2(p, Hx, ax); ay = ffma2(p, Hy, ay); az = ffma2(p, Hz, az); }
                    up[0][h] = ffma2(p, Hx, up[0][h]);
                    up[1][h] = ffma2(p, Hy, up[1][h]);
                    up[2][h] = ffma2(p, Hz, up[2][h]);
                }
                if (NORMS) {
                    const float2 n2 = ffma2(ax, ax, ffma2(ay, ay, fmul2(az, az)));
                    sum_dr += sqrt_approx(n2.x) + sqrt_approx(n2.y);
                }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) u[c] = make_float4(up[c][0].x, up[c][0].y, up[c][1].x, up[c][1].y);
        }
    }
};

// The tile is 64 x TY_: 32 rows at the fine levels; 8 rows where a level has fewer 64 x 32 tiles than the device has
// CTA slots (64 x 64 x 32: 64 tiles) -- four times the CTAs, each with a quarter of the serial work per phase.
// PERSISTENT: the grid is two CTAs per SM; a CTA walks tiles t = blockIdx.x, += gridDim.x (x fastest, so the CTAs
// running at the same time work on neighbouring tiles and share their halos in L2).  Phase 3 of tile t-1 and
// phase 1 of tile t share one barrier interval -- the y pass (pure FMA work out of shared memory) runs on some
// warps while others wait for phase 1's global loads.
// STOP (the paper's "comparison kernel"): phase 1 also adds up sum|dr| and sum|r| over
// the voxels of the tile proper (every voxel belongs to exactly one tile), per thread in fp64; every CTA leaves its two
// partial sums in its own slot and the last CTA to finish adds them in a fixed association, forms l = sum|dr| / sum|r|,
// files it and sets stop_iter when l(iter-10) - l(iter) <= stop_eps -- no second pass over m, s', r.
template <int K, int FORCE, int TY_, bool STOP>
__global__ void __launch_bounds__(FgT4Cfg<K, TY_>::NT, FgT4Cfg<K, TY_>::OCC)
k_force_gxy_t4(const float* __restrict__ m, const float* __restrict__ s, const float* __restrict__ rin,
               float* __restrict__ rout, int nx, int ny, int nz, float eps_den, GaussTaps gw, IterCtl ctl,
               StopCtl* sctl, int stop_iter_k, float stop_eps) {
    if (iter_skipped(ctl)) return;
    double acc_dr = 0.0, acc_r = 0.0;
    using C = FgT4Cfg<K, TY_>;
    constexpr int W = C::W, TX = C::TX, TY = C::TY, NT = C::NT, LX = C::LX, LY = C::LY, NG = C::NG, NRP = C::NRP;
    constexpr int UPP = C::UPP, XP = C::XP, XPP = C::XPP, KA = C::KA, NV = C::NV;
    extern __shared__ __align__(16) float smem_f[];
    float* U = smem_f;                        // [3][NRP][UPP]
    float* X = smem_f + 3 * NRP * UPP;        // [3][NRP][XPP]

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

        // ================= first interval: phase 1 of tile t, phase 3 of tile t-1
        {
            if (have) {
                // ---- phase 1: updated field at the tile + halo.  A task is a ROW PAIR of one group of four x-adjacent
                // points, all loads issued before either row is evaluated; rows 2rp and 2rp+1 are each other's y
                // neighbours (4 row loads of s' instead of 6).
                for (int p = tid; p < C::P1_TASKS; p += NT) {
                    const int rp = p / NG, g = p - rp * NG;
                    const int gy0 = clampi(y0 - K + 2 * rp, 0, ny - 1), gy1 = clampi(y0 - K + 2 * rp + 1, 0, ny - 1);
                    const int gx = x0 - KA + 4 * g;
                    const int gxc = clampi(gx, 0, nx - 4);
                    const unsigned i0 = (unsigned)z * (unsigned)plane + (unsigned)gy0 * (unsigned)nx + (unsigned)gxc;
                    const unsigned i1 = (unsigned)z * (unsigned)plane + (unsigned)gy1 * (unsigned)nx + (unsigned)gxc;
                    FgGroup<FORCE> G0, G1;
                    G0.load(m, s, rin, nz, (unsigned)plane, (unsigned)N, i0, z);
                    G1.load(m, s, rin, nz, (unsigned)plane, (unsigned)N, i1, z);
                    if (FORCE) {
                        const unsigned dl = gxc > 0 ? 1u : 0u, dr = 3u + (gxc + 4 < nx ? 1u : 0u);
                        const unsigned im = i0 - (gy0 > 0 ? (unsigned)nx : 0u), ip = i1 + (gy1 < ny - 1 ? (unsigned)nx : 0u);
                        const float4 sym0 = ldg4(s + im), syp1 = ldg4(s + ip);
                        G0.sl = __ldg(s + (i0 - dl)); G1.sl = __ldg(s + (i1 - dl));
                        G0.sr = __ldg(s + (i0 + dr)); G1.sr = __ldg(s + (i1 + dr));
                        // rows gy0, gy1 are adjacent, or both clamped to the same border row (then the two groups are equal)
                        const bool adj = gy1 != gy0;
                        G0.sym = sym0; G1.syp = syp1;
                        G0.syp = adj ? G1.sc : syp1;
                        G1.sym = adj ? G0.sc : sym0;
                        if (FORCE == kForceDouble) {
                            const float4 mym0 = ldg4(m + im), myp1 = ldg4(m + ip);
                            G0.ml = __ldg(m + (i0 - dl)); G1.ml = __ldg(m + (i1 - dl));
                            G0.mr = __ldg(m + (i0 + dr)); G1.mr = __ldg(m + (i1 + dr));
                            G0.mym = mym0; G1.myp = myp1;
                            G0.myp = adj ? G1.mm : myp1;
                            G1.mym = adj ? G0.mm : mym0;
                        }
                    }
                    float ndr0 = 0.f, nr0 = 0.f, ndr1 = 0.f, nr1 = 0.f;
                    G0.template finish<STOP>(eps_den, ndr0, nr0);
                    G1.template finish<STOP>(eps_den, ndr1, nr1);
                    if (STOP) {
                        // a group is wholly inside or wholly outside the tile proper and the volume (x0, KA, nx are multiples of 4)
                        const bool in_x = gx >= x0 && gx < x0 + TX && gx < nx;
                        const int rr = 2 * rp - K;
                        const bool in0 = in_x && rr >= 0 && rr < TY && y0 + rr < ny;
                        const bool in1 = in_x && rr + 1 >= 0 && rr + 1 < TY && y0 + rr + 1 < ny;
                        acc_dr += (double)((in0 ? ndr0 : 0.f) + (in1 ? ndr1 : 0.f));
                        acc_r += (double)((in0 ? nr0 : 0.f) + (in1 ? nr1 : 0.f));
                    }
                    // a group wholly outside the volume is the replicate border: the edge group's outermost value
                    if (gx < 0 || gx >= nx) {   // only in the tiles at the volume's x border
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            const float e0 = gx < 0 ? G0.u[c].x : G0.u[c].w, e1 = gx < 0 ? G1.u[c].x : G1.u[c].w;
                            G0.u[c] = make_float4(e0, e0, e0, e0);
                            G1.u[c] = make_float4(e1, e1, e1, e1);
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        float4* up = reinterpret_cast<float4*>(U + (c * NRP + rp) * UPP + 8 * g);
                        up[0] = make_float4(G0.u[c].x, G1.u[c].x, G0.u[c].y, G1.u[c].y);
                        up[1] = make_float4(G0.u[c].z, G1.u[c].z, G0.u[c].w, G1.u[c].w);
                    }
                }
            }
            if (have_prev) {
                // ---- phase 3 of tile t-1: y pass, lanes <-> column groups
                for (int tk = tid; tk < C::P3_TASKS; tk += NT) {
                    const int cg = tk % (TX / 4), q = tk / (TX / 4), h = q % (TY / LY), cc = q / (TY / LY);
                    const float* xb = X + cc * NRP * XPP + cg * 4;
                    float2 a0[LY], a1[LY];
#pragma unroll
                    for (int j = 0; j < LY; ++j) { a0[j] = make_float2(0.f, 0.f); a1[j] = make_float2(0.f, 0.f); }
#pragma unroll
                    for (int i = 0; i < LY + 2 * K; ++i) {
                        const int row = h * LY + i;       // LY is even: the parity of the row is the parity of i
                        const float4 f = *reinterpret_cast<const float4*>(xb + (row >> 1) * XPP + (i & 1) * XP);
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
        }
        if (!have) break;
        __syncthreads();

        // ================= second interval: phase 2 of tile t, x pass over two rows at once, lanes <-> row pairs.
        // Output column x0 + g*LX + j of both rows reads the pairs of columns OFF + g*LX + j + k: one packed FFMA2 per
        // tap and output pair.
        {
            for (int tk = tid; tk < C::P2_TASKS; tk += NT) {
                const int rp = tk % NRP, q = tk / NRP, g = q % (TX / LX), cc = q / (TX / LX);
                const float4* up = reinterpret_cast<const float4*>(U + (cc * NRP + rp) * UPP + 2 * g * LX) + C::O4;
                float2 v[2 * NV];
#pragma unroll
                for (int i = 0; i < NV; ++i) {
                    const float4 f = up[i];
                    v[2 * i] = make_float2(f.x, f.y); v[2 * i + 1] = make_float2(f.z, f.w);
                }
                float2 o[LX];
#pragma unroll
                for (int j = 0; j < LX; ++j) {
                    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
                    for (int k = 0; k < W; ++k) acc = ffma2(make_float2(gw.w[k], gw.w[k]), v[C::O2 / 2 + j + k], acc);
                    o[j] = acc;
                }
                float* xr = X + (cc * NRP + rp) * XPP + g * LX;
#pragma unroll
                for (int q4 = 0; q4 < LX / 4; ++q4) {
                    *reinterpret_cast<float4*>(xr + 4 * q4) = make_float4(o[4 * q4].x, o[4 * q4 + 1].x, o[4 * q4 + 2].x, o[4 * q4 + 3].x);
                    *reinterpret_cast<float4*>(xr + XP + 4 * q4) = make_float4(o[4 * q4].y, o[4 * q4 + 1].y, o[4 * q4 + 2].y, o[4 * q4 + 3].y);
                }
            }
        }
        __syncthreads();
        px0 = x0; py0 = y0; pz = z; have_prev = true;
    }
    if (STOP) {
        const int lane = tid & 31, warp = tid >> 5;
        __shared__ double sh[2][NT / 32];
        __shared__ bool last;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc_dr += __shfl_xor_sync(0xffffffffu, acc_dr, o);
            acc_r += __shfl_xor_sync(0xffffffffu, acc_r, o);
        }
        if (lane == 0) { sh[0][warp] = acc_dr; sh[1][warp] = acc_r; }
        __syncthreads();
        if (tid == 0) {
            double ta = 0.0, tb = 0.0;
            for (int w = 0; w < NT / 32; ++w) { ta += sh[0][w]; tb += sh[1][w]; }
            sctl->partial[2 * blockIdx.x] = ta; sctl->partial[2 * blockIdx.x + 1] = tb;
            __threadfence();
            last = atomicAdd(&sctl->ticket, 1u) == gridDim.x - 1;
        }
        __syncthreads();
        if (last) {   // fixed association: thread i takes CTAs i, i + NT, ... in rising order, then a fixed tree
            __threadfence();
            double sdr = 0.0, sr = 0.0;
            for (unsigned k = tid; k < gridDim.x; k += NT) { sdr += sctl->partial[2 * k]; sr += sctl->partial[2 * k + 1]; }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                sdr += __shfl_xor_sync(0xffffffffu, sdr, o);
                sr += __shfl_xor_sync(0xffffffffu, sr, o);
            }
            __syncthreads();
            if (lane == 0) { sh[0][warp] = sdr; sh[1][warp] = sr; }
            __syncthreads();
            if (tid == 0) {
                sdr = 0.0; sr = 0.0;
                for (int w = 0; w < NT / 32; ++w) { sdr += sh[0][w]; sr += sh[1][w]; }
                const double l = sr > 0.0 ? sdr / sr : (double)INFINITY;
                sctl->hist[stop_iter_k & 15] = l;
                if (stop_iter_k >= 10 && sctl->hist[(stop_iter_k - 10) & 15] - l <= (double)stop_eps) sctl->stop_iter = stop_iter_k;
                sctl->ticket = 0u;
                __threadfence();
            }
        }
    }
}

}  // namespace disc
