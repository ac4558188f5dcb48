// moments_v2.cuh -- patch moments + intensity correction, the warp-specialised sm_100a kernel (step (a)).
//
// Same sums as moments.cuh (PAPER.md:95 Eq. 3, :117-119 Eqs. 5-6, :458 A.4; readings A4, A5): separable
// sliding-window box sums of v and v^2 in fp64, cost independent of R.  What differs is the machinery:
//
//   * one fat CTA per SM owns a 32 x TY (x,y) tile and marches z through a chunk;
//   * three roles run concurrently on different slices, handing buffers over through mbarriers:
//       producer (1 thread)  3-D TMA tile loads of the zero-padded raw slice, NSTG slices ahead;
//       x pass   (NP1 thr.)  task = (row, run of 8 outputs), lanes <-> rows: fp32 -> fp64, slides S1 and S2
//                            along x, writes (S1,S2) pairs to a shared-memory exchange buffer (NXS deep);
//       y/z pass (NP2 thr.)  task = (column x, run of 4 rows, ONE of the two sums), lanes <-> (x, sum): slides
//                            its sum along y, updates its z window; the S1 and S2 threads of a column then
//                            swap two window sums by shuffle and each evaluates mu, var and the mode's
//                            output for two of the four voxels;
//   * the z window -- the last 2R+1 xy box sums of every column of the tile, fp64 -- lives in TENSOR MEMORY:
//     each y/z thread keeps a private ring in its TMEM lane and moves one slot per slice with
//     tcgen05.ld / tcgen05.st (8 words).  176 B per column (R = 5) would otherwise pin 180 KB of shared
//     memory for a 32x32 tile; in TMEM it costs no shared memory, no registers and no unrolled ring code.
//
// Requirements (checked by the launcher): nx % 4 == 0, 16-byte aligned volume (tensor-map rules).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "launch.h"
#include "pipeline.cuh"

namespace disc {

constexpr uint32_t pow2_tmem_cols(uint32_t n) { return n <= 32 ? 32 : n <= 64 ? 64 : n <= 128 ? 128 : n <= 256 ? 256 : 512; }

template <int R, int TY>
struct MomV2Cfg {
    static constexpr int W = 2 * R + 1;
    static constexpr int TX = 32;
    static constexpr int LX = 8, LY = 4;
    static constexpr int PX = TX + 2 * R, PY = TY + 2 * R;
    static constexpr int NP2 = 2 * TX * TY / LY;                       // y/z-pass threads (512 or 256): one per sum
    static constexpr int P1_TASKS = PY * (TX / LX);
    static constexpr int NP1 = (P1_TASKS + 31) / 32 * 32;              // x-pass threads
    static constexpr int NT = NP2 + NP1 + 32;                          // + the producer warp
    // The innermost TMA coordinate must be a multiple of 4 floats, so the box starts at x0 - RA (RA = R rounded
    // up to 4) and column x0 - R sits at offset OFF of a raw row; the box width is a multiple of 4 floats with
    // an odd number of 16-byte chunks (lanes <-> rows reads are then bank-conflict free).
    static constexpr int RA = (R + 3) / 4 * 4, OFF = RA - R;
    static constexpr int PXB = (((OFF + PX + 3) / 4) | 1) * 4;
#ifndef DISC_MOM_NSTG
#define DISC_MOM_NSTG 8
#define DISC_MOM_NXS 3
#define DISC_MOM_NAUX 8
#endif
    static constexpr int NSTG = DISC_MOM_NSTG, NXS = DISC_MOM_NXS, NAUX = DISC_MOM_NAUX;                  // raw stages, exchange buffers, aux stages
    static constexpr int XSP = TX + 1;                                 // exchange-row pitch in (S1,S2) pairs, odd
    static constexpr size_t raw_bytes = sizeof(float) * PY * PXB;      // one stage; multiple of 16
    static constexpr size_t raw_stride = (raw_bytes + 127) / 128 * 128;
    static constexpr size_t xs_bytes = sizeof(double2) * PY * XSP;
    static constexpr size_t aux_bytes = sizeof(float) * TX * TY;       // one stage of the per-voxel operand (no halo)
    static constexpr size_t smem_bytes = 128 + NSTG * raw_stride + NXS * xs_bytes + NAUX * aux_bytes;
    static constexpr int RING_WORDS = 2 * LY;                          // one ring slot of one thread: LY fp64 sums
    static constexpr uint32_t tmem_needed = (NP2 / 128) * RING_WORDS * W;
    static constexpr uint32_t tmem_cols = pow2_tmem_cols(tmem_needed);
    static_assert(tmem_needed <= 512, "z ring does not fit tensor memory: use the smaller tile");
    static_assert(NP2 % 128 == 0, "y/z warps must fill whole TMEM lane quadrant groups");
};

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(v[0]),
                 "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

template <int R, int TY, int MODE>
__global__ void __launch_bounds__(MomV2Cfg<R, TY>::NT, TY == 16 ? 2 : 1)
k_moments_v2(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap_aux,
             float* __restrict__ out0, float* __restrict__ out1, int nx, int ny, int nz, int zchunk, float eps_var,
             IterCtl ctl) {
    if (iter_skipped(ctl)) return;
    using C = MomV2Cfg<R, TY>;
    constexpr int W = C::W, PY = C::PY, PXB = C::PXB, LX = C::LX, LY = C::LY, XSP = C::XSP;
    constexpr int NP1 = C::NP1, NP2 = C::NP2, NSTG = C::NSTG, NXS = C::NXS, NAUX = C::NAUX, TX = C::TX;
    constexpr int RAWS = (int)(C::raw_stride / sizeof(float));
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float* raw = reinterpret_cast<float*>(smem_raw);                                          // [NSTG][PY][PXB]
    float* auxs = reinterpret_cast<float*>(smem_raw + (size_t)NSTG * C::raw_stride);           // [NAUX][TY][TX]
    double2* xs = reinterpret_cast<double2*>(smem_raw + (size_t)NSTG * C::raw_stride + (size_t)NAUX * C::aux_bytes);  // [NXS][PY][XSP]
    __shared__ uint64_t raw_full[NSTG], raw_empty[NSTG], xs_full[NXS], xs_empty[NXS], aux_full[NAUX], aux_empty[NAUX];
    __shared__ uint32_t tmem_base_s;
    __shared__ double inv_cnt_z[W + 1];

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, nz);
    const size_t plane = (size_t)nx * ny;
    const int zfirst = max(z0 - R, 0), zlast = min(z1 - 1 + R, nz - 1);   // slices that exist; the others are zero
    const int T = zlast - zfirst + 1;

    if (tid == 0) {
        for (int i = 0; i < NSTG; ++i) { mbar_init(&raw_full[i], 1); mbar_init(&raw_empty[i], NP1); }
        for (int i = 0; i < NXS; ++i) { mbar_init(&xs_full[i], NP1); mbar_init(&xs_empty[i], NP2); }
        for (int i = 0; i < NAUX; ++i) { mbar_init(&aux_full[i], 1); mbar_init(&aux_empty[i], NP2); }
        mbar_fence_init();
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                     "n"(C::tmem_cols)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    if (tid <= W) inv_cnt_z[tid] = tid > 0 ? 1.0 / (double)tid : 0.0;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = tmem_base_s;

    if (warp < NP2 / 32) {
        // ------------------------------------------------------------------ y pass, z window, evaluation
        // lane = 2*xl + q: q = 0 slides S1, q = 1 slides S2 of column x = 16*(warp & 1) + xl, rows yb .. yb+3
        static_assert(LY == 4, "the S1/S2 thread pair splits four voxels two and two");
        const int q = lane & 1, px = (warp & 1) * 16 + (lane >> 1), yb = (warp >> 1) * LY;
        const int gx = x0 + px;
        // this thread's ring: TMEM lane = its own lane of the warp's quadrant, 8 words per slice
        const uint32_t ring0 = tmem_base + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(warp >> 2) * (C::RING_WORDS * W);
        {
            uint32_t zero[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) zero[i] = 0u;
            for (int j = 0; j < W; ++j) tmem_st8(ring0 + j * C::RING_WORDS, zero);
        }
        double Z[LY];
#pragma unroll
        for (int o = 0; o < LY; ++o) Z[o] = 0.0;
        // the two voxels this thread evaluates: rows ye, ye + 1
        const int ye = yb + 2 * q;
        double inv_nxy[2];
        bool live[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const int gy = y0 + ye + k;
            const int cx = min(gx + R, nx - 1) - max(gx - R, 0) + 1;
            const int cy = min(gy + R, ny - 1) - max(gy - R, 0) + 1;
            live[k] = gx < nx && gy < ny;
            inv_nxy[k] = live[k] ? 1.0 / ((double)cx * (double)cy) : 0.0;
        }
        // output pointers of the thread's first voxel at slice z0; += plane per emitted slice
        const size_t o0 = (size_t)z0 * plane + (size_t)min(y0 + ye, ny - 1) * nx + min(gx, nx - 1);
        float* op0 = out0 + o0;
        float* op1 = MODE == kModeMoments ? out1 + o0 : nullptr;
        const double* xq = reinterpret_cast<const double*>(xs) + (size_t)(yb * XSP + px) * 2 + q;
        const float* auxq = auxs + ye * TX + px;
        int slot = 0, tv = 0;
        for (int zz = z0 - R; zz < z1 + R; ++zz) {
            const bool valid = zz >= 0 && zz < nz;   // uniform
            const int zo = zz - R;
            const bool emit = zo >= z0;
            uint32_t old[8];
            tmem_wait_st();                                  // the slot written W slices ago has landed
            tmem_ld8(ring0 + slot * C::RING_WORDS, old);
            double b[LY];
            if (valid) {
                const int buf = tv % NXS;
                mbar_wait(&xs_full[buf], (tv / NXS) & 1);
                const double* ip = xq + (size_t)buf * PY * XSP * 2;
                double v[LY + 2 * R];
#pragma unroll
                for (int i = 0; i < LY + 2 * R; ++i) v[i] = ip[i * XSP * 2];
                mbar_arrive(&xs_empty[buf]);
                // window sum of output 0 as a balanced tree (short dependency chains), then three slides
                double t[W];
#pragma unroll
                for (int i = 0; i < W; ++i) t[i] = v[i];
#pragma unroll
                for (int n = W; n > 1; n = (n + 1) / 2)
#pragma unroll
                    for (int i = 0; i < n / 2; ++i) t[i] = t[i] + t[n - 1 - i];
                b[0] = t[0];
#pragma unroll
                for (int o = 1; o < LY; ++o) b[o] = b[o - 1] + (v[o + 2 * R] - v[o - 1]);
                ++tv;
            } else {
#pragma unroll
                for (int o = 0; o < LY; ++o) b[o] = 0.0;
            }
            tmem_wait_ld();
            uint32_t nw[8];
#pragma unroll
            for (int o = 0; o < LY; ++o) {
                Z[o] += b[o] - __hiloint2double((int)old[2 * o + 1], (int)old[2 * o]);
                nw[2 * o] = (uint32_t)__double2loint(b[o]); nw[2 * o + 1] = (uint32_t)__double2hiint(b[o]);
            }
            tmem_st8(ring0 + slot * C::RING_WORDS, nw);
            slot = slot + 1 == W ? 0 : slot + 1;
            if (emit) {   // uniform
                // swap: the S1 thread hands over its sums of voxels 2,3 and receives S2 of voxels 0,1 (and vice versa)
                double mine[2], theirs[2];
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double give = q ? Z[k] : Z[2 + k];
                    mine[k] = q ? Z[2 + k] : Z[k];
                    theirs[k] = __shfl_xor_sync(0xffffffffu, give, 1);
                }
                // the per-voxel operand of the output slice (the volume itself for the z-score, the cached CBCT
                // z-score for the correction) arrives by TMA, prefetched NAUX slices ahead
                float pre[2] = {0.f, 0.f};
                if (MODE != kModeMoments) {
                    const int e = zo - z0, as = e % NAUX;
                    mbar_wait(&aux_full[as], (e / NAUX) & 1);
#pragma unroll
                    for (int k = 0; k < 2; ++k) pre[k] = auxq[(size_t)as * TX * TY + k * TX];
                    mbar_arrive(&aux_empty[as]);
                }
                const double inv_cz = inv_cnt_z[min(zo + R, nz - 1) - max(zo - R, 0) + 1];
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double z1s = q ? theirs[k] : mine[k], z2s = q ? mine[k] : theirs[k];
                    const double inv_n = inv_nxy[k] * inv_cz;
                    const double mu = z1s * inv_n;
                    const double var = fma(-mu, mu, z2s * inv_n);
                    const float varf = fmaxf((float)var, 0.f);
                    float r0;
                    if (MODE == kModeMoments) {
                        r0 = (float)mu;
                    } else if (MODE == kModeZscore) {
                        const float dv = (float)((double)pre[k] - mu);
                        r0 = var > (double)eps_var ? dv * rsqrtf(varf) : 0.f;
                    } else {
                        // sigma = var * rsqrt(var): two instructions instead of the IEEE square root's ten; the
                        // approximation's 2 ulp are 1e-7 of sigma, far inside the 1e-4 x range budget
                        const float sd = varf > 0.f ? varf * rsqrtf(varf) : 0.f;
                        r0 = fmaf(sd, pre[k], (float)mu);
                    }
                    if (live[k]) {
                        op0[(size_t)k * nx] = r0;
                        if (MODE == kModeMoments) op1[(size_t)k * nx] = varf;
                    }
                }
                op0 += plane;
                if (MODE == kModeMoments) op1 += plane;
            }
        }
        tmem_wait_st();
    } else if (warp < (NP2 + NP1) / 32) {
        // ------------------------------------------------------------------ x pass
        const int t1 = tid - NP2;
        const bool has = t1 < C::P1_TASKS;
        const int g = t1 / PY, r = t1 - g * PY;       // lanes <-> rows
        constexpr int O4 = C::OFF & ~3, O1 = C::OFF & 3;
        constexpr int NV = (O1 + LX + 2 * R + 3) / 4;
        for (int t = 0; t < T; ++t) {
            const int st = t % NSTG, buf = t % NXS;
            mbar_wait(&raw_full[st], (t / NSTG) & 1);
            double dd[NV * 4];
            if (has) {
                // the run starts at float OFF + g*LX of the row: read from the aligned chunk below it
                const float4* rp = reinterpret_cast<const float4*>(raw + (size_t)st * RAWS + r * PXB + g * LX + O4);
#pragma unroll
                for (int i = 0; i < NV; ++i) {
                    const float4 f = rp[i];
                    dd[4 * i] = (double)f.x; dd[4 * i + 1] = (double)f.y; dd[4 * i + 2] = (double)f.z; dd[4 * i + 3] = (double)f.w;
                }
            }
            mbar_arrive(&raw_empty[st]);
            if (t >= NXS) mbar_wait(&xs_empty[buf], ((t / NXS) - 1) & 1);
            if (has) {
                const double* d = dd + O1;
                // first window as balanced trees (short dependency chains), then LX-1 slides
                double t1[W], t2[W];
#pragma unroll
                for (int i = 0; i < W; ++i) { t1[i] = d[i]; t2[i] = d[i] * d[i]; }
#pragma unroll
                for (int n = W; n > 1; n = (n + 1) / 2)
#pragma unroll
                    for (int i = 0; i < n / 2; ++i) { t1[i] = t1[i] + t1[n - 1 - i]; t2[i] = t2[i] + t2[n - 1 - i]; }
                double s1 = t1[0], s2 = t2[0];
                double2* op = xs + (size_t)buf * PY * XSP + r * XSP + g * LX;
                op[0] = make_double2(s1, s2);
#pragma unroll
                for (int o = 1; o < LX; ++o) {
                    // d_new^2 - d_old^2 = (d_new - d_old)(d_new + d_old), exact in fp64 for fp32 inputs
                    const double e = d[o + 2 * R] - d[o - 1], f = d[o + 2 * R] + d[o - 1];
                    s1 += e;
                    s2 = fma(e, f, s2);
                    op[o] = make_double2(s1, s2);
                }
            }
            mbar_arrive(&xs_full[buf]);
        }
    } else if (tid == NP2 + NP1) {
        // ------------------------------------------------------------------ producer
        int t = 0;
        for (int zz = z0 - R; zz < z1 + R; ++zz) {
            if (zz >= 0 && zz < nz) {
                const int st = t % NSTG;
                if (t >= NSTG) mbar_wait(&raw_empty[st], ((t / NSTG) - 1) & 1);
                mbar_expect_tx(&raw_full[st], (uint32_t)C::raw_bytes);
                tma_load_3d(raw + (size_t)st * RAWS, &tmap, x0 - C::RA, y0 - R, zz, &raw_full[st]);
                ++t;
            }
            const int e = zz - R - z0;      // output slice of this step
            if (MODE != kModeMoments && e >= 0) {
                const int as = e % NAUX;
                if (e >= NAUX) mbar_wait(&aux_empty[as], ((e / NAUX) - 1) & 1);
                mbar_expect_tx(&aux_full[as], (uint32_t)C::aux_bytes);
                tma_load_3d(auxs + (size_t)as * TX * TY, &tmap_aux, x0, y0, z0 + e, &aux_full[as]);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(C::tmem_cols) : "memory");
}

}  // namespace disc
