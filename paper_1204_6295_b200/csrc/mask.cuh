// mask.cuh -- SURVEY NEXT-1: the paper's reliability mask and the interpolation / extrapolation of a, b
// (Eqs. (5)-(10); parameters PAPER.md:161, :165), plus the Fig.-9 averages of a and b
// (PAPER.md:398-402).  Everything is decided on the device: the parameters (Delta HU, HU_0, a_m, a_min, a_max) live in
// a MaskCtl in device memory that the kernels read, the fill passes stop through a device-side counter, so the
// registration still enqueues its whole schedule without a host synchronisation.
//
//   k_sum2            sum(ct), sum(cbct) -> Delta HU = mean(ct) - mean(cbct), HU_0 = 2 |Delta HU|
//   k_shift           cbct + Delta HU  ("globally adjust the intensity of CBCT", Alg. A1)
//   k_ab_mask         a = STD(M)/STD(S), b = E(M) - a E(S); xi by Eq. (7); a = b = 0 where xi = 1
//   k_select_*        a_m = lower median of a over the voxels with both variances > eps (radix select)
//   k_fill_list       Eqs. (8)-(10): all Jacobi passes over the cube T in ONE cooperative launch, over the compacted
//                     list of masked voxels that k_ab_mask wrote (grid barrier between passes)
//   k_fill_pass       the same, one launch per pass over the whole volume (volumes of >= 2^32 voxels only)
//   k_apply_ab        I'_s = a I_s + b, and the sums of a and b
#pragma once
#include <cooperative_groups.h>
#include <float.h>

#include "common.cuh"

namespace disc {

constexpr unsigned char kXiFree = 0;        // xi = 0: a, b from Eqs. (5)-(6)
constexpr unsigned char kXiMasked = 255;    // xi = 1 and not filled yet; 1..254: filled in that pass

struct MaskCtl {
    double sum_ct, sum_cbct;     // k_sum2 accumulators (block partials added in block order by the last block)
    double delta_hu;             // mean(ct) - mean(cbct)
    float hu0, a_m, a_min, a_max;
    // radix select of the median
    unsigned hist[256];
    unsigned long long count;    // qualifying voxels
    unsigned long long rank;     // remaining rank inside the current prefix
    unsigned prefix;             // bits of the median fixed so far
    // fill passes
    unsigned remaining, filled, prev_filled, ticket;
    unsigned n_list[257];        // k_fill_list: n_list[p] = length of the work list of pass p (slot 1: all xi = 1 voxels)
    // diagnostics of the running iteration
    double sum_a, sum_b;
    unsigned ticket2;
};

// ---------------------------------------------------------------- Delta HU
// Deterministic two-stage sum: every block writes its partial, the last block to finish adds them in block order.
static __global__ void __launch_bounds__(256)
k_sum2(const float* __restrict__ ct, const float* __restrict__ cbct, size_t N, double* __restrict__ partial, MaskCtl* ctl,
       float hu0_fixed) {
    double a = 0.0, b = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        a += (double)__ldg(ct + i);
        b += (double)__ldg(cbct + i);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    __shared__ double sh[2][8];
    __shared__ bool last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][warp] = a; sh[1][warp] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0.0, tb = 0.0;
        for (int w = 0; w < 8; ++w) { ta += sh[0][w]; tb += sh[1][w]; }
        partial[2 * blockIdx.x] = ta; partial[2 * blockIdx.x + 1] = tb;
        __threadfence();
        last = atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        double ta = 0.0, tb = 0.0;
        for (unsigned k = 0; k < gridDim.x; ++k) { ta += partial[2 * k]; tb += partial[2 * k + 1]; }
        ctl->sum_ct = ta; ctl->sum_cbct = tb;
        ctl->delta_hu = (ta - tb) / (double)N;
        ctl->hu0 = hu0_fixed >= 0.f ? hu0_fixed : (float)(2.0 * fabs(ctl->delta_hu));
        ctl->ticket = 0u;
    }
}

static __global__ void __launch_bounds__(256)
k_shift(const float* __restrict__ in, float* __restrict__ out, size_t N, const MaskCtl* __restrict__ ctl) {
    const double d = ctl->delta_hu;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x)
        out[i] = (float)((double)__ldg(in + i) + d);
}

static __global__ void k_mask_set(MaskCtl* ctl, float hu0, float a_min, float a_max) {
    if (hu0 >= 0.f) ctl->hu0 = hu0;
    if (a_min >= 0.f) { ctl->a_min = a_min; ctl->a_max = a_max; }
}

// ---------------------------------------------------------------- a, b and the mask
// In place: A holds E(M) on entry and a on exit, B holds VAR(M) on entry and b on exit.  With USE_MASK = false only
// Eqs. (5)-(6) are evaluated (xi = 0 everywhere): that is what the median of A before the DIR and the diagnostics of
// the unmasked path use.
template <bool USE_MASK>
__global__ void __launch_bounds__(256)
k_ab_mask(const float* __restrict__ m, const float* __restrict__ cbct, const float* __restrict__ mu_s,
          const float* __restrict__ var_s, float* __restrict__ A, float* __restrict__ B, unsigned char* __restrict__ xi,
          size_t N, float eps_var, MaskCtl* ctl, IterCtl ictl, unsigned* __restrict__ list, unsigned* __restrict__ queued) {
    if (iter_skipped(ictl)) return;   // after an early stop A, B already hold a, b (not E(M), VAR(M)): leave them
    const float hu0 = ctl->hu0, a_min = ctl->a_min, a_max = ctl->a_max;
    unsigned masked = 0;
    // the loop bound is rounded up to whole blocks: all threads of a block run the same number of rounds and meet at
    // the barriers of the list append below
    const size_t NB = (N + blockDim.x - 1) / blockDim.x * blockDim.x;
    __shared__ unsigned warp_cnt[8], blk_base;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < NB; i += (size_t)gridDim.x * blockDim.x) {
        bool x = false;
        if (i < N) {
            const float mu_m = A[i], var_m = B[i], vs = __ldg(var_s + i);
            const float a = vs > eps_var ? sqrtf(var_m / vs) : 0.f;          // Eq. (5); reading A5
            const float b = fmaf(-a, __ldg(mu_s + i), mu_m);                 // Eq. (6)
            if (USE_MASK) {
                // Eq. (7): the difference of two fp32 values is taken in fp64 (exact), as is the comparison
                const double d = fabs((double)__ldg(m + i) - (double)__ldg(cbct + i));
                x = d > (double)hu0 || a < a_min || a > a_max;
            }
            A[i] = x ? 0.f : a;                                              // "Initially a = b = 0 for xi = 1"
            B[i] = x ? 0.f : b;
            if (xi) xi[i] = x ? kXiMasked : kXiFree;
            masked += x ? 1u : 0u;
            if (USE_MASK && queued != nullptr && (i & 31) == 0) queued[i >> 5] = 0u;   // k_fill_list's "already queued" bits
        }
        if (USE_MASK && list != nullptr) {
            // compacted list of the masked voxels = the work list of fill pass 1 (the order is arbitrary and never
            // matters: a fill pass treats every listed voxel independently); one atomic per block and round
            const unsigned vote = __ballot_sync(0xffffffffu, x);
            const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
            if (lane == 0) warp_cnt[warp] = (unsigned)__popc(vote);
            __syncthreads();
            if (threadIdx.x == 0) {
                unsigned tot = 0;
                for (int w = 0; w < 8; ++w) tot += warp_cnt[w];
                blk_base = tot ? atomicAdd(&ctl->n_list[1], tot) : 0u;
            }
            __syncthreads();
            if (x) {
                unsigned off = blk_base;
                for (int w = 0; w < warp; ++w) off += warp_cnt[w];
                list[off + __popc(vote & ((1u << lane) - 1u))] = (unsigned)i;
            }
            __syncthreads();                                                 // warp_cnt, blk_base are reused next round
        }
    }
    // the count of masked voxels for k_fill_pass (the list path has it as n_list[1]); one same-address atomic per warp
    // is what this kernel's time would be made of (0.6 ns each), so only the fallback pays it
    if (USE_MASK && list == nullptr) {
        masked = __reduce_add_sync(0xffffffffu, masked);
        if ((threadIdx.x & 31) == 0 && masked) atomicAdd(&ctl->remaining, masked);
    }
}

// ---------------------------------------------------------------- median of A (reading A17)
// 4 passes of an 8-bit radix select on the bit pattern of a >= 0 (monotonic), over the voxels where Eq. (5) is a ratio of
// two positive deviations.  pass = 0 also counts the qualifying voxels.
static __global__ void __launch_bounds__(256)
k_select_hist(const float* __restrict__ var_s, const float* __restrict__ var_m, size_t N, float eps_var, int pass,
              MaskCtl* ctl) {
    __shared__ unsigned h[256];
    h[threadIdx.x] = 0u;
    __syncthreads();
    const unsigned prefix = ctl->prefix;
    const int shift = 24 - 8 * pass;
    const unsigned himask = pass == 0 ? 0u : 0xffffffffu << (shift + 8);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const float vs = __ldg(var_s + i), vm = __ldg(var_m + i);
        if (!(vs > eps_var && vm > eps_var)) continue;
        const unsigned bits = __float_as_uint(sqrtf(vm / vs));          // Eq. (5), the same expression as k_ab_mask
        if ((bits & himask) == (prefix & himask)) atomicAdd(&h[(bits >> shift) & 255u], 1u);
    }
    __syncthreads();
    if (h[threadIdx.x]) atomicAdd(&ctl->hist[threadIdx.x], h[threadIdx.x]);
}

static __global__ void k_select_step(int pass, MaskCtl* ctl) {
    if (pass == 0) {
        unsigned long long n = 0;
        for (int b = 0; b < 256; ++b) n += ctl->hist[b];
        ctl->count = n;
        ctl->rank = n ? (n - 1) / 2 : 0;                                 // lower median
    }
    unsigned long long r = ctl->rank;
    int b = 0;
    if (ctl->count) {
        for (; b < 255; ++b) {
            if (r < ctl->hist[b]) break;
            r -= ctl->hist[b];
        }
    }
    ctl->rank = r;
    ctl->prefix |= (unsigned)b << (24 - 8 * pass);
    for (int k = 0; k < 256; ++k) ctl->hist[k] = 0u;
    if (pass == 3) {
        ctl->a_m = ctl->count ? __uint_as_float(ctl->prefix) : 1.f;      // no qualifying voxel: a_m = 1
        ctl->a_min = 0.5f * ctl->a_m;
        ctl->a_max = 1.5f * ctl->a_m;
        ctl->prefix = 0u;
    }
}

// ---------------------------------------------------------------- Eqs. (8)-(10)
// One Jacobi pass `pass` (1..254): a voxel with xi = masked looks at the voxels of T (cube of radius rt, truncated to
// the volume) that were available before this pass (stamp < pass), takes w = exp(-((D)^2 - min D^2) / h^2) (the same
// quotient as Eqs. (8)-(9), normalised by the largest weight so that it cannot underflow to 0/0) and, if there is one,
// writes its a, b and stamps itself with `pass`.  Stamps written in this pass are >= pass, so nobody reads them in this
// pass: the update is in place and race free.  The last block rolls the counters; when nothing is left, or a pass
// filled nothing, the remaining passes fall through.
static __global__ void __launch_bounds__(128)
k_fill_pass(const float* __restrict__ cbct, float* __restrict__ A, float* __restrict__ B, unsigned char* __restrict__ xi,
            int nx, int ny, int nz, int rt, float inv_h2, int pass, MaskCtl* ctl, IterCtl ictl) {
    if (iter_skipped(ictl)) return;
    {
        const volatile MaskCtl* c = ctl;
        if (c->remaining == 0u || (pass > 1 && c->prev_filled == 0u)) return;
    }
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y, z = blockIdx.z;
    unsigned mine = 0;
    if (x < nx) {
        const size_t i0 = ((size_t)z * ny + y) * nx + x;
        if (xi[i0] == kXiMasked) {
            const float s0 = __ldg(cbct + i0);
            const int xa = max(x - rt, 0), xb = min(x + rt, nx - 1);
            const int ya = max(y - rt, 0), yb = min(y + rt, ny - 1);
            const int za = max(z - rt, 0), zb = min(z + rt, nz - 1);
            float dmin = FLT_MAX;
            for (int c = za; c <= zb; ++c)
                for (int b = ya; b <= yb; ++b) {
                    const size_t row = ((size_t)c * ny + b) * nx;
                    for (int a = xa; a <= xb; ++a) {
                        if (xi[row + a] >= pass) continue;
                        const float d = __ldg(cbct + row + a) - s0;
                        dmin = fminf(dmin, d * d);
                    }
                }
            if (dmin < FLT_MAX) {
                float sw = 0.f, sa = 0.f, sb = 0.f;
                for (int c = za; c <= zb; ++c)
                    for (int b = ya; b <= yb; ++b) {
                        const size_t row = ((size_t)c * ny + b) * nx;
                        for (int a = xa; a <= xb; ++a) {
                            if (xi[row + a] >= pass) continue;
                            const float d = __ldg(cbct + row + a) - s0;
                            const float w = __expf(-(d * d - dmin) * inv_h2);      // Eq. (10)
                            sw += w;
                            sa = fmaf(w, A[row + a], sa);
                            sb = fmaf(w, B[row + a], sb);
                        }
                    }
                A[i0] = sa / sw;                                                   // Eqs. (8), (9)
                B[i0] = sb / sw;
                __threadfence();
                xi[i0] = (unsigned char)pass;
                mine = 1u;
            }
        }
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    __shared__ unsigned blk;
    __shared__ bool last;
    if (threadIdx.x == 0) blk = 0u;
    __syncthreads();
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(&blk, mine);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (blk) atomicAdd(&ctl->filled, blk);
        __threadfence();
        const unsigned total = gridDim.x * gridDim.y * gridDim.z;
        last = atomicAdd(&ctl->ticket, 1u) == total - 1;
        if (last) {
            __threadfence();
            const unsigned f = atomicAdd(&ctl->filled, 0u);
            ctl->remaining -= f;
            ctl->prev_filled = f;
            ctl->filled = 0u;
            ctl->ticket = 0u;
            __threadfence();
        }
    }
}

// All passes in one cooperative launch (every block of the grid is resident; a grid barrier separates the passes), each
// pass over a work list instead of the volume.  Pass 1 works on the list of all xi = 1 voxels that k_ab_mask wrote.  A
// voxel can be filled in pass p > 1 only if a voxel of its cube T was filled in pass p - 1 (else it would have been
// filled earlier), so whoever fills a voxel in pass p puts the still unfilled voxels of ITS cube T on the list of pass
// p + 1 (T is symmetric); a bit per voxel (`queued`, cleared by k_ab_mask and again by the pass that takes the voxel
// off its list) keeps a voxel from being listed twice.  Every voxel on the list of a pass p > 1 therefore does get
// filled in that pass, the cost of a pass is proportional to what it fills, and the interior of a large masked region
// is looked at once (pass 1) instead of once per pass.  An empty next list is exactly "nothing left, or a pass that
// filled nothing".  Same arithmetic, same order of the sums over T and same stamps as k_fill_pass.
// A pass reads a, b and stamps < pass only of voxels written before the last grid barrier; a stamp written in the
// running pass reads either 255 or `pass`, both "not available", and at worst lists a voxel that is filled already
// (skipped when its turn comes).  a, b, xi are read with plain (coherent) loads, never __ldg: they change during the
// launch.  The two lists alternate between list_a (pass 1, 3, ...) and list_b (pass 2, 4, ...).
// The loops over T run over all (2 rt + 1)^3 offsets with clamped addresses and an "inside the volume" predicate, every
// load issued before anything depends on it.  (Measured at 256x256x128, 25 % masked: 724 us against 790 us for loops over
// the clipped ranges with `continue`; fully unrolled compile-time radii took 212 registers, one block per SM, 2.7 ms.)
static __global__ void __launch_bounds__(256)
k_fill_list(const float* __restrict__ cbct, float* A, float* B, unsigned char* xi, unsigned* list_a, unsigned* list_b,
            unsigned* queued, int nx, int ny, int nz, int rt, float inv_h2, int max_passes, MaskCtl* ctl, IterCtl ictl) {
    if (iter_skipped(ictl)) return;                       // uniform over the grid: nobody reaches a barrier
    unsigned n = ctl->n_list[1];
    if (n == 0u) return;                                  // idem
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const unsigned stride = gridDim.x * blockDim.x;
    // voxels found for the next pass are collected per block in shared memory and appended to the global list with one
    // atomic per block and round (a single global counter bumped once per voxel serialises the whole grid)
    constexpr unsigned kQ = 2048;
    __shared__ unsigned q[kQ], qn, qbase;
    for (int pass = 1; pass <= max_passes; ++pass) {
        const unsigned* cur = (pass & 1) ? list_a : list_b;
        unsigned* nxt = (pass & 1) ? list_b : list_a;
        unsigned* n_next = &ctl->n_list[pass + 1];
        // rounds are uniform over the block (barriers inside)
        for (unsigned e0 = blockIdx.x * blockDim.x; e0 < n; e0 += stride) {
            if (threadIdx.x == 0) qn = 0u;
            __syncthreads();
            const unsigned e = e0 + threadIdx.x;
            const unsigned i0 = e < n ? cur[e] : 0u;
            bool todo = e < n;
            if (todo && pass > 1) atomicAnd(&queued[i0 >> 5], ~(1u << (i0 & 31)));   // off the list: may be listed again
            if (todo && xi[i0] != kXiMasked) todo = false;
            if (todo) {
                const int x = (int)(i0 % (unsigned)nx), y = (int)((i0 / (unsigned)nx) % (unsigned)ny), z = (int)(i0 / ((unsigned)nx * (unsigned)ny));
                const float s0 = __ldg(cbct + i0);
                // offsets -W..W per axis; a neighbour outside the volume has its address clamped and `in` false
                const int W = rt;
                float dmin = FLT_MAX;
                for (int dz = -W; dz <= W; ++dz) {
                    for (int dy = -W; dy <= W; ++dy) {
                        const int c = z + dz, b = y + dy;
                        const bool in_zy = c >= 0 && c < nz && b >= 0 && b < ny;
                        const size_t row = ((size_t)min(max(c, 0), nz - 1) * ny + min(max(b, 0), ny - 1)) * nx;
                        for (int dx = -W; dx <= W; ++dx) {
                            const int a = x + dx;
                            const bool in = in_zy && a >= 0 && a < nx;
                            const size_t j = row + min(max(a, 0), nx - 1);
                            const unsigned char st = xi[j];
                            const float d = __ldg(cbct + j) - s0;
                            if (in && st < pass) dmin = fminf(dmin, d * d);
                        }
                    }
                }
                if (dmin < FLT_MAX) {
                    float sw = 0.f, sa = 0.f, sb = 0.f;
                    for (int dz = -W; dz <= W; ++dz) {
                        for (int dy = -W; dy <= W; ++dy) {
                            const int c = z + dz, b = y + dy;
                            const bool in_zy = c >= 0 && c < nz && b >= 0 && b < ny;
                            const size_t row = ((size_t)min(max(c, 0), nz - 1) * ny + min(max(b, 0), ny - 1)) * nx;
                            for (int dx = -W; dx <= W; ++dx) {
                                const int a = x + dx;
                                const bool in = in_zy && a >= 0 && a < nx;
                                const size_t j = row + min(max(a, 0), nx - 1);
                                const unsigned char st = xi[j];
                                const float cv = __ldg(cbct + j), av = A[j], bv = B[j];   // unused when not available
                                if (!in) continue;
                                if (st >= pass) {
                                    // an unfilled voxel of T: it can be filled in the next pass, from this one
                                    const unsigned w = (unsigned)j;
                                    if (st == kXiMasked && w != i0 && pass < max_passes) {
                                        const unsigned bit = 1u << (w & 31);
                                        // the plain read spares most of the atomics (a stale 0 only costs one)
                                        if (!(*reinterpret_cast<volatile unsigned*>(&queued[w >> 5]) & bit) &&
                                            !(atomicOr(&queued[w >> 5], bit) & bit)) {
                                            const unsigned pos = atomicAdd(&qn, 1u);
                                            if (pos < kQ) q[pos] = w;
                                            else nxt[atomicAdd(n_next, 1u)] = w;     // block queue full: straight to the list
                                        }
                                    }
                                    continue;
                                }
                                const float d = cv - s0;
                                const float wgt = __expf(-(d * d - dmin) * inv_h2);    // Eq. (10)
                                sw += wgt;
                                sa = fmaf(wgt, av, sa);
                                sb = fmaf(wgt, bv, sb);
                            }
                        }
                    }
                    A[i0] = sa / sw;                                                   // Eqs. (8), (9)
                    B[i0] = sb / sw;
                    xi[i0] = (unsigned char)pass;
                }
            }
            __syncthreads();
            const unsigned cnt = qn < kQ ? qn : kQ;
            if (threadIdx.x == 0 && cnt) qbase = atomicAdd(n_next, cnt);
            __syncthreads();
            for (unsigned k = threadIdx.x; k < cnt; k += blockDim.x) nxt[qbase + k] = q[k];
            __syncthreads();
        }
        grid.sync();
        n = *reinterpret_cast<volatile unsigned*>(n_next);
        if (n == 0u) break;                               // nothing left, or a pass that filled nothing
    }
}

static __global__ void k_fill_reset(MaskCtl* ctl, IterCtl ictl) {
    if (iter_skipped(ictl)) return;
    ctl->remaining = 0u; ctl->filled = 0u; ctl->prev_filled = 0u; ctl->ticket = 0u;
    for (int p = 0; p < 257; ++p) ctl->n_list[p] = 0u;
}

// ---------------------------------------------------------------- I'_s = a I_s + b and Fig. 9 (e), (f)
// out may be NULL (diagnostics only).  diag (may be NULL): [0] += sum a, [1] += sum b of this iteration, through block
// partials added in block order by the last block (deterministic); slot = where the two averages are filed.
static __global__ void __launch_bounds__(256)
k_apply_ab(const float* __restrict__ cbct, const float* __restrict__ A, const float* __restrict__ B,
           float* __restrict__ out, size_t N, double* __restrict__ partial, MaskCtl* ctl, double* __restrict__ mean_a,
           double* __restrict__ mean_b, int slot, IterCtl ictl) {
    if (iter_skipped(ictl)) return;
    double sa = 0.0, sb = 0.0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
        const float a = A[i], b = B[i];
        if (out) out[i] = fmaf(a, __ldg(cbct + i), b);
        sa += (double)a; sb += (double)b;
    }
    if (!mean_a) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { sa += __shfl_xor_sync(0xffffffffu, sa, o); sb += __shfl_xor_sync(0xffffffffu, sb, o); }
    __shared__ double sh[2][8];
    __shared__ bool last;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][warp] = sa; sh[1][warp] = sb; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double ta = 0.0, tb = 0.0;
        for (int w = 0; w < 8; ++w) { ta += sh[0][w]; tb += sh[1][w]; }
        partial[2 * blockIdx.x] = ta; partial[2 * blockIdx.x + 1] = tb;
        __threadfence();
        last = atomicAdd(&ctl->ticket2, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (last && threadIdx.x == 0) {
        __threadfence();
        double ta = 0.0, tb = 0.0;
        for (unsigned k = 0; k < gridDim.x; ++k) { ta += partial[2 * k]; tb += partial[2 * k + 1]; }
        mean_a[slot] = ta / (double)N;
        mean_b[slot] = tb / (double)N;
        ctl->ticket2 = 0u;
    }
}

}  // namespace disc
