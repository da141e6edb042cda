// arranger.cuh -- the split arranger (steps a-5..a-7 of DESIGN.md): stand-alone per-cell
// histogram, and the destination-driven stable scatter for a state that was grouped by cell
// at the last arrange and has moved by at most w_acc cells since.
#pragma once
#include "pic_device.cuh"

namespace pic {

// ---- a-5: per-cell histogram of the live particles (warp-aggregated atomics) -------------
constexpr int HIST_THREADS = 256;
constexpr int HIST_ITEMS = 4;

__global__ void __launch_bounds__(HIST_THREADS) hist_kernel(const int *__restrict__ cell, int *__restrict__ count,
                                                            const DevState *st)
{
    const int n = st->n;
    const long long i0 = ((long long)blockIdx.x * HIST_THREADS + threadIdx.x) * HIST_ITEMS;
    int c[HIST_ITEMS];
    if (i0 + HIST_ITEMS <= n) {
        int4 t = *reinterpret_cast<const int4 *>(cell + i0);
        c[0] = t.x; c[1] = t.y; c[2] = t.z; c[3] = t.w;
    } else {
#pragma unroll
        for (int q = 0; q < HIST_ITEMS; ++q) c[q] = (i0 + q < n) ? cell[i0 + q] : -1;
    }
#pragma unroll
    for (int q = 0; q < HIST_ITEMS; ++q) warp_hist_add(count, c[q], c[q] >= 0);
}

// ---- initial-state validation (pic_create) -------------------------------------------------
// Checks 0 <= x < L, cell == min(floor(x*inv_dx), nc-1), all live; notes whether the state is grouped
// by cell; records the initial speed bound max |v|^2 (float, rounded up) in st->vmax2.
__global__ void validate_kernel(const double *__restrict__ x, const double *__restrict__ vx, const double *__restrict__ vy,
                                const double *__restrict__ vz, const int *__restrict__ cell, PushConst k, DevState *st)
{
    const int n = st->n;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = i < n;
    int err = 0;
    unsigned m = 0;
    if (valid) {
        const int c = cell[i];
        const double xv = x[i];
        if (c < 0 || c >= k.nc || !(xv >= 0.0) || !(xv < k.L)) err = ERR_BAD_INITIAL;
        else {
            int cf = (int)floor(__dmul_rn(xv, k.inv_dx));
            if (cf > k.nc - 1) cf = k.nc - 1;
            if (cf != c) err = ERR_BAD_INITIAL;
        }
        if (i > 0 && cell[i - 1] > c) err |= ERR_NOT_GROUPED;
        const double a = vx[i], b = vy[i], d = vz[i];
        m = __float_as_uint(__double2float_ru(a * a + b * b + d * d));
    }
    err = (int)__reduce_or_sync(FULL, (unsigned)err);
    m = __reduce_max_sync(FULL, m);
    if ((threadIdx.x & 31) == 0) {
        if (err) atomicOr(&st->status, err);
        if (m > *(volatile unsigned *)&st->vmax2) atomicMax(&st->vmax2, m);
    }
}

// ---- a-7: destination-driven stable scatter ---------------------------------------------------
// One warp per destination cell c.  Every particle now in cell c sat, at the last arrange, in a
// cell within w_acc of c (circularly for a periodic grid), i.e. in the source slot range given
// by the OLD offsets of those cells.  The warp walks that range in ascending slot order (so
// the order of equal keys is the source order: the sort is stable), picks the slots whose
// cell equals c by ballot, ranks them by popc, and copies the five fields to
// offset_new[c] + rank.  Writes are contiguous per cell; no atomics; bitwise deterministic.
struct ScatterArgs {
    const double *sx, *svx, *svy, *svz;
    const int *scell;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const int *off_old;   // nc+1, offsets of the source grouping
    const int *count_new; // nc
    const int *off_new;   // nc+1
    DevState *st;
    const int *only_if; // if not NULL: the kernel returns at once unless *only_if != 0
    int nc, periodic, w_limit;
    int general_follows; // the host has enqueued the general path behind this kernel (else declining is an error)
};

constexpr int SCATTER_THREADS = 256;

__device__ __forceinline__ int scatter_range(const ScatterArgs &a, int c, int base, int cnt, int found, int sa, int sb,
                                             int lane)
{
    // walk source slots [sa, sb) in 32-wide chunks aligned to 32 slots
    for (int i = (sa & ~31) + lane; (i - lane) < sb && found < cnt; i += 32) {
        int cc = (i >= sa && i < sb) ? __ldg(a.scell + i) : -2;
        unsigned m = __ballot_sync(FULL, cc == c);
        if (cc == c) {
            int d = base + found + __popc(m & ((1u << lane) - 1u));
            a.dx[d] = a.sx[i];
            a.dvx[d] = a.svx[i];
            a.dvy[d] = a.svy[i];
            a.dvz[d] = a.svz[i];
            a.dcell[d] = c;
        }
        found += __popc(m);
    }
    return found;
}

__global__ void __launch_bounds__(SCATTER_THREADS) scatter_fast_kernel(ScatterArgs a)
{
    if (a.only_if && !*a.only_if) return;
    const int W = a.st->w_acc;
    if (W > a.w_limit) {
        if (blockIdx.x == 0 && threadIdx.x == 0) {
            a.st->need_general = 1;
            // the host's displacement bound said this could not happen and nothing runs behind: never silent
            if (!a.general_follows) atomicOr(&a.st->status, ERR_ARRANGE_SKIPPED);
        }
        return;
    }
    const int lane = threadIdx.x & 31;
    const int warps_per_block = SCATTER_THREADS / 32;
    const long long nwarps = (long long)gridDim.x * warps_per_block;
    for (long long cw = (long long)blockIdx.x * warps_per_block + (threadIdx.x >> 5); cw < a.nc; cw += nwarps) {
        const int c = (int)cw;
        const int cnt = a.count_new[c];
        if (cnt == 0) continue;
        const int base = a.off_new[c];
        int lo = c - W, hi = c + W; // inclusive source-cell window
        int found = 0;
        if (!a.periodic || 2LL * W + 1 >= a.nc) {
            if (a.periodic) { lo = 0; hi = a.nc - 1; }
            lo = max(lo, 0); hi = min(hi, a.nc - 1);
            found = scatter_range(a, c, base, cnt, found, a.off_old[lo], a.off_old[hi + 1], lane);
        } else if (lo < 0) {
            // cells [0, hi] come first in slot order, then the wrapped cells [lo+nc, nc-1]
            found = scatter_range(a, c, base, cnt, found, 0, a.off_old[hi + 1], lane);
            found = scatter_range(a, c, base, cnt, found, a.off_old[lo + a.nc], a.off_old[a.nc], lane);
        } else if (hi >= a.nc) {
            found = scatter_range(a, c, base, cnt, found, 0, a.off_old[hi - a.nc + 1], lane);
            found = scatter_range(a, c, base, cnt, found, a.off_old[lo], a.off_old[a.nc], lane);
        } else {
            found = scatter_range(a, c, base, cnt, found, a.off_old[lo], a.off_old[hi + 1], lane);
        }
    }
}

} // namespace pic
