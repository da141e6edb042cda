// tilesort.cuh -- the split arranger's stable scatter (step a-7 of DESIGN.md) for a state that was
// grouped by cell at the last arrange and has moved by at most w_acc cells since: a counting sort whose
// ranks are built tile by tile, O(1) work per particle whatever the displacement.
//
//   tile_hist_kernel     per tile of TILE consecutive source slots: the window of destination cells it
//                        touches (circular on a periodic grid) and the per-cell counts inside the window
//   tile_base_kernel     per destination cell c: walk the tiles that can hold particles of c (those
//                        overlapping the source slots of cells c-W .. c+W, from the OLD offsets) in ascending
//                        order and turn their counts into first slots: off_new[c] + particles of c in earlier tiles
//   tile_scatter_kernel  per tile: rank every particle inside its (tile, cell) group in slot order
//                        (per-warp segments, __match_any_sync / popc, per-warp running counters) and copy
//                        its five fields to first slot + rank
// Equal keys keep their source order (earlier tile, earlier warp segment, earlier row, lower lane): the
// sort is stable; there are no atomics on global memory; the result is bitwise deterministic.
// A tile whose window exceeds TS_WIN cells (very sparse regions) declines the whole path
// (DevState::tile_declined); the destination-driven scatter_fast_kernel launched behind takes over.
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int TS_THREADS = 256;
constexpr int TS_WARPS = TS_THREADS / 32;
constexpr int TS_ROWS = 8;                           // rows of 32 slots per warp segment
constexpr int TS_TILE = TS_THREADS * TS_ROWS;        // 2048 source slots per tile
constexpr int TS_WIN = 1024;                         // destination cells per tile window

static inline long long ts_ntiles(long long n) { return (n + TS_TILE - 1) / TS_TILE; }
static inline size_t ts_workspace_bytes(long long capacity)
{
    const size_t nt = (size_t)ts_ntiles(capacity) + 1;
    return ((nt * sizeof(int2) + 255) & ~(size_t)255) + nt * TS_WIN * sizeof(int);
}

struct TileArgs {
    const double *sx, *svx, *svy, *svz;
    const int *scell;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const int *off_old; // nc+1 (off_old[nc] = slots in use)
    const int *off_new; // nc+1
    int2 *tinfo;        // per tile: {first cell of the window, cells in the window (0: no live particle, -1: declined)}
    int *thist;         // per tile TS_WIN entries: counts, then first slots
    DevState *st;
    int nc, periodic, w_limit;
    int general_follows; // the host has enqueued the general path behind (else declining is an error)
};

// bin of cell c in a window starting at cell cmin (circular on a periodic grid)
__device__ __forceinline__ int ts_bin(int c, int cmin, int nc, int periodic)
{
    int u = c - cmin;
    if (periodic) {
        if (u < 0) u += nc;
        else if (u >= nc) u -= nc;
    }
    return u;
}

__global__ void __launch_bounds__(TS_THREADS) tile_hist_kernel(TileArgs a)
{
    __shared__ int s_hist[TS_WIN];
    __shared__ int s_lo[TS_WARPS], s_hi[TS_WARPS], s_ref;
    const int n = a.off_old[a.nc];
    const int t = blockIdx.x;
    const long long base = (long long)t * TS_TILE;
    if (base >= n) {
        if (threadIdx.x == 0) a.tinfo[t] = make_int2(0, 0);
        return;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int c[TS_ROWS];
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r) {
        const long long i = base + r * TS_THREADS + threadIdx.x;
        c[r] = i < n ? a.scell[i] : -1;
    }
    // reference cell: the largest live cell index of the tile; cells are measured relative to it (circularly)
    if (threadIdx.x == 0) s_ref = -1;
    __syncthreads();
    {
        int cm = -1;
#pragma unroll
        for (int r = 0; r < TS_ROWS; ++r) cm = max(cm, c[r]);
        cm = __reduce_max_sync(FULL, cm);
        if (lane == 0 && cm >= 0) atomicMax(&s_ref, cm);
    }
    __syncthreads();
    if (s_ref < 0) { // no live particle in the tile
        if (threadIdx.x == 0) a.tinfo[t] = make_int2(0, 0);
        return;
    }
    const int ref = s_ref, half = a.nc >> 1;
    int lo = 0x7fffffff, hi = -0x7fffffff;
    int rel[TS_ROWS];
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r) {
        rel[r] = 0;
        if (c[r] >= 0) {
            int d = c[r] - ref;
            if (a.periodic) {
                if (d > half) d -= a.nc;
                else if (d < -half) d += a.nc;
            }
            rel[r] = d;
            lo = min(lo, d);
            hi = max(hi, d);
        }
    }
    lo = __reduce_min_sync(FULL, lo);
    hi = __reduce_max_sync(FULL, hi);
    if (lane == 0) { s_lo[warp] = lo; s_hi[warp] = hi; }
    __syncthreads();
    lo = 0x7fffffff; hi = -0x7fffffff;
    for (int w = 0; w < TS_WARPS; ++w) { lo = min(lo, s_lo[w]); hi = max(hi, s_hi[w]); }
    const int win = hi - lo + 1;
    if (win > TS_WIN || win > a.nc) {
        if (threadIdx.x == 0) {
            a.tinfo[t] = make_int2(0, -1);
            a.st->tile_declined = 1;
        }
        return;
    }
    for (int b = threadIdx.x; b < win; b += TS_THREADS) s_hist[b] = 0;
    __syncthreads();
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r)
        if (c[r] >= 0) atomicAdd(&s_hist[rel[r] - lo], 1);
    __syncthreads();
    int *h = a.thist + (size_t)t * TS_WIN;
    for (int b = threadIdx.x; b < win; b += TS_THREADS) h[b] = s_hist[b];
    if (threadIdx.x == 0) a.tinfo[t] = make_int2(ref + lo < 0 ? ref + lo + a.nc : ref + lo, win);
}

// One thread per destination cell: exclusive scan of the tiles' counts of that cell, in tile order.
__global__ void __launch_bounds__(256) tile_base_kernel(TileArgs a)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= a.nc) return;
    DevState *st = a.st;
    if (*(volatile int *)&st->tile_declined) return;
    const int W = st->w_acc;
    if (W > a.w_limit) { // the displacement bound is too large for a window: the general path must run
        if (c == 0) {
            st->need_general = 1;
            if (!a.general_follows) atomicOr(&st->status, ERR_ARRANGE_SKIPPED);
        }
        return;
    }
    const int nc = a.nc;
    // source slot ranges that can hold particles of c, in ascending slot order (as scatter_fast_kernel)
    int ra0, ra1, rb0 = 0, rb1 = 0;
    const int lo = c - W, hi = c + W;
    if (!a.periodic || 2LL * W + 1 >= nc) {
        const int l = a.periodic ? 0 : max(lo, 0), h = a.periodic ? nc - 1 : min(hi, nc - 1);
        ra0 = a.off_old[l]; ra1 = a.off_old[h + 1];
    } else if (lo < 0) {
        ra0 = 0; ra1 = a.off_old[hi + 1];
        rb0 = a.off_old[lo + nc]; rb1 = a.off_old[nc];
    } else if (hi >= nc) {
        ra0 = 0; ra1 = a.off_old[hi - nc + 1];
        rb0 = a.off_old[lo]; rb1 = a.off_old[nc];
    } else {
        ra0 = a.off_old[lo]; ra1 = a.off_old[hi + 1];
    }
    int run = a.off_new[c];
    int tnext = 0; // first tile not yet visited
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const int s0 = pass ? rb0 : ra0, s1 = pass ? rb1 : ra1;
        if (s1 <= s0) continue;
        const int t0 = max(s0 / TS_TILE, tnext), t1 = (s1 - 1) / TS_TILE;
        for (int t = t0; t <= t1; ++t) {
            const int2 info = a.tinfo[t];
            if (info.y <= 0) continue;
            const int u = ts_bin(c, info.x, nc, a.periodic);
            if ((unsigned)u < (unsigned)info.y) {
                int *h = a.thist + (size_t)t * TS_WIN + u;
                const int cnt = *h;
                *h = run;
                run += cnt;
            }
        }
        tnext = max(tnext, t1 + 1);
    }
}

// One block per tile; warp w owns the slots [w*256, w*256+256) of the tile, row by row.
__global__ void __launch_bounds__(TS_THREADS) tile_scatter_kernel(TileArgs a)
{
    extern __shared__ int ts_smem[]; // [TS_WARPS + 1][win]: per-warp counters, then the tile's first slots
    DevState *st = a.st;
    if (*(volatile int *)&st->tile_declined || *(volatile int *)&st->need_general) return;
    const int n = a.off_old[a.nc];
    const int t = blockIdx.x;
    const int2 info = a.tinfo[t];
    const int win = info.y, cmin = info.x;
    if (win <= 0) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    int *wc = ts_smem + warp * win;
    int *tb = ts_smem + TS_WARPS * win;
    for (int b = threadIdx.x; b < TS_WARPS * win; b += TS_THREADS) ts_smem[b] = 0;
    {
        const int *h = a.thist + (size_t)t * TS_WIN;
        for (int b = threadIdx.x; b < win; b += TS_THREADS) tb[b] = h[b];
    }
    __syncthreads();
    const long long base = (long long)t * TS_TILE + warp * (TS_ROWS * 32);
    int bin[TS_ROWS];
    // sweep A: per-warp counts of every window cell
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r) {
        const long long i = base + r * 32 + lane;
        const int c = i < n ? a.scell[i] : -1;
        bin[r] = c >= 0 ? ts_bin(c, cmin, a.nc, a.periodic) : -1;
        const unsigned live = __ballot_sync(FULL, bin[r] >= 0);
        if (bin[r] >= 0) {
            const unsigned m = __match_any_sync(live, bin[r]);
            if ((m & lt) == 0) wc[bin[r]] += __popc(m);
        }
        __syncwarp();
    }
    __syncthreads();
    // first slot of every (warp, cell) group: the tile's first slot of the cell + the earlier warps' counts
    for (int b = threadIdx.x; b < win; b += TS_THREADS) {
        int run = tb[b];
#pragma unroll
        for (int w = 0; w < TS_WARPS; ++w) {
            const int cnt = ts_smem[w * win + b];
            ts_smem[w * win + b] = run;
            run += cnt;
        }
    }
    __syncthreads();
    // sweep B: rank inside the group in slot order, copy.  The source fields of four rows are loaded ahead of
    // the ranking so that their latency overlaps it.
#pragma unroll
    for (int r0 = 0; r0 < TS_ROWS; r0 += 4) {
        double x[4], vx[4], vy[4], vz[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const long long i = base + (r0 + q) * 32 + lane;
            if (bin[r0 + q] >= 0) { x[q] = a.sx[i]; vx[q] = a.svx[i]; vy[q] = a.svy[i]; vz[q] = a.svz[i]; }
            else { x[q] = vx[q] = vy[q] = vz[q] = 0.0; }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int bq = bin[r0 + q];
            const unsigned live = __ballot_sync(FULL, bq >= 0);
            if (bq >= 0) {
                const unsigned m = __match_any_sync(live, bq);
                const int d = wc[bq] + __popc(m & lt);
                __syncwarp(live);
                if ((m & lt) == 0) wc[bq] += __popc(m);
                int c = cmin + bq;
                if (c >= a.nc) c -= a.nc;
                a.dx[d] = x[q];
                a.dvx[d] = vx[q];
                a.dvy[d] = vy[q];
                a.dvz[d] = vz[q];
                a.dcell[d] = c;
            }
            __syncwarp();
        }
    }
}

} // namespace pic
