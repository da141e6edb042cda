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
constexpr int TS_WIN = 512;                          // destination cells per tile window

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
        // four tiles at a time: their window descriptors, then their counts, are loaded independently of one another
        // (the walk is a latency chain otherwise: up to ~20 tiles per cell in the dense part of config 5)
        for (int tq = t0; tq <= t1; tq += 4) {
            int2 info[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) info[q] = tq + q <= t1 ? __ldg(a.tinfo + tq + q) : make_int2(0, 0);
            int *h[4];
            int cnt[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int u = info[q].y > 0 ? ts_bin(c, info[q].x, nc, a.periodic) : -1;
                h[q] = (unsigned)u < (unsigned)info[q].y ? a.thist + (size_t)(tq + q) * TS_WIN + u : nullptr;
                cnt[q] = h[q] ? *h[q] : 0;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (h[q]) *h[q] = run;
                run += cnt[q];
            }
        }
        tnext = max(tnext, t1 + 1);
    }
}

// Dynamic shared memory of tile_scatter_kernel: per-warp counters (16-bit: a warp segment has 256 slots, a tile 2048),
// the tile's first slot and first staging place per window cell, and the staging area in which the tile is put into
// DESTINATION order before it is written.  39 KB: five blocks per SM.
constexpr size_t TS_SMEM_WC = (size_t)TS_WARPS * TS_WIN * sizeof(unsigned short);
constexpr size_t TS_SMEM_TB = (size_t)TS_WIN * sizeof(int);
constexpr size_t TS_SMEM_LBASE = ((size_t)(TS_WIN + 1) * sizeof(unsigned short) + 15) & ~(size_t)15;
constexpr size_t TS_SMEM_BYTES = TS_SMEM_WC + TS_SMEM_TB + TS_SMEM_LBASE + (size_t)TS_TILE * (sizeof(int) + sizeof(unsigned short) + sizeof(double));

// One block per tile; warp w owns the slots [w*256, w*256+256) of the tile, row by row.
// Every particle gets its rank k among the tile's particles bound for the same cell (earlier warps' counts + rank in
// slot order inside the warp), hence its final slot d = (tile's first slot of the cell) + k and its place in the
// tile's own destination order lpos = (particles of the tile bound for lower cells) + k.  Field by field the tile is
// then staged in shared memory in that order and written out with consecutive threads on consecutive slots of a run:
// a tile that spreads over W cells writes W contiguous runs instead of 2048 scattered 8-byte stores (14.4 -> 8.2
// sectors per request at config 5).
__global__ void __launch_bounds__(TS_THREADS) tile_scatter_kernel(TileArgs a)
{
    extern __shared__ __align__(16) unsigned char ts_raw[];
    unsigned short *wc_all = reinterpret_cast<unsigned short *>(ts_raw);                              // [TS_WARPS][win]
    int *tb = reinterpret_cast<int *>(ts_raw + TS_SMEM_WC);                                           // [win] tile's first slot
    unsigned short *lbase = reinterpret_cast<unsigned short *>(ts_raw + TS_SMEM_WC + TS_SMEM_TB);     // [win + 1]
    double *stage = reinterpret_cast<double *>(ts_raw + TS_SMEM_WC + TS_SMEM_TB + TS_SMEM_LBASE);     // [TS_TILE] one field
    int *sdest = reinterpret_cast<int *>(stage + TS_TILE);                                            // [TS_TILE] final slot
    unsigned short *sbin = reinterpret_cast<unsigned short *>(sdest + TS_TILE);                       // [TS_TILE] window cell
    __shared__ int s_scan[TS_WARPS];
    DevState *st = a.st;
    if (*(volatile int *)&st->tile_declined || *(volatile int *)&st->need_general) return;
    const int n = a.off_old[a.nc];
    const int t = blockIdx.x;
    const int2 info = a.tinfo[t];
    const int win = info.y, cmin = info.x;
    if (win <= 0) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    unsigned short *wc = wc_all + warp * win;
    for (int b = threadIdx.x; b < TS_WARPS * win; b += TS_THREADS) wc_all[b] = 0;
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
            if ((m & lt) == 0) wc[bin[r]] = (unsigned short)(wc[bin[r]] + __popc(m));
        }
        __syncwarp();
    }
    __syncthreads();
    // per window cell: the warps' counts become their first ranks (exclusive over the warps), and the tile's count,
    // by a block-wide exclusive scan over the cells, the cell's first place in the staging order
    {
        constexpr int PER = TS_WIN / TS_THREADS; // window cells per thread, consecutive
        int cnt[PER], tsum = 0;
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            const int b = threadIdx.x * PER + q;
            int run = 0;
            if (b < win) {
#pragma unroll
                for (int w = 0; w < TS_WARPS; ++w) {
                    const int k = wc_all[w * win + b];
                    wc_all[w * win + b] = (unsigned short)run;
                    run += k;
                }
            }
            cnt[q] = run;
            tsum += run;
        }
        int incl = tsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int u = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) s_scan[warp] = incl;
        __syncthreads();
        int pre = incl - tsum;
        for (int w = 0; w < warp; ++w) pre += s_scan[w];
#pragma unroll
        for (int q = 0; q < PER; ++q) {
            const int b = threadIdx.x * PER + q;
            if (b <= win) lbase[b] = (unsigned short)pre;
            pre += cnt[q];
        }
        if (threadIdx.x == TS_THREADS - 1) lbase[TS_WIN] = (unsigned short)pre; // a full window ends behind the last thread's cells
    }
    __syncthreads();
    const int nlive = lbase[win];
    // sweep B: rank inside the (tile, cell) group in slot order -> final slot and staging place of every particle
    int lpos[TS_ROWS];
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r) {
        const int bq = bin[r];
        const unsigned live = __ballot_sync(FULL, bq >= 0);
        lpos[r] = -1;
        if (bq >= 0) {
            const unsigned m = __match_any_sync(live, bq);
            const int k = wc[bq] + __popc(m & lt);
            __syncwarp(live);
            if ((m & lt) == 0) wc[bq] = (unsigned short)(wc[bq] + __popc(m));
            const int lp = lbase[bq] + k;
            lpos[r] = lp;
            sdest[lp] = tb[bq] + k;
            sbin[lp] = (unsigned short)bq;
        }
        __syncwarp();
    }
    // the four fp64 fields, one after the other through the staging area; the cell index rides with the first
    const double *src[4] = {a.sx, a.svx, a.svy, a.svz};
    double *dst[4] = {a.dx, a.dvx, a.dvy, a.dvz};
    double v[TS_ROWS];
#pragma unroll
    for (int r = 0; r < TS_ROWS; ++r) v[r] = lpos[r] >= 0 ? src[0][base + r * 32 + lane] : 0.0;
#pragma unroll
    for (int f = 0; f < 4; ++f) {
        __syncthreads(); // sdest / sbin complete (f = 0); the previous field has left the staging area (f > 0)
#pragma unroll
        for (int r = 0; r < TS_ROWS; ++r)
            if (lpos[r] >= 0) stage[lpos[r]] = v[r];
        if (f < 3) { // the next field's loads fly while this one is written out
#pragma unroll
            for (int r = 0; r < TS_ROWS; ++r) v[r] = lpos[r] >= 0 ? src[f + 1][base + r * 32 + lane] : 0.0;
        }
        __syncthreads();
        for (int i = threadIdx.x; i < nlive; i += TS_THREADS) {
            const int g = sdest[i];
            dst[f][g] = stage[i];
            if (f == 0) {
                int c = cmin + (int)sbin[i];
                if (c >= a.nc) c -= a.nc;
                a.dcell[g] = c;
            }
        }
    }
}

} // namespace pic
