// scan.cuh -- device-wide exclusive prefix sum of int32 counts (step a-6 of DESIGN.md) as a
// single-pass chained scan with decoupled look-back: each tile publishes its aggregate, then
// its inclusive prefix, in one 64-bit word (flag << 32 | value); tiles are handed out by an
// atomic ticket so that a waiting tile's predecessors are always already running.
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 16;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

// Scratch: tile_state[ntiles] 64-bit words + one ticket word, all zero before the launch.
static inline size_t scan_scratch_words(long long m) { return (size_t)((m + SCAN_TILE - 1) / SCAN_TILE) + 1; }

struct ScanFold {      // optional bookkeeping done by tile 0 / the last tile for the arranger
    DevState *st;      // may be NULL
    int reset;         // fold step_max into w_acc starting from 0 (an arrange ran before this step)
    int set_n;         // store the grand total into st->n
    int set_vmax;      // a mover step ran just before: commit its speed bound (vmax2 = vmax2_next)
    const int *guard;  // if not NULL: return at once unless *guard != 0
};

// out[i] = sum_{k<i} in[k] for i in [0, m]; out has m+1 elements (out[m] = total).
__global__ void __launch_bounds__(SCAN_THREADS) scan_exclusive_kernel(const int *in, int *out,
                                                                      int m, unsigned long long *tile_state,
                                                                      ScanFold fold)
{
    if (fold.guard && !*fold.guard) return;
    __shared__ int s_tile;
    __shared__ int s_warp[SCAN_THREADS / 32];
    __shared__ int s_prefix;
    const int ntiles = (m + SCAN_TILE - 1) / SCAN_TILE;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(tile_state + ntiles);
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(ticket, 1u);
    __syncthreads();
    const int tile = s_tile;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    if (tile == 0 && threadIdx.x == 0 && fold.st) {
        int w = (fold.reset ? 0 : fold.st->w_acc) + fold.st->step_max;
        fold.st->w_acc = w > W_UNKNOWN ? W_UNKNOWN : w;
        fold.st->step_max = 0;
        fold.st->need_general = 0;
        fold.st->used_general = 0;
        fold.st->tile_declined = 0;
        if (fold.set_vmax) {
            fold.st->vmax2 = fold.st->vmax2_next;
            fold.st->vmax2_next = 0;
        }
    }

    const long long base = (long long)tile * SCAN_TILE + (long long)threadIdx.x * SCAN_ITEMS;
    int v[SCAN_ITEMS];
    if (base + SCAN_ITEMS <= m) {
        const int4 *p = reinterpret_cast<const int4 *>(in + base);
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS / 4; ++q) {
            int4 t = p[q];
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; ++q) v[q] = (base + q < m) ? in[base + q] : 0;
    }
    int tsum = 0;
#pragma unroll
    for (int q = 0; q < SCAN_ITEMS; ++q) tsum += v[q];

    // block-wide exclusive scan of the thread sums
    int incl = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int wpre = 0, total = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        int t = s_warp[w];
        if (w < warp) wpre += t;
        total += t;
    }
    int excl = wpre + incl - tsum;

    // publish and look back (warp 0)
    if (warp == 0) {
        volatile unsigned long long *ts = tile_state;
        if (lane == 0)
            ts[tile] = ((unsigned long long)(tile == 0 ? 2u : 1u) << 32) | (unsigned int)total;
        int prefix = 0;
        int idx = tile - 1;
        while (idx >= 0) {
            int my = idx - lane;
            unsigned long long w;
            unsigned flag;
            do {
                w = my >= 0 ? ts[my] : (2ull << 32);
                flag = (unsigned)(w >> 32);
            } while (__any_sync(FULL, flag == 0));
            unsigned incl_mask = __ballot_sync(FULL, flag == 2);
            int val = (int)(unsigned)w;
            if (incl_mask) {
                int first = __ffs(incl_mask) - 1; // nearest predecessor holding an inclusive prefix
                int contrib = (lane <= first) ? val : 0;
                prefix += __reduce_add_sync(FULL, contrib);
                break;
            }
            prefix += __reduce_add_sync(FULL, val);
            idx -= 32;
        }
        if (lane == 0) {
            if (tile > 0) ts[tile] = (2ull << 32) | (unsigned int)(prefix + total);
            s_prefix = prefix;
        }
    }
    __syncthreads();
    int run = s_prefix + excl;
    if (base + SCAN_ITEMS <= m) {
        int4 *p = reinterpret_cast<int4 *>(out + base);
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS / 4; ++q) {
            int4 t;
            t.x = run; run += v[4 * q];
            t.y = run; run += v[4 * q + 1];
            t.z = run; run += v[4 * q + 2];
            t.w = run; run += v[4 * q + 3];
            p[q] = t;
        }
    } else {
#pragma unroll
        for (int q = 0; q < SCAN_ITEMS; ++q) {
            if (base + q < m) out[base + q] = run;
            run += v[q];
        }
    }
    if (tile == ntiles - 1 && threadIdx.x == 0) {
        int grand = s_prefix + total;
        out[m] = grand;
        if (fold.st && fold.set_n) {
            fold.st->n = grand;
            fold.st->wall_arr = fold.st->wall[0] + fold.st->wall[1]; // the mover of this step has finished: stream order
        }
    }
}

} // namespace pic
