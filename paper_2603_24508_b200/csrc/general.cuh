// general.cuh -- the general arranger path (any input order, any displacement): a stable LSD
// radix sort (8-bit digits) of (cell, slot) pairs followed by a gather of the five fields.
// Correct for every input; runs only when scatter_fast_kernel has declined (state not grouped
// by cell, or displacement bound above FAST_W_LIMIT).  Every kernel is launched unconditionally
// with a small persistent grid and returns at once unless DevState::need_general is set, so the
// usual path pays a few empty launches and no host round trip.
#pragma once
#include "pic_device.cuh"
#include "scan.cuh"

namespace pic {

constexpr int FAST_W_LIMIT = 96; // largest displacement bound (cells) the fast scatter accepts
constexpr int GEN_THREADS = 256;
constexpr int GEN_ITEMS = 8;
constexpr int GEN_TILE = GEN_THREADS * GEN_ITEMS;
constexpr int GEN_RADIX = 256;

static inline long long gen_ntiles(long long n) { return (n + GEN_TILE - 1) / GEN_TILE; }
static inline long long general_scan_elems(long long capacity) { return GEN_RADIX * gen_ntiles(capacity) + 1; }
static inline size_t gen_align(size_t b) { return (b + 255) & ~(size_t)255; }

static inline size_t general_workspace_bytes(long long capacity)
{
    size_t cap = (size_t)capacity;
    return 4 * gen_align(4 * cap) + gen_align(4 * (size_t)general_scan_elems(capacity)) + 256;
}

struct GeneralArgs {
    const double *sx, *svx, *svy, *svz;
    const int *scell;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const int *off_old;
    DevState *st;
    int nc;
    long long n_ub;
    void *ws;
    size_t ws_bytes;
    unsigned long long *scan_scratch;
};

__global__ void gen_fail_kernel(DevState *st)
{
    if (st->need_general) atomicOr(&st->status, ERR_NEED_WORKSPACE);
}

// pairs: key = cell (dead -> nc, sorts last), val = source slot
__global__ void __launch_bounds__(GEN_THREADS) gen_init_kernel(const int *__restrict__ cell, int *__restrict__ key,
                                                               int *__restrict__ val, int nc, const DevState *st, const int *n_src)
{
    if (!st->need_general) return;
    const int n = *n_src;
    for (long long i = (long long)blockIdx.x * GEN_THREADS + threadIdx.x; i < n; i += (long long)gridDim.x * GEN_THREADS) {
        int c = cell[i];
        key[i] = c >= 0 ? c : nc;
        val[i] = (int)i;
    }
}

// per-tile digit histogram, stored digit-major: hist[digit * ntiles + tile]
__global__ void __launch_bounds__(GEN_THREADS) gen_hist_kernel(const int *__restrict__ key, int *__restrict__ hist,
                                                               int shift, int ntiles, const DevState *st, const int *n_src)
{
    if (!st->need_general) return;
    __shared__ int s_h[GEN_RADIX];
    const int n = *n_src;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        s_h[threadIdx.x] = 0;
        __syncthreads();
        long long base = (long long)tile * GEN_TILE;
#pragma unroll
        for (int r = 0; r < GEN_ITEMS; ++r) {
            long long i = base + r * GEN_THREADS + threadIdx.x;
            if (i < n) atomicAdd(&s_h[(key[i] >> shift) & (GEN_RADIX - 1)], 1);
        }
        __syncthreads();
        hist[(long long)threadIdx.x * ntiles + tile] = s_h[threadIdx.x];
        __syncthreads();
    }
}

// stable scatter of one digit pass.  Items are taken in rounds of 256 consecutive slots; in a
// round the rank of an item among equal digits is (items of earlier rounds) + (items of
// earlier warps in this round) + (earlier lanes of its warp, by match_any/popc).
__global__ void __launch_bounds__(GEN_THREADS) gen_scatter_kernel(const int *__restrict__ key_in, const int *__restrict__ val_in,
                                                                  int *__restrict__ key_out, int *__restrict__ val_out,
                                                                  const int *__restrict__ hist_scanned, int shift, int ntiles,
                                                                  const DevState *st, const int *n_src)
{
    if (!st->need_general) return;
    __shared__ int s_run[GEN_RADIX];                   // digit -> items already placed in this tile
    __shared__ int s_w[GEN_THREADS / 32][GEN_RADIX];   // per-warp digit counts of the round, then bases
    const int n = *n_src;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        s_run[threadIdx.x] = hist_scanned[(long long)threadIdx.x * ntiles + tile];
        long long base = (long long)tile * GEN_TILE;
        for (int r = 0; r < GEN_ITEMS; ++r) {
#pragma unroll
            for (int w = 0; w < GEN_THREADS / 32; ++w) s_w[w][threadIdx.x] = 0;
            __syncthreads();
            long long i = base + r * GEN_THREADS + threadIdx.x;
            bool valid = i < n;
            int k = 0, v = 0, dgt = 0, rank = 0;
            unsigned act = __ballot_sync(FULL, valid);
            if (valid) {
                k = key_in[i]; v = val_in[i];
                dgt = (k >> shift) & (GEN_RADIX - 1);
                unsigned m = __match_any_sync(act, dgt);
                rank = __popc(m & ((1u << lane) - 1u));
                if (rank == 0) s_w[warp][dgt] = __popc(m);
            }
            __syncthreads();
            {   // thread d: exclusive prefix over warps for digit d, advance the running base
                int run = s_run[threadIdx.x];
#pragma unroll
                for (int w = 0; w < GEN_THREADS / 32; ++w) {
                    int c = s_w[w][threadIdx.x];
                    s_w[w][threadIdx.x] = run;
                    run += c;
                }
                s_run[threadIdx.x] = run;
            }
            __syncthreads();
            if (valid) {
                int d = s_w[warp][dgt] + rank;
                key_out[d] = k;
                val_out[d] = v;
            }
            __syncthreads();
        }
    }
}

__global__ void __launch_bounds__(GEN_THREADS) gen_gather_kernel(GeneralArgs a, const int *__restrict__ key, const int *__restrict__ val)
{
    if (!a.st->need_general) return;
    const int n_live = a.st->n;
    if (blockIdx.x == 0 && threadIdx.x == 0) a.st->used_general = 1;
    for (long long d = (long long)blockIdx.x * GEN_THREADS + threadIdx.x; d < n_live; d += (long long)gridDim.x * GEN_THREADS) {
        int i = val[d];
        a.dx[d] = a.sx[i];
        a.dvx[d] = a.svx[i];
        a.dvy[d] = a.svy[i];
        a.dvz[d] = a.svz[i];
        a.dcell[d] = key[d];
    }
}

// Host side: enqueue the whole guarded general path.  Returns 0 or a pic_status.
static inline int general_arrange(const GeneralArgs &a, cudaStream_t stream, int sm_count, unsigned long long *launches)
{
    if (a.n_ub <= 0) return 0;
    const size_t cap_bytes = gen_align(4 * (size_t)a.n_ub);
    const long long ntiles = gen_ntiles(a.n_ub);
    const size_t hist_elems = (size_t)GEN_RADIX * ntiles + 1;
    const size_t need = 4 * cap_bytes + gen_align(4 * hist_elems);
    if (!a.ws || a.ws_bytes < need) {
        gen_fail_kernel<<<1, 1, 0, stream>>>(a.st);
        ++*launches;
        return cudaGetLastError() == cudaSuccess ? 0 : -3;
    }
    char *w = static_cast<char *>(a.ws);
    int *key[2] = {reinterpret_cast<int *>(w), reinterpret_cast<int *>(w + cap_bytes)};
    int *val[2] = {reinterpret_cast<int *>(w + 2 * cap_bytes), reinterpret_cast<int *>(w + 3 * cap_bytes)};
    int *hist = reinterpret_cast<int *>(w + 4 * cap_bytes);
    const int grid = sm_count * 4;
    const int *n_src = a.off_old + a.nc; // slots in use before this arrange
    gen_init_kernel<<<grid, GEN_THREADS, 0, stream>>>(a.scell, key[0], val[0], a.nc, a.st, n_src);
    ++*launches;
    int bits = 1;
    while ((1LL << bits) <= a.nc) ++bits; // keys are 0..nc
    int cur = 0;
    for (int shift = 0; shift < bits; shift += 8) {
        gen_hist_kernel<<<grid, GEN_THREADS, 0, stream>>>(key[cur], hist, shift, (int)ntiles, a.st, n_src);
        ++*launches;
        const int m = (int)(GEN_RADIX * ntiles);
        if (cudaMemsetAsync(a.scan_scratch, 0, scan_scratch_words(m) * sizeof(unsigned long long), stream) != cudaSuccess) return -3;
        ScanFold nofold{nullptr, 0, 0, 0, &a.st->need_general};
        scan_exclusive_kernel<<<(m + SCAN_TILE - 1) / SCAN_TILE, SCAN_THREADS, 0, stream>>>(hist, hist, m, a.scan_scratch, nofold);
        ++*launches;
        gen_scatter_kernel<<<grid, GEN_THREADS, 0, stream>>>(key[cur], val[cur], key[cur ^ 1], val[cur ^ 1], hist, shift,
                                                            (int)ntiles, a.st, n_src);
        ++*launches;
        cur ^= 1;
    }
    gen_gather_kernel<<<grid, GEN_THREADS, 0, stream>>>(a, key[cur], val[cur]);
    ++*launches;
    return cudaGetLastError() == cudaSuccess ? 0 : -3;
}

} // namespace pic
