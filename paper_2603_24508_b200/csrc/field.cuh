// field.cuh -- the field solve on the device (PIC phase (iii): "the field solver, which computes
// the electric ... fields by solving ... Poisson's equations"; BIT1's "native Poisson solver ... and
// smoothing operators"; readings S23-S28 of DESIGN.md section 12):
//     rho --[1-2-1 binomial filter, `passes` times]--> rho_s --[(phi[j-1] - 2 phi[j] + phi[j+1])/dx^2 = -rho_s[j]]--> phi
//         --[E = -dphi/dx, centred; one-sided at walls]--> E on the nc+1 nodes, written where the mover gathers it.
//
// The tridiagonal system has constant coefficients, so the elimination is a DOUBLE PREFIX SUM, not a recurrence:
// with r[j] = dx^2 (rho_s[j] - mean), S[j] = sum_{k=1..j} r[k] and T[j] = sum_{m=1..j-1} S[m],
//     phi[j] = j*F - T[j],      F = T[nc] / nc          (phi[0] = phi[nc] = 0)
// (F is phi[1] - phi[0]; each further difference phi[j+1] - phi[j] drops by S[j]: that IS the difference equation).
// Both sums come out of ONE scan with the associative operator on segments (len, s, t):
//     (lenA, sA, tA) o (lenB, sB, tB) = (lenA + lenB, sA + sB, tA + tB + lenB*sA)
// where s = sum r over the segment and t = sum of the segment's own inclusive prefix sums.  Nothing here is a dense
// contraction and the whole problem is 8-24 MB, so it is a handful of small HBM/L2-bound kernels, all with a
// fixed summation tree (bitwise reproducible, no atomics on the data path):
//   field_smooth_kernel   one pass of the filter (ping-pong between two library-owned arrays)
//   field_sum_kernel      per tile: sum of rho_s over the tile's distinct nodes (periodic grids: the mean)
//   field_tile_kernel     per tile of 2048 nodes: the aggregate (s, t) of the tile
//   field_chain_kernel    one block: exclusive scan of the tile aggregates, F, and (periodic) the mean
//   field_phi_kernel      per tile: in-tile scan + tile prefix -> phi[j]; per-tile sum of phi (periodic gauge)
//   field_e_kernel        E from phi (zero-mean gauge applied on a periodic grid), max |E| for the host's
//                         displacement bound, optional copy of phi for the caller
// On a periodic grid rho is neutralised first (uniform background) and phi is returned with zero mean; the gauge
// phi[0] = 0 used in between satisfies node 0's equation by itself because the neutralised rho sums to zero.
#pragma once
#include <cooperative_groups.h>
#include "pic_device.cuh"

namespace pic {

constexpr int FLD_THREADS = 256;
constexpr int FLD_ITEMS = 8;
constexpr int FLD_TILE = FLD_THREADS * FLD_ITEMS; // nodes per tile
constexpr int FLD_MAX_TILES = 1 << 20;

static inline int fld_ntiles(int nc) { return (nc + 1 + FLD_TILE - 1) / FLD_TILE; }

struct FieldSeg { // aggregate of a segment of consecutive nodes
    double s, t;
    double len; // number of nodes, as a double (exact below 2^53)
};

__device__ __forceinline__ FieldSeg fld_combine(const FieldSeg &a, const FieldSeg &b)
{
    FieldSeg c;
    c.s = a.s + b.s;
    c.t = (a.t + b.t) + b.len * a.s;
    c.len = a.len + b.len;
    return c;
}

__device__ __forceinline__ FieldSeg fld_shfl_up(const FieldSeg &v, int o)
{
    FieldSeg r;
    r.s = __shfl_up_sync(FULL, v.s, o);
    r.t = __shfl_up_sync(FULL, v.t, o);
    r.len = __shfl_up_sync(FULL, v.len, o);
    return r;
}

struct FieldArgs {
    const double *rho; // nc+1, the (smoothed) charge density
    double *phi;       // nc+1, library scratch
    double *E;         // nc+1 (+pad), the sim's field array
    double *phi_out;   // optional caller copy of phi (nc+1) or NULL
    double *tile_s, *tile_t; // per tile aggregates, then exclusive prefixes
    double *tile_sum;  // per tile: sum of rho (periodic), later sum of phi
    double *tile_lo;   // per tile: low word of the double-double sum of rho
    double *scal;      // [0] mean of rho, [1] F, [2] mean of phi, [3] low word of the mean of rho
    unsigned long long *emax_bits; // max |E| as the bits of a non-negative double
    unsigned *ticket;  // two arrival counters (zero between launches): the last block of a reduction finishes it
    int nc, periodic, ntiles;
    double dx2, inv_dx;
    const int *frozen; // pic_cycle: set on the device when a fused step of the cycle declined -- E must keep the field
                       // that step was issued under until the host has redone it (NULL outside pic_cycle)
};

// one pass of the 1-2-1 filter (S27, S28): ((left + 2*centre) + right) * 0.25
__device__ __forceinline__ void field_smooth_block(const double *__restrict__ in, double *__restrict__ out, int nc, int periodic,
                                                   int vb)
{
    const int j = vb * FLD_THREADS + threadIdx.x;
    if (j > nc) return;
    double left, right, centre;
    if (periodic) {
        const int jj = j == nc ? 0 : j;
        left = in[jj == 0 ? nc - 1 : jj - 1];
        right = in[jj == nc - 1 ? 0 : jj + 1];
        centre = in[jj];
    } else {
        left = in[j == 0 ? 0 : j - 1];
        right = in[j == nc ? nc : j + 1];
        centre = in[j];
    }
    const double t = __dmul_rn(2.0, centre);
    out[j] = __dmul_rn(__dadd_rn(__dadd_rn(left, t), right), 0.25);
}

__global__ void __launch_bounds__(FLD_THREADS) field_smooth_kernel(const double *__restrict__ in, double *__restrict__ out, int nc,
                                                                   int periodic)
{
    field_smooth_block(in, out, nc, periodic, blockIdx.x);
}

// block-wide sum with a fixed tree (warp shuffles, then warp 0 over the warp sums)
__device__ __forceinline__ double fld_block_sum(double v, double *s_w)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) s_w[warp] = v;
    __syncthreads();
    double r = 0.0;
#pragma unroll
    for (int w = 0; w < FLD_THREADS / 32; ++w) r += s_w[w];
    return r;
}

// Double-double accumulation (error-free TwoSum, Knuth): the mean of rho that neutralises a periodic grid must be
// known far below one ulp, because an error d in it leaves a uniform charge d behind, i.e. a parabola d dx^2 nc^2/8
// in phi: at 10^6 nodes a plain binary64 mean (d ~ 1e-16 |mean|) would already cost ~1e-5 dx^2 |mean|.
struct FieldDD { double hi, lo; };

__device__ __forceinline__ FieldDD fld_dd_add(FieldDD a, double b)
{
    const double s = __dadd_rn(a.hi, b);
    const double bb = __dsub_rn(s, a.hi);
    const double e = __dadd_rn(__dsub_rn(a.hi, __dsub_rn(s, bb)), __dsub_rn(b, bb));
    return FieldDD{s, __dadd_rn(a.lo, e)};
}

__device__ __forceinline__ FieldDD fld_dd_add(FieldDD a, FieldDD b)
{
    FieldDD r = fld_dd_add(a, b.hi);
    r.lo = __dadd_rn(r.lo, b.lo);
    return r;
}

// per tile: double-double sum of rho over the distinct nodes 0..nc-1 (only needed on a periodic grid)
// (vb = the tile, nvb = number of tiles: blockIdx.x / gridDim.x of field_sum_kernel, or the virtual block of the
// one-kernel solve; the same holds for the other *_block functions below)
__device__ __forceinline__ void field_sum_block(const FieldArgs &a, int vb, int nvb)
{
    __shared__ FieldDD s_w[FLD_THREADS / 32];
    const int base = vb * FLD_TILE + threadIdx.x * FLD_ITEMS;
    FieldDD v{0.0, 0.0};
#pragma unroll
    for (int q = 0; q < FLD_ITEMS; ++q)
        if (base + q < a.nc) v = fld_dd_add(v, a.rho[base + q]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        FieldDD u;
        u.hi = __shfl_xor_sync(FULL, v.hi, o);
        u.lo = __shfl_xor_sync(FULL, v.lo, o);
        v = fld_dd_add(v, u); // both partners add the same two values: the result is the same in every lane to
                              // the last bit only up to the order of hi/lo; lane 0's value is the one used
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) s_w[warp] = v;
    __syncthreads();
    __shared__ int s_last;
    if (threadIdx.x == 0) {
        FieldDD r{0.0, 0.0};
        for (int w = 0; w < FLD_THREADS / 32; ++w) r = fld_dd_add(r, s_w[w]);
        a.tile_sum[vb] = r.hi;
        a.tile_lo[vb] = r.lo;
        __threadfence();
        s_last = atomicAdd(a.ticket, 1u) == (unsigned)nvb - 1u;
    }
    __syncthreads();
    if (s_last) { // the last tile to arrive adds the tile sums: every thread a fixed subset, then a fixed tree
        __threadfence();
        FieldDD sum{0.0, 0.0};
        for (int t = threadIdx.x; t < a.ntiles; t += FLD_THREADS)
            sum = fld_dd_add(sum, FieldDD{((volatile double *)a.tile_sum)[t], ((volatile double *)a.tile_lo)[t]});
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            FieldDD u;
            u.hi = __shfl_down_sync(FULL, sum.hi, o);
            u.lo = __shfl_down_sync(FULL, sum.lo, o);
            sum = fld_dd_add(sum, u);
        }
        __syncthreads();
        if (lane == 0) s_w[warp] = sum;
        __syncthreads();
        if (threadIdx.x == 0) {
            FieldDD tot{0.0, 0.0};
            for (int w = 0; w < FLD_THREADS / 32; ++w) tot = fld_dd_add(tot, s_w[w]);
            const double n = (double)a.nc;
            const double q = tot.hi / n;
            const double rem = __fma_rn(-q, n, tot.hi); // exact remainder of the division
            a.scal[0] = q;
            a.scal[3] = __dadd_rn(rem, tot.lo) / n;
            *a.ticket = 0u;
        }
    }
}

__global__ void __launch_bounds__(FLD_THREADS) field_sum_kernel(FieldArgs a) { field_sum_block(a, blockIdx.x, gridDim.x); }

// r[j] of the solve: dx^2 (rho[j] - mean) on the unknown nodes 1..nc-1, zero elsewhere; mean = mhi + mlo
__device__ __forceinline__ double fld_r(const FieldArgs &a, int j, double mhi, double mlo)
{
    return (j >= 1 && j <= a.nc - 1) ? a.dx2 * __dsub_rn(__dsub_rn(a.rho[j], mhi), mlo) : 0.0;
}

// The in-tile scan: thread-local over FLD_ITEMS nodes, then an ordered scan of the thread aggregates.
// Returns the exclusive prefix (segment before this thread's first node, inside the tile) and, via `total`
// (valid in every thread), the tile aggregate.
__device__ __forceinline__ FieldSeg fld_tile_scan(const double (&r)[FLD_ITEMS], FieldSeg *s_w, FieldSeg &total)
{
    FieldSeg me{0.0, 0.0, (double)FLD_ITEMS};
#pragma unroll
    for (int q = 0; q < FLD_ITEMS; ++q) {
        me.s += r[q];
        me.t += me.s;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    FieldSeg inc = me;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const FieldSeg up = fld_shfl_up(inc, o);
        if (lane >= o) inc = fld_combine(up, inc);
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    FieldSeg wpre{0.0, 0.0, 0.0};
    total = FieldSeg{0.0, 0.0, 0.0};
#pragma unroll
    for (int w = 0; w < FLD_THREADS / 32; ++w) {
        const FieldSeg v = s_w[w];
        if (w == warp) wpre = total;
        total = fld_combine(total, v);
    }
    FieldSeg ex = fld_shfl_up(inc, 1); // exclusive inside the warp
    if (lane == 0) ex = FieldSeg{0.0, 0.0, 0.0};
    return fld_combine(wpre, ex);
}

__device__ __forceinline__ void field_tile_block(const FieldArgs &a, int vb)
{
    __shared__ FieldSeg s_w[FLD_THREADS / 32];
    const FieldDD mean{a.scal[0], a.scal[3]}; // zero on a bounded grid; written by field_sum_kernel on a periodic one
    const int base = vb * FLD_TILE + threadIdx.x * FLD_ITEMS;
    double r[FLD_ITEMS];
#pragma unroll
    for (int q = 0; q < FLD_ITEMS; ++q) r[q] = fld_r(a, base + q, mean.hi, mean.lo);
    FieldSeg total;
    fld_tile_scan(r, s_w, total);
    if (threadIdx.x == 0) {
        a.tile_s[vb] = total.s;
        a.tile_t[vb] = total.t;
    }
}

__global__ void __launch_bounds__(FLD_THREADS) field_tile_kernel(FieldArgs a) { field_tile_block(a, blockIdx.x); }

// One block: exclusive scan of the tile aggregates in tile order (every tile is FLD_TILE nodes long), then F.
__device__ __forceinline__ void field_chain_block(const FieldArgs &a)
{
    __shared__ FieldSeg s_w[FLD_THREADS / 32];
    __shared__ FieldSeg s_carry;
    if (threadIdx.x == 0) s_carry = FieldSeg{0.0, 0.0, 0.0};
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int t0 = 0; t0 < a.ntiles; t0 += FLD_THREADS) {
        const int t = t0 + threadIdx.x;
        FieldSeg me{0.0, 0.0, 0.0};
        if (t < a.ntiles) me = FieldSeg{a.tile_s[t], a.tile_t[t], (double)FLD_TILE};
        FieldSeg inc = me;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const FieldSeg up = fld_shfl_up(inc, o);
            if (lane >= o) inc = fld_combine(up, inc);
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        FieldSeg wpre = s_carry, total = s_carry;
#pragma unroll
        for (int w = 0; w < FLD_THREADS / 32; ++w) {
            const FieldSeg v = s_w[w];
            if (w == warp) wpre = total;
            total = fld_combine(total, v);
        }
        FieldSeg ex = fld_shfl_up(inc, 1);
        if (lane == 0) ex = FieldSeg{0.0, 0.0, 0.0};
        const FieldSeg pre = fld_combine(wpre, ex); // everything before tile t
        if (t < a.ntiles) {
            a.tile_s[t] = pre.s;
            a.tile_t[t] = pre.t;
        }
        __syncthreads();
        if (threadIdx.x == 0) s_carry = total;
        __syncthreads();
    }
    // T[nc] = sum_{m=1..nc-1} S[m]: r is zero outside 1..nc-1, so the inclusive sums over nodes 0..nc-1 give it:
    // t over all tiles counts S[m] for m up to the padded end; remove the (constant) tail S[nc-1] * (#nodes >= nc).
    if (threadIdx.x == 0) {
        const FieldSeg all = s_carry;
        const double tail = (double)((long long)a.ntiles * FLD_TILE - a.nc); // nodes nc .. end of the last tile
        const double Tnc = all.t - tail * all.s;
        a.scal[1] = Tnc / (double)a.nc;
    }
}

__global__ void __launch_bounds__(FLD_THREADS) field_chain_kernel(FieldArgs a) { field_chain_block(a); }

// per tile: phi[j] = j*F - T[j], T[j] = sum of S over the nodes before j (exclusive); per-tile sum of phi
__device__ __forceinline__ void field_phi_block(const FieldArgs &a, int vb, int nvb)
{
    __shared__ FieldSeg s_w[FLD_THREADS / 32];
    __shared__ double s_sum[FLD_THREADS / 32];
    const double mhi = a.scal[0], mlo = a.scal[3], F = a.scal[1];
    const int base = vb * FLD_TILE + threadIdx.x * FLD_ITEMS;
    double r[FLD_ITEMS];
#pragma unroll
    for (int q = 0; q < FLD_ITEMS; ++q) r[q] = fld_r(a, base + q, mhi, mlo);
    FieldSeg total;
    const FieldSeg ex = fld_tile_scan(r, s_w, total);
    const FieldSeg tpre{a.tile_s[vb], a.tile_t[vb], (double)vb * (double)FLD_TILE};
    const FieldSeg pre = fld_combine(tpre, ex); // all nodes before `base`: pre.s = S[base-1], pre.t = sum_{m<base} S[m]
    double S = pre.s, T = pre.t, psum = 0.0;
#pragma unroll
    for (int q = 0; q < FLD_ITEMS; ++q) {
        const int j = base + q;
        // here S = S[j-1], T = T[j] = sum_{m<=j-1} S[m]
        if (j <= a.nc) {
            const double p = (j == 0 || j == a.nc) ? 0.0 : (double)j * F - T;
            a.phi[j] = p;
            if (j < a.nc) psum += p;
        }
        S += r[q];
        T += S;
    }
    psum = fld_block_sum(psum, s_sum);
    __shared__ int s_last;
    if (threadIdx.x == 0) {
        a.tile_sum[vb] = psum;
        __threadfence();
        s_last = atomicAdd(a.ticket + 1, 1u) == (unsigned)nvb - 1u;
    }
    __syncthreads();
    if (s_last) { // last tile: the mean of phi (the gauge of a periodic grid), by a fixed tree over the tile sums
        __threadfence();
        double sum = 0.0;
        if (a.periodic)
            for (int t = threadIdx.x; t < a.ntiles; t += FLD_THREADS) sum += ((volatile double *)a.tile_sum)[t];
        sum = fld_block_sum(sum, s_sum);
        if (threadIdx.x == 0) {
            a.scal[2] = sum / (double)a.nc;
            a.ticket[1] = 0u;
        }
    }
}

__global__ void __launch_bounds__(FLD_THREADS) field_phi_kernel(FieldArgs a) { field_phi_block(a, blockIdx.x, gridDim.x); }

// E from phi (S26), gauge shift on a periodic grid (S25), max |E|, optional copy of phi
__device__ __forceinline__ void field_e_block(const FieldArgs &a, int vb)
{
    __shared__ unsigned long long s_max;
    if (threadIdx.x == 0) s_max = 0ull;
    __syncthreads();
    if (a.frozen && *(volatile const int *)a.frozen) return; // block-uniform
    const double pm = a.scal[2]; // zero on a bounded grid
    const int nc = a.nc;
    const int j = vb * FLD_THREADS + threadIdx.x;
    double e = 0.0;
    if (j <= nc) {
        const double mh = -0.5 * a.inv_dx, m1 = -a.inv_dx;
        double p;
        if (a.periodic) {
            const int jj = j == nc ? 0 : j;
            const double pr = __dsub_rn(a.phi[jj == nc - 1 ? 0 : jj + 1], pm), pl = __dsub_rn(a.phi[jj == 0 ? nc - 1 : jj - 1], pm);
            e = __dmul_rn(__dsub_rn(pr, pl), mh);
            p = __dsub_rn(a.phi[jj], pm);
        } else {
            if (j == 0) e = __dmul_rn(__dsub_rn(a.phi[1], a.phi[0]), m1);
            else if (j == nc) e = __dmul_rn(__dsub_rn(a.phi[nc], a.phi[nc - 1]), m1);
            else e = __dmul_rn(__dsub_rn(a.phi[j + 1], a.phi[j - 1]), mh);
            p = a.phi[j];
        }
        a.E[j] = e;
        if (a.phi_out) a.phi_out[j] = p;
    }
    unsigned long long b = (unsigned long long)__double_as_longlong(fabs(e)); // non-negative doubles order like their bits
    if (!(fabs(e) <= 1.79769313486231570e308)) b = 0x7ff0000000000000ull;      // NaN / inf: the bound becomes +inf
    b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, 16));
    b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, 8));
    b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, 4));
    b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, 2));
    b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, 1));
    if ((threadIdx.x & 31) == 0 && b) atomicMax(&s_max, b);
    __syncthreads();
    if (threadIdx.x == 0 && s_max > *(volatile unsigned long long *)a.emax_bits) atomicMax(a.emax_bits, s_max);
}

__global__ void __launch_bounds__(FLD_THREADS) field_e_kernel(FieldArgs a) { field_e_block(a, blockIdx.x); }

// The whole solve as ONE cooperative kernel: the phases above, run by a grid of resident blocks that walk the virtual
// blocks of each phase and meet at a grid-wide barrier between phases.  The data is 0.5 - 24 MB and every phase a few
// microseconds: as six or seven launches the solve is launch latency (35 us at 65 K nodes of which 24 us are kernels).
// Same block-level code, same fixed summation trees, same tickets: bit-identical to the separate kernels.
// rho_in: the charge density as deposited; f0 / f1: the filter's ping-pong arrays; a.rho is set here to whichever array
// holds the filtered density.  emax_bits is cleared here (the separate-kernel path uses a memset).
__global__ void __launch_bounds__(FLD_THREADS) field_solve_kernel(FieldArgs a, const double *rho_in, double *f0, double *f1, int passes)
{
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const int nc = a.nc;
    const int nblk = (nc + 1 + FLD_THREADS - 1) / FLD_THREADS;
    const int G = (int)gridDim.x;
    if (blockIdx.x == 0 && threadIdx.x == 0) *a.emax_bits = 0ull;
    const double *cur = rho_in;
    for (int p = 0; p < passes; ++p) {
        double *out = (p & 1) ? f1 : f0;
        for (int vb = blockIdx.x; vb < nblk; vb += G) field_smooth_block(cur, out, nc, a.periodic, vb);
        grid.sync();
        cur = out;
    }
    a.rho = cur;
    if (a.periodic) {
        for (int vb = blockIdx.x; vb < a.ntiles; vb += G) {
            field_sum_block(a, vb, a.ntiles);
            __syncthreads(); // the block's shared arrays are reused by its next virtual block
        }
        grid.sync();
    }
    for (int vb = blockIdx.x; vb < a.ntiles; vb += G) {
        field_tile_block(a, vb);
        __syncthreads();
    }
    grid.sync();
    if (blockIdx.x == 0) field_chain_block(a);
    grid.sync();
    for (int vb = blockIdx.x; vb < a.ntiles; vb += G) {
        field_phi_block(a, vb, a.ntiles);
        __syncthreads();
    }
    grid.sync();
    for (int vb = blockIdx.x; vb < nblk; vb += G) {
        field_e_block(a, vb);
        __syncthreads();
    }
}

// max |E| of a field array handed over on the device (pic_set_field_device)
__global__ void __launch_bounds__(FLD_THREADS) field_emax_kernel(const double *__restrict__ E, int nc, unsigned long long *emax_bits)
{
    __shared__ unsigned long long s_max;
    if (threadIdx.x == 0) s_max = 0ull;
    __syncthreads();
    const int j = blockIdx.x * FLD_THREADS + threadIdx.x;
    const double e = j <= nc ? fabs(E[j]) : 0.0;
    unsigned long long b = (unsigned long long)__double_as_longlong(e);
    if (!(e <= 1.79769313486231570e308)) b = 0x7ff0000000000000ull;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) b = max(b, (unsigned long long)__shfl_xor_sync(FULL, b, o));
    if ((threadIdx.x & 31) == 0 && b) atomicMax(&s_max, b);
    __syncthreads();
    if (threadIdx.x == 0 && s_max > *(volatile unsigned long long *)emax_bits) atomicMax(emax_bits, s_max);
}

} // namespace pic
