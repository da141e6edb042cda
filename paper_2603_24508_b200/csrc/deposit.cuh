// deposit.cuh -- charge deposition on the arranged state (PIC phase (ii); SURVEY.md
// section 8(f) rank 1): linear (cloud-in-cell) weights, the transpose of the
// mover's gather.  Because the particles of cell c occupy the slots [offset[c], offset[c+1]) the
// scatter-add becomes a segmented reduction: half a warp (or a warp) per cell sums (1-w) and w over its particles
// (lane-strided partial sums, then a fixed shuffle tree: no atomics, bitwise deterministic), and one
// thread per node adds the two cells that touch it.  8 B read per particle.
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int DEP_THREADS = 256;

struct DepositArgs {
    const double *x;
    const int *off;  // nc+1 offsets of the arranged state
    double2 *cs;     // per cell: {sum (1-w), sum w}
    int nc;
    double inv_dx;
};

// LPC lanes per cell (16: half a warp; 32 for very large cells): the lanes stride
// over the cell's particles with eight loads in flight each (8*LPC particles per round trip), then a fixed
// shuffle tree inside the lane group.
template <int LPC>
__global__ void __launch_bounds__(DEP_THREADS) deposit_cell_kernel(DepositArgs a)
{
    const int sub = threadIdx.x & (LPC - 1);
    const long long c = ((long long)blockIdx.x * DEP_THREADS + threadIdx.x) / LPC;
    const bool live = c < a.nc;
    const int s0 = live ? a.off[c] : 0, s1 = live ? a.off[c + 1] : 0;
    const double cf = (double)c; // = floor(x*inv_dx), clamped to nc-1, for every particle of the cell (invariant)
    double a0 = 0.0, a1 = 0.0;
    for (int i = s0 + sub; i < s1; i += 8 * LPC) {
        double xv[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) xv[q] = i + LPC * q < s1 ? a.x[i + LPC * q] : 0.0;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            if (i + LPC * q < s1) {
                const double w = __dsub_rn(__dmul_rn(xv[q], a.inv_dx), cf);
                a0 += 1.0 - w;
                a1 += w;
            }
        }
    }
#pragma unroll
    for (int o = LPC / 2; o > 0; o >>= 1) {
        a0 += __shfl_xor_sync(FULL, a0, o);
        a1 += __shfl_xor_sync(FULL, a1, o);
    }
    if (live && sub == 0) a.cs[c] = make_double2(a0, a1);
}

// rho[j] = weight * (sum (1-w) over cell j + sum w over cell j-1); nodes 0 and nc of a periodic grid are one
// point and carry the same sum.  accumulate: add to rho instead of overwriting it (several species).
__global__ void deposit_node_kernel(const double2 *__restrict__ cs, int nc, int periodic, double weight, int accumulate,
                                    double *__restrict__ rho)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > nc) return;
    double v;
    if (periodic && (j == 0 || j == nc)) v = cs[0].x + cs[nc - 1].y;
    else v = (j < nc ? cs[j].x : 0.0) + (j > 0 ? cs[j - 1].y : 0.0);
    const double out = __dmul_rn(v, weight);
    rho[j] = accumulate ? rho[j] + out : out;
}

} // namespace pic
