// mover.cuh -- the stand-alone particle mover kernel (steps a-1..a-5 of DESIGN.md): one
// thread moves two neighbouring particles with 128-bit loads/stores of the fp64 SoA arrays.
// Used when a step is not followed by an arrange, or when the fused push+arrange kernel
// (fused.cuh) is switched off or has declined a step.
#pragma once
#include "pic_device.cuh"

namespace pic {

struct MoverArgs {
    double *x, *vx, *vy, *vz;
    int *cell;
    const double *E;  // nc+1 nodes
    int *count;       // per-cell histogram of the new cells (HIST only), pre-zeroed
    DevState *st;
    PushConst k;
};

constexpr int MOVER_THREADS = 256;

template <bool READ_CELL, bool HIST>
__global__ void __launch_bounds__(MOVER_THREADS) mover_kernel(MoverArgs a)
{
    __shared__ int s_max;
    __shared__ unsigned s_vmax;
    if (threadIdx.x == 0) { s_max = 0; s_vmax = 0; }
    __syncthreads();

    const int n = a.st->n;
    const int lane = threadIdx.x & 31;
    int dmax = 0, nleft = 0, nright = 0, bad = 0;
    float vm2 = 0.f; // upper bound of max |v'|^2 (feeds the next step's displacement bound)
    // one pair of neighbouring particles per thread and iteration (the grid covers the array in one iteration)
    const long long pairs = ((long long)n + 1) / 2;
    for (long long pb = (long long)blockIdx.x * MOVER_THREADS; pb < pairs; pb += (long long)gridDim.x * MOVER_THREADS) {
    const long long i0 = 2 * (pb + threadIdx.x);

    double x[2], vx[2], vy[2], vz[2];
    int c[2] = {-1, -1};
    bool have[2] = {i0 < n, i0 + 1 < n};
    if (have[1]) {
        double2 t;
        t = *reinterpret_cast<const double2 *>(a.x + i0);  x[0] = t.x;  x[1] = t.y;
        t = *reinterpret_cast<const double2 *>(a.vx + i0); vx[0] = t.x; vx[1] = t.y;
        t = *reinterpret_cast<const double2 *>(a.vy + i0); vy[0] = t.x; vy[1] = t.y;
        t = *reinterpret_cast<const double2 *>(a.vz + i0); vz[0] = t.x; vz[1] = t.y;
        if (READ_CELL) { int2 ci = *reinterpret_cast<const int2 *>(a.cell + i0); c[0] = ci.x; c[1] = ci.y; }
        else { c[0] = 0; c[1] = 0; }
    } else if (have[0]) {
        x[0] = a.x[i0]; vx[0] = a.vx[i0]; vy[0] = a.vy[i0]; vz[0] = a.vz[i0];
        c[0] = READ_CELL ? a.cell[i0] : 0;
        x[1] = vx[1] = vy[1] = vz[1] = 0.0;
    } else {
        x[0] = x[1] = vx[0] = vx[1] = vy[0] = vy[1] = vz[0] = vz[1] = 0.0;
    }

    int cn[2] = {-1, -1};
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        bool live = have[q] && c[q] >= 0;
        if (live) {
            double xs, jf; int j;
            if (gather_cell(a.k, x[q], xs, jf, j)) {
                double E0 = __ldg(a.E + j), E1 = __ldg(a.E + j + 1);
                PushOut o;
                push_core(a.k, x[q], vx[q], vy[q], vz[q], xs, jf, j, E0, E1, o);
                x[q] = o.x; vx[q] = o.vx; vy[q] = o.vy; vz[q] = o.vz;
                vm2 = fmaxf(vm2, __double2float_ru(o.vx * o.vx + o.vy * o.vy + o.vz * o.vz));
                cn[q] = o.cell;
                dmax = max(dmax, o.dcell);
                nleft += (o.wall == 1); nright += (o.wall == 2);
            } else {
                bad = 1;
                // left untouched as the oracle does; without a stored cell index to keep, flag it dead so that the
                // arrange behind this step stays self-consistent (it is dropped) while ERR_OUT_OF_DOMAIN is reported
                cn[q] = READ_CELL ? c[q] : -1;
                live = false;
            }
        }
        if (HIST) warp_hist_add(a.count, cn[q], live && cn[q] >= 0);
    }

    if (have[1]) {
        *reinterpret_cast<double2 *>(a.x + i0) = make_double2(x[0], x[1]);
        *reinterpret_cast<double2 *>(a.vx + i0) = make_double2(vx[0], vx[1]);
        *reinterpret_cast<double2 *>(a.vy + i0) = make_double2(vy[0], vy[1]);
        *reinterpret_cast<double2 *>(a.vz + i0) = make_double2(vz[0], vz[1]);
        *reinterpret_cast<int2 *>(a.cell + i0) = make_int2(cn[0], cn[1]);
    } else if (have[0]) {
        a.x[i0] = x[0]; a.vx[i0] = vx[0]; a.vy[i0] = vy[0]; a.vz[i0] = vz[0];
        a.cell[i0] = cn[0];
    }
    }

    // wall counters (ballot/popc: one atomic per warp that absorbed something), error flag,
    // displacement bound (one atomic per block, and only while it still raises the maximum)
    unsigned any = __ballot_sync(FULL, (nleft | nright | bad) != 0);
    if (any) {
        int l = __reduce_add_sync(FULL, nleft), r = __reduce_add_sync(FULL, nright);
        int b = __reduce_or_sync(FULL, (unsigned)bad);
        if (lane == 0) {
            if (l) atomicAdd(&a.st->wall[0], (unsigned long long)l);
            if (r) atomicAdd(&a.st->wall[1], (unsigned long long)r);
            if (b) atomicOr(&a.st->status, ERR_OUT_OF_DOMAIN);
        }
    }
    int wmax = __reduce_max_sync(FULL, dmax);
    if (lane == 0 && wmax > 0) atomicMax(&s_max, wmax);
    unsigned vmw = __reduce_max_sync(FULL, __float_as_uint(vm2));
    if (lane == 0 && vmw) atomicMax(&s_vmax, vmw);
    __syncthreads();
    if (threadIdx.x == 0) {
        if (s_max > *(volatile int *)&a.st->step_max) atomicMax(&a.st->step_max, s_max);
        if (s_vmax > *(volatile unsigned *)&a.st->vmax2_next) atomicMax(&a.st->vmax2_next, s_vmax);
    }
}

// End of a mover step that is not followed by an arrange: fold the step's displacement
// maximum into the bound since the last arrange (reset = an arrange ran just before this step).
__global__ void end_step_kernel(DevState *st, int reset)
{
    int w = (reset ? 0 : st->w_acc) + st->step_max;
    st->w_acc = w > W_UNKNOWN ? W_UNKNOWN : w;
    st->step_max = 0;
    st->vmax2 = st->vmax2_next;
    st->vmax2_next = 0;
}

} // namespace pic
