// pic_device.cuh -- device-side state, constants and the per-particle push shared by the
// mover kernels of libpic (sm_100a).  The arithmetic contract is DESIGN.md section 3: every
// floating-point step is one IEEE-754 binary64 round-to-nearest operation written with the
// __d*_rn intrinsics, which nvcc never contracts into FMA.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pic {

constexpr unsigned FULL = 0xffffffffu;

// deferred device-side error bits (DevState::status)
constexpr int ERR_OUT_OF_DOMAIN = 1;  // a live particle's gather cell fell outside [0, nc-1]
constexpr int ERR_NEED_WORKSPACE = 2; // general arranger needed but no / too small workspace
constexpr int ERR_BAD_INITIAL = 4;    // initial state violates cell == floor(x/dx), live, in range
constexpr int ERR_NOT_GROUPED = 8;    // (info) initial state is not grouped by cell
constexpr int ERR_ARRANGE_SKIPPED = 32; // the fast arranger declined on the device but the general path was not enqueued

constexpr int W_UNKNOWN = 1 << 29; // displacement bound of a state that is not grouped by cell

// Small per-species block in device memory, owned by the library.
struct DevState {
    int n;            // slots in use (live + flagged dead); = n_live right after an arrange
    int w_acc;        // bound on |cell - cell at last arrange| over all live particles
    int step_max;     // max |dcell| seen by the mover step in flight
    int status;       // ERR_* bits
    int need_general; // fast arranger declined (w_acc too large); the general path must run
    int used_general; // the last arrange ran the general path
    int fused_disabled; // sticky: a fused step has declined (fail_step says which); later fused launches exit at once
    unsigned long long wall[2];      // cumulative absorbed at x<0 / x>=L
    unsigned long long wall_pend[2]; // fused step in flight: absorbed, not yet committed
    unsigned long long wall_arr;     // wall[0] + wall[1] at the last arrange (n - absorbed since = live particles)
    unsigned vmax2, vmax2_next;      // float bits (rounded up) of max |v|^2: current state / step in flight
    int n_next;                      // fused step in flight: particle count after it
    int abort;                       // fused step in flight: some CTA declined
    int abort_reason;                // FA_* bits of every decline so far (diagnostics)
    int f_OL, f_AR;                  // fused step in flight: leavers of cell 0 downwards / wrapped arrivals in cell 0
    int maxcount, maxcount_next;     // upper bound of the largest per-cell count: current state / step in flight
    int maxdef;                      // fused step: most right-movers of one cell that overflowed the deferred queue (0: never)
    int fail_step;                   // step id (FusedArgs::step_id) of the first fused step that declined
    int tile_declined;               // tilesort.cuh: a tile's window was too wide; scatter_fast_kernel takes the arrange
};

// Per-species Boris constants (computed once on the host) and grid.
struct PushConst {
    double h, tx, ty, tz, sx, sy, sz;
    double inv_dx, dt, L;
    int nc;
    int periodic;
};

struct PushOut {
    double x, vx, vy, vz;
    int cell;  // new cell, -1 if absorbed
    int wall;  // 0 none, 1 left, 2 right
    int dcell; // |new cell - gather cell| (circular for periodic), 0 if absorbed
    int bad;   // 1 if the gather cell was outside the domain (particle left untouched)
};

// One mover step of one live particle given the two node values of its gather cell.
// jf/j: floor(x*inv_dx) already computed by the caller (it needs j to fetch E).
__device__ __forceinline__ void push_core(const PushConst &k, double x, double vx, double vy, double vz,
                                          double xs, double jf, int j, double E0, double E1, PushOut &o)
{
    // (a-1) gather: E_p = E[j] + w*(E[j+1]-E[j])
    double w = __dsub_rn(xs, jf);
    double dE = __dsub_rn(E1, E0);
    double Ep = __dadd_rn(E0, __dmul_rn(w, dE));
    // (a-2) Boris: half kick, v' = v- + v- x t, v+ = v- + v' x s, half kick; E = (Ex,0,0)
    double hE = __dmul_rn(k.h, Ep);
    double ux = __dadd_rn(vx, hE), uy = vy, uz = vz;
    double px = __dadd_rn(ux, __dsub_rn(__dmul_rn(uy, k.tz), __dmul_rn(uz, k.ty)));
    double py = __dadd_rn(uy, __dsub_rn(__dmul_rn(uz, k.tx), __dmul_rn(ux, k.tz)));
    double pz = __dadd_rn(uz, __dsub_rn(__dmul_rn(ux, k.ty), __dmul_rn(uy, k.tx)));
    double wx = __dadd_rn(ux, __dsub_rn(__dmul_rn(py, k.sz), __dmul_rn(pz, k.sy)));
    double wy = __dadd_rn(uy, __dsub_rn(__dmul_rn(pz, k.sx), __dmul_rn(px, k.sz)));
    double wz = __dadd_rn(uz, __dsub_rn(__dmul_rn(px, k.sy), __dmul_rn(py, k.sx)));
    double nvx = __dadd_rn(wx, hE);
    // (a-3) position advance
    double xn = __dadd_rn(x, __dmul_rn(nvx, k.dt));
    // (a-4) boundary and new cell
    int wall = 0;
    if (k.periodic) {
        if (xn >= k.L) {
            xn = __dsub_rn(xn, k.L);
        } else if (xn < 0.0) {
            xn = __dadd_rn(xn, k.L);
            if (xn >= k.L) xn = 0.0;
        }
    } else {
        if (xn < 0.0) wall = 1;
        else if (xn >= k.L) wall = 2;
    }
    int cn = -1, d = 0;
    if (!wall) {
        cn = (int)floor(__dmul_rn(xn, k.inv_dx));
        if (cn > k.nc - 1) cn = k.nc - 1;
        d = abs(cn - j);
        if (k.periodic) d = min(d, k.nc - d);
    }
    o.x = xn; o.vx = nvx; o.vy = wy; o.vz = wz;
    o.cell = cn; o.wall = wall; o.dcell = d; o.bad = 0;
}

// Gather-cell computation with the oracle's domain check: returns false (and leaves the
// particle alone) when x is outside [0, L].
__device__ __forceinline__ bool gather_cell(const PushConst &k, double x, double &xs, double &jf, int &j)
{
    xs = __dmul_rn(x, k.inv_dx);
    jf = floor(xs);
    if (!(jf >= 0.0) || jf > (double)k.nc) return false;
    j = (int)jf;
    if (j > k.nc - 1) { j = k.nc - 1; jf = (double)j; }
    return true;
}

// Warp-aggregated histogram increment: one atomic per distinct cell per warp.
__device__ __forceinline__ void warp_hist_add(int *__restrict__ count, int c, bool valid)
{
    unsigned act = __ballot_sync(FULL, valid);
    if (valid) {
        unsigned m = __match_any_sync(act, c);
        if ((threadIdx.x & 31) == (__ffs(m) - 1)) atomicAdd(count + c, __popc(m));
    }
}

} // namespace pic
