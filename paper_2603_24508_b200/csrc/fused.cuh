// fused.cuh -- single-pass push + arrange: one streaming kernel per step
// when every step is followed by an arrange.  68 B of DRAM traffic per particle instead of 144 B.
//
// The source state is grouped by cell (offsets off_old) and a particle moves at most one cell per
// step (verified per particle).  Then the arranged position of every particle follows from LOCAL
// counts only -- no device-wide scan:
//     class of a particle in source cell c:  L (to c-1), S (stays), R (to c+1),
//                                             X (leaves cell 0 downwards / cell nc-1 upwards:
//                                                absorbed, or wrapped on a periodic grid)
//     off_new[c]   = off_old[c] + shift - R(c-1) + L(c)                      (c >= 1; off_new[0] = 0)
//     count_new[c] = pre(c) + R(c-1) + S(c) + L(c+1) + post(c)
//     new cell c holds, in stable order:  [pre(c)] [R-movers of c-1] [S of c] [L-movers of c+1] [post(c)]
// with OL / OR = number of X particles of cell 0 / nc-1, AR = OR on a periodic grid else 0,
// shift = AR - OL, pre(nc-1) = OL and post(0) = AR on a periodic grid (wrapped arrivals), else 0.
// This IS the histogram + exclusive scan + stable scatter of the split path, with the scan
// telescoped into the flux through the cell borders.
//
// fused_edge_kernel (one small block) pushes cells 0, 1, nc-2, nc-1, publishes OL / AR, counts the
// walls and writes the wrapped particles.  fused_kernel streams everything else: each 32-thread
// CTA owns a chunk of CPC consecutive cells, cuts it greedily into tiles of whole cells that fit
// RMAX rows of 32 slots, stages tile after tile in shared memory with TMA bulk copies
// (cp.async.bulk + mbarrier; the E nodes of the chunk are staged once the same way), pushes each
// tile into REGISTERS (the stage is refilled at once, so the next tile's copies overlap the rest),
// ranks with ballot/popc prefix counts per class, and stores every particle straight to its final slot.  Across tiles it
// carries the counts of the previous cell; right-movers of a tile's last cell wait (a few
// particles, in shared memory) for the next tile's first-cell count.  Chunk ends push one halo
// cell redundantly instead of talking to the neighbour CTA.  Anything unexpected (a particle
// moving two cells, a cell larger than a tile) declines the whole step: the source buffers are
// untouched, the step's id is recorded, later fused launches exit at once, and the host redoes
// the declined steps with the split kernels (mover / scan / scatter) at its next synchronising call.
// A step is three launches: fused_edge_kernel, fused_kernel (programmatic dependent launch: its prologue overlaps
// the edge kernel, griddepcontrol.wait holds it before it reads OL / AR or writes anything), fused_commit_kernel
// (one thread: commits n, the wall counters and the bounds, or records the decline; no fence or arrival counter
// in the streaming kernel).
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int FUSED_MIN_NC = 16;
constexpr int FUSED_CPC_DEFAULT = 32;  // cells per chunk (per CTA) on grids of many waves (measured optimum at config 4)
constexpr int FUSED_CPC_SEARCH = 64;   // largest chunk the per-launch search considers on smaller grids
constexpr int FUSED_CPC_MAX = 256;
constexpr int FUSED_CPC_TAPER = 64;    // chunk size of the bulk of a many-wave grid under the tapered schedule
constexpr int FUSED_SEGS = 4;          // segments of the chunk schedule (chunk sizes CPC, CPC/2, CPC/4, CPC/8)
constexpr int FUSED_KMAX = 31;         // cells per tile (one lane per cell border)
constexpr int FUSED_DEF = 32;          // deferred right-movers of a tile's last cell: the usual queue ...
constexpr int FUSED_DEF_BIG = 128;     // ... and the one taken after a step has overflowed it (strongly drifting flows)
constexpr int FUSED_XCAP = 256;        // edge kernel: leavers per edge cell
constexpr int FUSED_TELEMETRY_STEPS = 4; // fused steps between two asynchronous copies of DevState to the host
constexpr int FUSED_RETRY_STEPS = 16;  // split steps after a decline before the fused path is tried again
constexpr int FUSED_SMEM_SM = 233472;  // shared memory per SM (228 KB), 1 KB reserved per CTA

constexpr int FA_BAD_PARTICLE = 1; // moved more than one cell / left the gather range / broke the grouping
constexpr int FA_TILE_OVERFLOW = 2; // a cell does not fit a tile (RMAX*32 slots)
constexpr int FA_DEFER_OVERFLOW = 4;
constexpr int FA_EDGE_OVERFLOW = 8;

struct FusedArgs {
    const double *sx, *svx, *svy, *svz;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const double *E;
    const int *off_old; // nc+1
    int *count_new, *off_new;
    DevState *st;
    PushConst k;
    long long capacity; // slots allocated in every particle array
    int CPC;
    int SCAP; // largest tile, in slots (<= RMAX*32, even)
    int NST;  // stages of the ring: 1 or 2
    int step_id; // low 31 bits of the species' step counter before this step
    // Chunk schedule: CTAs seg_blk[s] .. seg_blk[s+1]-1 own seg_cpc[s] cells each, starting at cell seg_cell[s]
    // (seg_cell[nseg] = nc, unused seg_blk = INT_MAX).  Large chunks first (little halo work), then ever smaller ones
    // so that the CTAs that run last are short and every SM runs dry at about the same time (pic.cu: fused_schedule).
    int seg_blk[FUSED_SEGS], seg_cell[FUSED_SEGS + 1], seg_cpc[FUSED_SEGS];
    // pic_cycle (steps of several species, deposition and field solve enqueued without a host check in between): one
    // flag per sim, set by the commit kernel of whichever species declines a step; from then on no species starts
    // another fused step and the field is not replaced, until the host has redone the cycle (NULL outside pic_cycle)
    int *frozen;
};

// Dynamic shared memory of one fused_kernel CTA (one warp): NST stages of CAP = RMAX*32 slots.
struct FusedLayout {
    int stage_bytes; // x, vx, vy, vz [CAP]
    int off_E, off_offs, off_cell, off_row, off_base, off_q, off_mbar, total;
};

__host__ __device__ inline FusedLayout fused_layout(int CAP, int CPC, int NST, int DEF = FUSED_DEF)
{
    FusedLayout L;
    L.stage_bytes = 32 * CAP;
    int o = NST * L.stage_bytes;
    L.off_E = o;    o += 8 * (CPC + 6);
    L.off_offs = o; o += 4 * (CPC + 4);
    o = (o + 15) & ~15;
    L.off_cell = o; o += 8 * (FUSED_KMAX + 1); // {first slot, count} of the tile's cells
    L.off_row = o;  o += 16 * 16;              // per row: the three class ballots and the running counts before it
    L.off_base = o; o += 8 * 4 * 32;           // per (class, cell): {slot base, destination cell}; class 3 = nothing to store
    L.off_q = o;    o += DEF * 40;
    L.off_mbar = o; o += 32;
    L.total = o;
    return L;
}

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(mbar)
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity)
{
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done)
                     : "r"(mbar), "r"(parity)
                     : "memory");
    }
}

__device__ __forceinline__ int round_up2(int v) { return (v + 1) & ~1; }

// Class of a pushed particle that sat in cell j: 0 = L, 1 = S, 2 = R, 3 = X; sets bad for anything else.
__device__ __forceinline__ int fused_classify(const PushConst &k, int j, const PushOut &o, int &bad)
{
    if (o.wall) {
        if ((o.wall == 1 && j != 0) || (o.wall == 2 && j != k.nc - 1)) bad = 1;
        return 3;
    }
    const int d = o.cell - j;
    if (d == 0) return 1;
    if (d == 1) return 2;
    if (d == -1) return 0;
    if (k.periodic && ((j == k.nc - 1 && o.cell == 0) || (j == 0 && o.cell == k.nc - 1))) return 3;
    bad = 1;
    return 3;
}

// ---- edge kernel: cells 0, 1, nc-2, nc-1 (one warp each) ------------------------------------------
// Publishes OL / AR (DevState::f_OL / f_AR), the new particle count and the pending wall counts of
// the step, and on a periodic grid writes the wrapped particles to their final slots:
//   from cell nc-1 into the END of new cell 0   : off_old[1] - OL - R(0) + L(1) + rank
//   from cell 0 into the START of new cell nc-1 : off_old[nc-1] + shift - R(nc-2) + L(nc-1) + rank
__global__ void __launch_bounds__(128) fused_edge_kernel(FusedArgs a)
{
    __shared__ double qx[2][FUSED_XCAP], qvx[2][FUSED_XCAP], qvy[2][FUSED_XCAP], qvz[2][FUSED_XCAP];
    __shared__ int cL[4], cR[4], cX[4];
    __shared__ int s_bad;
    DevState *st = a.st;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const int nc = a.k.nc;
    // programmatic dependent launch: the streaming kernel behind may start now; it waits (griddepcontrol.wait) for
    // this grid to complete before it reads anything written here or writes anything at all
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    // this kernel is itself launched programmatically behind the previous step's commit kernel (its launch overlaps
    // that kernel): everything it reads -- the state that step wrote, its offsets, DevState -- is complete after this
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
    if (st->fused_disabled || (a.frozen && *(volatile int *)a.frozen)) {
        if (threadIdx.x == 0) st->abort = 1;
        return;
    }
    const int cell = warp == 0 ? 0 : warp == 1 ? 1 : warp == 2 ? nc - 2 : nc - 1;
    const int s0 = a.off_old[cell], s1 = a.off_old[cell + 1];
    const int ql = warp == 0 ? 0 : 1; // list of this warp (only warps 0 and 3 can see class X)
    int nL = 0, nS = 0, nR = 0, nX = 0, bad = 0;
    // Batches of EDGE_ROWS rows of 32 slots: all of a batch's particle loads are issued before anything waits for one
    // of them, then all its E loads -- the kernel is a chain of memory latencies (the streaming kernel behind waits for
    // it), so a cell costs two round trips instead of two per row.
    constexpr int EDGE_ROWS = 8;
    for (int b0 = s0; b0 < s1; b0 += 32 * EDGE_ROWS) {
        double x[EDGE_ROWS], vx[EDGE_ROWS], vy[EDGE_ROWS], vz[EDGE_ROWS], xs[EDGE_ROWS], jf[EDGE_ROWS], E0[EDGE_ROWS], E1[EDGE_ROWS];
        int jj[EDGE_ROWS];
        bool ok[EDGE_ROWS];
#pragma unroll
        for (int r = 0; r < EDGE_ROWS; ++r) {
            const int i = b0 + 32 * r + lane;
            x[r] = vx[r] = vy[r] = vz[r] = 0.0;
            if (i < s1) { x[r] = a.sx[i]; vx[r] = a.svx[i]; vy[r] = a.svy[i]; vz[r] = a.svz[i]; }
        }
#pragma unroll
        for (int r = 0; r < EDGE_ROWS; ++r) {
            const int i = b0 + 32 * r + lane;
            jj[r] = cell;
            ok[r] = i < s1 && gather_cell(a.k, x[r], xs[r], jf[r], jj[r]) && jj[r] == cell;
            E0[r] = E1[r] = 0.0;
            if (ok[r]) { E0[r] = __ldg(a.E + jj[r]); E1[r] = __ldg(a.E + jj[r] + 1); }
        }
#pragma unroll
        for (int r = 0; r < EDGE_ROWS; ++r) {
            const int i = b0 + 32 * r + lane;
            if (b0 + 32 * r >= s1) break; // warp-uniform
            int g = -1;
            PushOut o;
            if (ok[r]) {
                push_core(a.k, x[r], vx[r], vy[r], vz[r], xs[r], jf[r], jj[r], E0[r], E1[r], o);
                g = fused_classify(a.k, jj[r], o, bad);
            } else if (i < s1) {
                bad = 1;
            }
            const unsigned mL = __ballot_sync(FULL, g == 0), mS = __ballot_sync(FULL, g == 1);
            const unsigned mR = __ballot_sync(FULL, g == 2), mX = __ballot_sync(FULL, g == 3);
            if (g == 3) {
                const int rk = nX + __popc(mX & lt);
                if (warp == 0 || warp == 3) {
                    if (rk < FUSED_XCAP) {
                        qx[ql][rk] = o.x; qvx[ql][rk] = o.vx; qvy[ql][rk] = o.vy; qvz[ql][rk] = o.vz;
                    } else {
                        bad |= 2; // more leavers than the list holds
                    }
                } else {
                    bad |= 1; // class X out of cell 1 or nc-2: the particle moved two cells
                }
            }
            nL += __popc(mL); nS += __popc(mS); nR += __popc(mR); nX += __popc(mX);
        }
    }
    bad = (int)__reduce_or_sync(FULL, (unsigned)bad);
    if (lane == 0) {
        cL[warp] = nL; cR[warp] = nR; cX[warp] = nX;
        if (bad) atomicOr(&s_bad, bad);
    }
    __syncthreads();
    const int OL = cX[0], OR = cX[3];
    const int AR = a.k.periodic ? OR : 0;
    if (threadIdx.x == 0) {
        if (s_bad) {
            st->abort = 1;
            atomicOr(&st->abort_reason, (s_bad & 1 ? FA_BAD_PARTICLE : 0) | (s_bad & 2 ? FA_EDGE_OVERFLOW : 0));
        }
        const int n_old = a.off_old[nc];
        st->f_OL = OL;
        st->f_AR = AR;
        st->n_next = a.k.periodic ? n_old : n_old - OL - OR;
        st->wall_pend[0] = a.k.periodic ? 0ull : (unsigned long long)OL;
        st->wall_pend[1] = a.k.periodic ? 0ull : (unsigned long long)OR;
    }
    if (!a.k.periodic || s_bad) return;
    if (warp == 0) { // wrapped downwards out of cell 0 -> start of new cell nc-1
        const long long base = (long long)a.off_old[nc - 1] + (AR - OL) - cR[2] + cL[3];
        for (int r = lane; r < OL; r += 32) {
            const long long p = base + r;
            a.dx[p] = qx[0][r]; a.dvx[p] = qvx[0][r]; a.dvy[p] = qvy[0][r]; a.dvz[p] = qvz[0][r];
            a.dcell[p] = nc - 1;
        }
    } else if (warp == 3) { // wrapped upwards out of cell nc-1 -> end of new cell 0
        const long long base = (long long)a.off_old[1] - OL - cR[0] + cL[1];
        for (int r = lane; r < OR; r += 32) {
            const long long p = base + r;
            a.dx[p] = qx[1][r]; a.dvx[p] = qvx[1][r]; a.dvy[p] = qvy[1][r]; a.dvz[p] = qvz[1][r];
            a.dcell[p] = 0;
        }
    }
}


// ---- main kernel ---------------------------------------------------------------------------------
enum { FK_REAL = 0, FK_HALO = 1, FK_VIRTUAL = 2, FK_NONE = 3 };

struct FusedItem {
    int cA, cB, kind; // cells [cA, cB)
};

struct FusedCtx { // uniform per CTA
    int C0, C1, Cm, nc;
    int CAP; // largest tile, in slots
    int STR; // slots between the x, vx, vy, vz arrays of a stage
    const int *offs; // offs[c - Cm] = off_old[c] for the chunk's cells and one halo cell on each side
};

__device__ __forceinline__ int fused_slots(const FusedCtx &X, int a, int b)
{
    const int sa = X.offs[a - X.Cm];
    return round_up2((sa & 1) + X.offs[b - X.Cm] - sa);
}

// The chunk's work items in order: [halo cell C0-1] tiles of whole cells (greedy: as many cells as
// fit CAP slots, at most 31) ... [halo cell C1 | virtual end of the grid].
__device__ __forceinline__ FusedItem fused_next_item(const FusedCtx &X, int &phase, int &cur, int lane, int &bad)
{
    FusedItem I{0, 0, FK_NONE};
    if (phase == 0) {
        phase = 1;
        cur = X.C0;
        if (X.C0 > 0) I = FusedItem{X.C0 - 1, X.C0, FK_HALO};
    }
    if (I.kind == FK_NONE && phase == 1) {
        if (cur < X.C1) {
            const int b = cur + 1 + lane;
            const bool fits = lane < FUSED_KMAX && b <= X.C1 && fused_slots(X, cur, b) <= X.CAP;
            const int nb = __popc(__ballot_sync(FULL, fits)); // fits holds for a prefix of the lanes
            if (nb == 0) {
                bad |= FA_TILE_OVERFLOW;
                phase = 3;
            } else {
                I = FusedItem{cur, cur + nb, FK_REAL};
                cur += nb;
            }
        } else {
            phase = 3;
            I = X.C1 < X.nc ? FusedItem{X.C1, X.C1 + 1, FK_HALO} : FusedItem{X.nc, X.nc, FK_VIRTUAL};
        }
    }
    if (I.kind == FK_HALO && fused_slots(X, I.cA, I.cB) > X.CAP) {
        bad |= FA_TILE_OVERFLOW;
        phase = 3;
        I.kind = FK_NONE;
    }
    return I;
}

// lane 0: start the bulk copies of one item's particles into a stage
__device__ __forceinline__ void fused_issue(const FusedArgs &a, const FusedCtx &X, FusedItem I, double *stage, unsigned mb)
{
    if (I.kind == FK_NONE || I.kind == FK_VIRTUAL) return;
    const int sA = X.offs[I.cA - X.Cm], n = X.offs[I.cB - X.Cm] - sA;
    if (n <= 0) return;
    const int pad = sA & 1;
    const long long g0 = sA - pad;
    int cnt = round_up2(pad + n);
    bool tail = false;
    if (g0 + cnt > a.capacity) { cnt -= 2; tail = true; } // the array's last, odd, element
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mb), "r"(32u * (unsigned)cnt) : "memory");
    if (cnt > 0) {
        const unsigned bytes = 8u * (unsigned)cnt;
        bulk_g2s(stage, a.sx + g0, bytes, mb);
        bulk_g2s(stage + X.STR, a.svx + g0, bytes, mb);
        bulk_g2s(stage + 2 * X.STR, a.svy + g0, bytes, mb);
        bulk_g2s(stage + 3 * X.STR, a.svz + g0, bytes, mb);
    }
    if (tail) {
        const int li = pad + n - 1;
        const long long gi = (long long)sA + n - 1;
        stage[li] = a.sx[gi]; stage[X.STR + li] = a.svx[gi]; stage[2 * X.STR + li] = a.svy[gi]; stage[3 * X.STR + li] = a.svz[gi];
    }
}

// Sweep 1a of fused_kernel for rows R0 .. R0+CNT-1 of a tile: push into registers and classify.  The
// same sequence of rounded operations as push_core, written as straight-line
// code without branches or warp collectives so that the rows' dependency chains interleave.  Slots
// outside the tile (the alignment pad, the tail of the last row, rows behind it inside the group)
// push whatever the stage holds there (every row lies inside the stage; no address depends on it)
// and are masked out.
// TMA: the tile's x, vx, vy, vz were staged in shared memory by bulk copies (p0..p3 point into the stage, E nodes
// in the shared window pE); otherwise they are read straight from global memory (p0..p3 = the arrays at the tile's
// first slot, read-only path; slot index clamped to imax so that no load leaves the arrays; pE = the E array).
// EDGE = the tile holds cell 0, nc-2 or nc-1: only there can a particle wrap / be absorbed (class X), can
// floor(x/dx) need the clamp of reading S8, or can x leave the gather range legitimately.  Elsewhere a new cell
// more than one away from the source cell marks the particle bad (it moved more than one cell, left the grid,
// or the grouping is broken) and no clamp is needed: the source cells are 1 .. nc-3.
// cellinfo[cl] = {first slot, count} of the tile's cells from off_old: a slot outside its cell's range
// means the grouping is broken.  W_[r] = class << 5 | local cell | bad << 8 (class 3: nothing to store).
template <bool PERIODIC, bool EDGE, bool BZ0, bool TMA, int RMAX, int R0, int CNT>
__device__ __forceinline__ void fused_sweep1a(const PushConst &k, const double *pE, const int2 *cellinfo, int lane,
                                              int pad, int n, int cA, int ncell, double (&X_)[RMAX], double (&VX_)[RMAX],
                                              double (&VY_)[RMAX], double (&VZ_)[RMAX], int (&W_)[RMAX])
{
    const int nc = k.nc;
#pragma unroll
    for (int r = R0; r < R0 + CNT; ++r) {
        const int i = (r << 5) + lane;
        const bool valid = (unsigned)(i - pad) < (unsigned)n;
        const double x = X_[r], vx = VX_[r], vy = VY_[r], vz = VZ_[r]; // loaded by fused_load_rows
        const double xs = __dmul_rn(x, k.inv_dx);
        int jc = __double2int_rd(xs);
        double jf = (double)jc; // = floor(xs) whenever the particle is inside the grid (anything else is declined)
        bool inr = true;
        if (EDGE) {
            inr = xs >= 0.0 && jc <= nc;
            if (jc > nc - 1) { jc = nc - 1; jf = (double)(nc - 1); }
        }
        const int cl = jc - cA;
        inr = inr && (unsigned)cl < (unsigned)ncell;
        const int j = inr ? jc : cA;
        if (!inr) jf = (double)cA;
        const int2 sc = cellinfo[j - cA];
        const bool inside = (unsigned)(i - sc.x) < (unsigned)sc.y;
        double E0, E1;
        if (TMA) { E0 = pE[j]; E1 = pE[j + 1]; }
        else { E0 = __ldg(pE + j); E1 = __ldg(pE + j + 1); }
        const double w = __dsub_rn(xs, jf);
        const double dE = __dsub_rn(E1, E0);
        const double Ep = __dadd_rn(E0, __dmul_rn(w, dE));
        const double hE = __dmul_rn(k.h, Ep);
        const double ux = __dadd_rn(vx, hE), uy = vy, uz = vz;
        double qx, qy, qz, wx, wy, wz;
        if (BZ0) {
            // Bz = 0 (so tz = sz = 0): the products with tz / sz are exact zeros and a + (0 - b) == a - b, a + (b - 0) == a + b
            // bit for bit (only the sign of a zero can differ)
            qx = __dsub_rn(ux, __dmul_rn(uz, k.ty));
            qy = __dadd_rn(uy, __dmul_rn(uz, k.tx));
            qz = __dadd_rn(uz, __dsub_rn(__dmul_rn(ux, k.ty), __dmul_rn(uy, k.tx)));
            wx = __dsub_rn(ux, __dmul_rn(qz, k.sy));
            wy = __dadd_rn(uy, __dmul_rn(qz, k.sx));
            wz = __dadd_rn(uz, __dsub_rn(__dmul_rn(qx, k.sy), __dmul_rn(qy, k.sx)));
        } else {
            qx = __dadd_rn(ux, __dsub_rn(__dmul_rn(uy, k.tz), __dmul_rn(uz, k.ty)));
            qy = __dadd_rn(uy, __dsub_rn(__dmul_rn(uz, k.tx), __dmul_rn(ux, k.tz)));
            qz = __dadd_rn(uz, __dsub_rn(__dmul_rn(ux, k.ty), __dmul_rn(uy, k.tx)));
            wx = __dadd_rn(ux, __dsub_rn(__dmul_rn(qy, k.sz), __dmul_rn(qz, k.sy)));
            wy = __dadd_rn(uy, __dsub_rn(__dmul_rn(qz, k.sx), __dmul_rn(qx, k.sz)));
            wz = __dadd_rn(uz, __dsub_rn(__dmul_rn(qx, k.sy), __dmul_rn(qy, k.sx)));
        }
        const double nvx = __dadd_rn(wx, hE);
        const double xn = __dadd_rn(x, __dmul_rn(nvx, k.dt));
        double xw = xn;
        int g;
        bool good;
        if (EDGE) {
            bool legit = false;
            int wall = 0;
            if (PERIODIC) {
                const double xm = __dsub_rn(xn, k.L), xp = __dadd_rn(xn, k.L);
                xw = xn >= k.L ? xm : (xn < 0.0 ? (xp >= k.L ? 0.0 : xp) : xn);
            } else {
                wall = xn < 0.0 ? 1 : (xn >= k.L ? 2 : 0);
            }
            const int cn = min(__double2int_rd(__dmul_rn(xw, k.inv_dx)), nc - 1);
            const int d = cn - j;
            g = (unsigned)(d + 1) <= 2u ? d + 1 : 3;
            // class X: out of cell 0 downwards / out of cell nc-1 upwards only
            if (PERIODIC) {
                legit = (j == nc - 1 && cn == 0) || (j == 0 && cn == nc - 1);
            } else {
                if (wall) g = 3;
                legit = (wall == 1 && j == 0) || (wall == 2 && j == nc - 1);
            }
            good = valid && inr && inside && (g < 3 || legit);
        } else {
            const int d = __double2int_rd(__dmul_rn(xn, k.inv_dx)) - j;
            g = (unsigned)(d + 1) <= 2u ? d + 1 : 3;
            good = valid && inr && inside && g < 3;
        }
        if (!good) g = 3;
        W_[r] = (g << 5) | (j - cA) | ((valid && !good) ? 256 : 0);
        X_[r] = xw; VX_[r] = nvx; VY_[r] = wy; VZ_[r] = wz;
    }
}

// Row groups of the sweeps.  Width 0: rows 4 by 4 while at least four more can follow, then 2, 1, 1 (for RMAX = 8:
// {0-3} {4,5} {6} {7}; a tile pushes at most one surplus row).  Width W > 0: groups of W rows ({0-3} {4-7}).  A group
// runs if its first row is inside the tile; rows of it behind the tile are masked out (class X, nothing stored), so
// that a group is straight-line code whose rows' dependency chains interleave.  (Width 4 everywhere measured equal at
// config 4 and 8 % slower at config 2, where the surplus rows count: profiles/r02_variants.md.)
#ifndef FUSED_W1A
#define FUSED_W1A 0 // sweep 1a (and the loads)
#endif
#ifndef FUSED_W1B
#define FUSED_W1B 0 // sweep 1b
#endif
#ifndef FUSED_W2
#define FUSED_W2 0  // sweep 2
#endif
__host__ __device__ constexpr int fused_ngroups(int rmax, int w) { return w ? (rmax + w - 1) / w : rmax / 4 + 2; }
__host__ __device__ constexpr int fused_group_start(int rmax, int w, int gi)
{
    return w ? w * gi : (gi < rmax / 4 - 1 ? 4 * gi : 4 * (rmax / 4 - 1) + (gi == rmax / 4 - 1 ? 0 : (gi == rmax / 4 ? 2 : 3)));
}
__host__ __device__ constexpr int fused_group_count(int rmax, int w, int gi)
{
    return w ? (w * gi + w <= rmax ? w : rmax - w * gi) : (gi < rmax / 4 - 1 ? 4 : (gi == rmax / 4 - 1 ? 2 : 1));
}

// The tile's x, vx, vy, vz from the stage (or, without TMA, from global memory) into the register tile, by the same
// row groups as the sweeps.  Done for the whole tile BEFORE the arithmetic, so that the stage is free again at once
// and the next tile's bulk copies are in flight during all of this tile's work.
template <bool TMA, int RMAX>
__device__ __forceinline__ void fused_load_rows(const double *p0, const double *p1, const double *p2, const double *p3, int imax,
                                                int lane, int nrows, double (&X_)[RMAX], double (&VX_)[RMAX],
                                                double (&VY_)[RMAX], double (&VZ_)[RMAX])
{
#pragma unroll
    for (int gi = 0; gi < fused_ngroups(RMAX, FUSED_W1A); ++gi) {
        const int g0 = fused_group_start(RMAX, FUSED_W1A, gi), gn = fused_group_count(RMAX, FUSED_W1A, gi);
        if (g0 < nrows) {
#pragma unroll
            for (int r = g0; r < g0 + gn; ++r) {
                const int i = (r << 5) + lane;
                if (TMA) {
                    X_[r] = p0[i]; VX_[r] = p1[i]; VY_[r] = p2[i]; VZ_[r] = p3[i];
                } else {
                    const int il = min(i, imax);
                    X_[r] = __ldg(p0 + il); VX_[r] = __ldg(p1 + il); VY_[r] = __ldg(p2 + il); VZ_[r] = __ldg(p3 + il);
                }
            }
        }
    }
}

template <bool PERIODIC, bool EDGE, bool BZ0, bool TMA, int RMAX>
__device__ __forceinline__ void fused_sweep1a_all(const PushConst &k, const double *pE, const int2 *cellinfo, int lane,
                                                  int pad, int n, int nrows, int cA, int ncell, double (&X_)[RMAX], double (&VX_)[RMAX],
                                                  double (&VY_)[RMAX], double (&VZ_)[RMAX], int (&W_)[RMAX])
{
#define FUSED_ROWS(GI) \
    if constexpr (GI < fused_ngroups(RMAX, FUSED_W1A)) if (fused_group_start(RMAX, FUSED_W1A, GI) < nrows) \
        fused_sweep1a<PERIODIC, EDGE, BZ0, TMA, RMAX, fused_group_start(RMAX, FUSED_W1A, GI), fused_group_count(RMAX, FUSED_W1A, GI)>( \
            k, pE, cellinfo, lane, pad, n, cA, ncell, X_, VX_, VY_, VZ_, W_);
    FUSED_ROWS(0) FUSED_ROWS(1) FUSED_ROWS(2) FUSED_ROWS(3) FUSED_ROWS(4) FUSED_ROWS(5)
#undef FUSED_ROWS
}

// TMA = true: particles and the chunk's E window are staged in shared memory by bulk copies (cp.async.bulk + mbarrier).
// TMA = false (option "fused_tma" = 0, the A/B variant of profiles/): plain read-only global loads into the same
// registers, E through the read-only path; no stage, no mbarrier.
// DEF = capacity of the queue of right-movers deferred to the next tile (FUSED_DEF, or FUSED_DEF_BIG after an overflow).
template <int RMAX, bool PERIODIC, bool BZ0, bool TMA, int DEF>
__global__ void __launch_bounds__(32, RMAX == 8 ? 16 : (RMAX == 12 ? 10 : 8)) fused_kernel(FusedArgs a)
{
    static_assert(RMAX == 8 || RMAX == 12 || RMAX == 16, "row groups of sweep 1a are written for these sizes");
    extern __shared__ __align__(128) unsigned char fused_smem[];
    constexpr int CAP = RMAX * 32;
    const FusedLayout L = fused_layout(CAP, a.CPC, a.NST, DEF);
    double *sE = reinterpret_cast<double *>(fused_smem + L.off_E);
    int *offs = reinterpret_cast<int *>(fused_smem + L.off_offs);
    int2 *cellinfo = reinterpret_cast<int2 *>(fused_smem + L.off_cell); // {first slot, count} of the tile's cells
    int4 *rowinfo = reinterpret_cast<int4 *>(fused_smem + L.off_row);   // per row: ballots L, S, R; running counts before it
    int2 *basd = reinterpret_cast<int2 *>(fused_smem + L.off_base);     // [class*32 + cell]: {slot base, destination cell}
    double *qx = reinterpret_cast<double *>(fused_smem + L.off_q), *qvx = qx + DEF, *qvy = qx + 2 * DEF, *qvz = qx + 3 * DEF;
    int *qpos = reinterpret_cast<int *>(qx + 4 * DEF);
    const unsigned mb0 = smem_u32(fused_smem + L.off_mbar), mb1 = mb0 + 8, mbE = mb0 + 16;
    const int lane = threadIdx.x;
    const unsigned lt = (1u << lane) - 1u;
    DevState *st = a.st;
    const int nc = a.k.nc;
    int bad = 0;  // FA_* bits
    int mc = 0;   // largest new per-cell count seen by this lane

    // CTAs are dispatched in blockIdx order: the schedule's large chunks run first, its small ones last.
    int sg_blk = 0, sg_cell = 0, sg_cpc = a.seg_cpc[0], sg_end = a.seg_cell[1];
#pragma unroll
    for (int sg = 1; sg < FUSED_SEGS; ++sg)
        if ((int)blockIdx.x >= a.seg_blk[sg]) { sg_blk = a.seg_blk[sg]; sg_cell = a.seg_cell[sg]; sg_cpc = a.seg_cpc[sg]; sg_end = a.seg_cell[sg + 1]; }
    {
        FusedCtx X;
        X.C0 = sg_cell + ((int)blockIdx.x - sg_blk) * sg_cpc;
        X.C1 = min(X.C0 + sg_cpc, sg_end);
        X.Cm = max(X.C0 - 1, 0);
        X.nc = nc;
        X.CAP = a.SCAP;
        X.STR = CAP;
        X.offs = offs;
        const int Cm = X.Cm, Cp = min(X.C1 + 1, nc);
        // Prologue: reads only what was complete before the edge kernel of this step started (off_old, E, the source
        // particles), writes nothing outside shared memory -- under programmatic dependent launch it overlaps that
        // kernel.
        for (int idx = lane; idx <= Cp - Cm; idx += 32) offs[idx] = a.off_old[Cm + idx];
        const int ea = Cm & ~1;
        const double *sEs = sE - ea; // E node j of the chunk's window sits at sEs[j]
        const unsigned cap32 = (unsigned)a.capacity;
        if (TMA && lane == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(mb0) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(mb1) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(mbE) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
            // E nodes Cm .. Cp of the chunk (16-byte aligned window; E is padded)
            const unsigned eb = 8u * (unsigned)round_up2(Cp + 1 - ea);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mbE), "r"(eb) : "memory");
            bulk_g2s(sE, a.E + ea, eb, mbE);
        }
        __syncwarp();
        int phase = 0, cur = 0;
        FusedItem I0 = fused_next_item(X, phase, cur, lane, bad);
        FusedItem I1 = fused_next_item(X, phase, cur, lane, bad);
        const bool two = a.NST == 2;
        double *stage0 = reinterpret_cast<double *>(fused_smem), *stage1 = reinterpret_cast<double *>(fused_smem + L.stage_bytes);
        if (TMA && lane == 0) {
            fused_issue(a, X, I0, stage0, mb0);
            if (two) fused_issue(a, X, I1, stage1, mb1);
        }
        // From here on the edge kernel's results are needed (abort flag, OL, AR) and global memory is written: wait for
        // it (a no-op without programmatic dependent launch: stream order has done it).
        asm volatile("griddepcontrol.wait;\n" ::: "memory");
        if (TMA) mbar_wait(mbE, 0);
        if (*(volatile int *)&st->abort) {
            // a fused step declined earlier: this launch must not touch anything.  Let the bulk copies already under
            // way land before the CTA gives its shared memory back.
            if (TMA) {
                if (I0.kind <= FK_HALO && offs[I0.cB - Cm] > offs[I0.cA - Cm]) mbar_wait(mb0, 0);
                if (two && I1.kind <= FK_HALO && offs[I1.cB - Cm] > offs[I1.cA - Cm]) mbar_wait(mb1, 0);
            }
            I0.kind = FK_NONE;
        }
        const int OL = st->f_OL, AR = st->f_AR, shift = AR - OL;
        // carry across tiles: class counts of the previous tile's last cell
        int pvL = 0, pvS = 0, pvR = 0;
        int pvRR = 0;    // R of the cell before the carried one
        int pv_off = 0;  // off_old of the carried cell
        int pv_real = 0; // the carried cell belongs to this chunk (finalize it)
        int ndef = 0;    // deferred right-movers of the carried cell
        unsigned ph0 = 0, ph1 = 0;

        for (int it = 0; I0.kind != FK_NONE; ++it) {
            const FusedItem I2 = fused_next_item(X, phase, cur, lane, bad);
            const int kind = I0.kind, cA = I0.cA, cB = I0.cB, ncell = cB - cA;
            const int sA = kind == FK_VIRTUAL ? 0 : offs[cA - Cm];
            const int n = kind == FK_VIRTUAL ? 0 : offs[cB - Cm] - sA;
            const int pad = sA & 1, gbase = sA - pad;
            const int nrows = n > 0 ? (pad + n + 31) >> 5 : 0;
            // lane q: first slot of local cell q (q = ncell: the end of the tile), from off_old
            int st_q = pad + n;
            if (kind != FK_VIRTUAL && lane <= ncell) {
                st_q = offs[cA - Cm + lane] - gbase;
                if (lane < ncell) cellinfo[lane] = make_int2(st_q, offs[cA - Cm + lane + 1] - gbase - st_q);
            }
            __syncwarp();
            const bool odd = two && (it & 1);
            double *px = odd ? stage1 : stage0;
            if (TMA && n > 0) {
                if (odd) { mbar_wait(mb1, ph1); ph1 ^= 1u; }
                else     { mbar_wait(mb0, ph0); ph0 ^= 1u; }
            }

            // ---- sweep 1a: push into registers and classify (fused_sweep1a) ----------------------------------
            double X_[RMAX], VX_[RMAX], VY_[RMAX], VZ_[RMAX];
            int W_[RMAX]; // 1a: class << 5 | cell | bad << 8;  1b: class prefix count << 8 | class*32 + cell
            {
                const double *p0 = TMA ? px : a.sx + gbase, *p1 = TMA ? px + CAP : a.svx + gbase;
                const double *p2 = TMA ? px + 2 * CAP : a.svy + gbase, *p3 = TMA ? px + 3 * CAP : a.svz + gbase;
                const int imax = TMA ? CAP - 1 : (int)min((long long)(CAP - 1), a.capacity - 1 - gbase);
                fused_load_rows<TMA, RMAX>(p0, p1, p2, p3, imax, lane, nrows, X_, VX_, VY_, VZ_);
            }
            __syncwarp();
            // the stage has been read into registers: refill it with the next item to load
            if (TMA && lane == 0) fused_issue(a, X, two ? I2 : I1, px, odd ? mb1 : mb0);
            {
                const double *pE = TMA ? sEs : a.E;
                if (cA == 0 || cB >= nc - 1)
                    fused_sweep1a_all<PERIODIC, true, BZ0, TMA, RMAX>(a.k, pE, cellinfo, lane, pad, n, nrows, cA, ncell, X_, VX_, VY_, VZ_, W_);
                else
                    fused_sweep1a_all<PERIODIC, false, BZ0, TMA, RMAX>(a.k, pE, cellinfo, lane, pad, n, nrows, cA, ncell, X_, VX_, VY_, VZ_, W_);
            }
            __syncwarp();

            // ---- sweep 1b: prefix counts per class (ballot/popc); the row's ballots are kept for the cell borders ---
            int runL = 0, runS = 0, runR = 0; // running class counts of the tile (warp-uniform)
            int wor = 0;
#pragma unroll
            for (int gi = 0; gi < fused_ngroups(RMAX, FUSED_W1B); ++gi) {
                if (fused_group_start(RMAX, FUSED_W1B, gi) < nrows) {
#pragma unroll
                    for (int r = fused_group_start(RMAX, FUSED_W1B, gi); r < fused_group_start(RMAX, FUSED_W1B, gi) + fused_group_count(RMAX, FUSED_W1B, gi); ++r) {
                        const int w = W_[r];
                        wor |= w;
                        const bool isL = (w & 96) == 0, isS = (w & 96) == 32;
                        const unsigned mL = __ballot_sync(FULL, isL), mS = __ballot_sync(FULL, isS), mR = __ballot_sync(FULL, (w & 96) == 64);
                        if (lane == 0) rowinfo[r] = make_int4((int)mL, (int)mS, (int)mR, runL | (runS << 10) | (runR << 20));
                        const unsigned mo = isL ? mL : (isS ? mS : mR);
                        const int rn = isL ? runL : (isS ? runS : runR);
                        W_[r] = ((rn + __popc(mo & lt)) << 8) | (w & 127); // class 3 keeps a key >= 96: nothing is stored for it
                        runL += __popc(mL); runS += __popc(mS); runR += __popc(mR);
                    }
                }
            }
            if (wor & 256) bad |= FA_BAD_PARTICLE;
            const unsigned run = (unsigned)(runL | (runS << 10) | (runR << 20));
            __syncwarp();

            // ---- per-cell phase (lane q = local cell q; lane ncell = the end of the tile) ---------------------
            // class prefix counts at the first slot of cell q, from the ballots of the row that holds it
            unsigned ps = run;
            if ((st_q >> 5) < nrows) {
                const int4 ri = rowinfo[st_q >> 5];
                const unsigned below = (1u << (st_q & 31)) - 1u;
                ps = (unsigned)ri.w + ((unsigned)__popc((unsigned)ri.x & below) | ((unsigned)__popc((unsigned)ri.y & below) << 10) |
                                       ((unsigned)__popc((unsigned)ri.z & below) << 20));
            }
            const unsigned c3 = __shfl_down_sync(FULL, ps, 1) - ps; // class counts of cell q (fields cannot borrow)
            const bool mycell = kind != FK_VIRTUAL && lane < ncell;
            const int Lc = mycell ? (int)(c3 & 1023u) : 0, Sc = mycell ? (int)((c3 >> 10) & 1023u) : 0, Rc = mycell ? (int)(c3 >> 20) : 0;
            const int psL = (int)(ps & 1023u), psS = (int)((ps >> 10) & 1023u), psR = (int)(ps >> 20);
            int Rm1 = __shfl_up_sync(FULL, Rc, 1);
            if (lane == 0) Rm1 = pvR;
            int Lp1 = __shfl_down_sync(FULL, Lc, 1);
            if (lane >= ncell - 1) Lp1 = 0; // last cell: added when the next tile knows it
            const int Lc0 = __shfl_sync(FULL, Lc, 0);
            bool oob = false;
            if (kind == FK_REAL && lane < ncell) {
                const int c = cA + lane;
                const int oo = gbase + st_q, oo1 = oo + cellinfo[lane].y;
                const int pre_c = (PERIODIC && c == nc - 1) ? OL : 0;
                const int pre_c1 = (PERIODIC && c + 1 == nc - 1) ? OL : 0;
                basd[lane] = make_int2(oo + (c == 1 ? -OL : shift) - Rm1 - psL, c - 1);
                basd[32 + lane] = make_int2(oo + (c >= 1 ? shift : 0) + Lc + pre_c - psS, c);
                basd[64 + lane] = make_int2(oo1 + shift - Rc + Lp1 + pre_c1 - psR, c + 1);
                // slot ranges of the three classes of this cell (ranks are below the class counts): all stores of
                // sweep 2 stay inside the arrays, or the tile is declined before any of them is issued
                const int bL = oo + (c == 1 ? -OL : shift) - Rm1, bS = oo + (c >= 1 ? shift : 0) + Lc + pre_c,
                          bR = oo1 + shift - Rc + Lp1 + pre_c1;
                oob = (Lc && ((unsigned)bL >= cap32 || (unsigned)(bL + Lc - 1) >= cap32)) ||
                      (Sc && ((unsigned)bS >= cap32 || (unsigned)(bS + Sc - 1) >= cap32)) ||
                      (Rc && ((unsigned)bR >= cap32 || (unsigned)(bR + Rc - 1) >= cap32));
                if (lane < ncell - 1) { // count / offset of cell c (the tile's last cell waits for the next tile)
                    const int cn = pre_c + Rm1 + Sc + Lp1 + (c == 0 ? AR : 0);
                    a.count_new[c] = cn;
                    a.off_new[c] = c == 0 ? 0 : oo + shift - Rm1 + Lc;
                    mc = max(mc, cn);
                }
            }
            if (pv_real && lane == 0) { // count / offset of the previous tile's last cell
                const int c = cA - 1;
                const int pre_c = (PERIODIC && c == nc - 1) ? OL : 0;
                const int cn = pre_c + pvRR + pvS + Lc0 + (c == 0 ? AR : 0);
                const int o0 = c == 0 ? 0 : pv_off + shift - pvRR + pvL;
                a.count_new[c] = cn;
                a.off_new[c] = o0;
                if (c == nc - 1) a.off_new[nc] = o0 + cn;
                mc = max(mc, cn);
            }
            if (ndef) { // right-movers of the previous tile's last cell: their cell is cA, its L count is known now
#pragma unroll
                for (int q0 = 0; q0 < DEF; q0 += 32) {
                    const int q = q0 + lane;
                    if (q < ndef) {
                        const int p = qpos[q] + Lc0;
                        if ((unsigned)p >= cap32) bad |= FA_BAD_PARTICLE;
                        else {
                            a.dx[p] = qx[q]; a.dvx[p] = qvx[q]; a.dvy[p] = qvy[q]; a.dvz[p] = qvz[q];
                            a.dcell[p] = cA;
                        }
                    }
                    if (DEF > 32 && q0 + 32 >= ndef) break;
                }
                ndef = 0;
            }
            __syncwarp();

            // ---- sweep 2: every particle straight to its final slot ----------------------------------
            const bool tile_oob = __any_sync(FULL, oob);
            if (tile_oob) bad |= FA_BAD_PARTICLE;
            if (kind == FK_REAL && !tile_oob) {
                const int kdef = 64 + ncell - 1;                                 // class R of the tile's last cell
                const int lastq = max(ncell - 1, 0);
                const int rdef = __shfl_sync(FULL, st_q, lastq) >> 5;            // first row that can hold it
                const int psRlast = __shfl_sync(FULL, psR, lastq);               // R particles of the tile before that cell
                const int nRlast = __shfl_sync(FULL, Rc, lastq);                 // its right-movers: deferred to the next tile
                if (nRlast > DEF) { // the host learns how many there were and takes the larger queue when it comes back
                    bad |= FA_DEFER_OVERFLOW;
                    if (lane == 0) atomicMax(&st->maxdef, nRlast);
                }
#pragma unroll
                for (int gi = 0; gi < fused_ngroups(RMAX, FUSED_W2); ++gi) {
                    if (fused_group_start(RMAX, FUSED_W2, gi) < nrows) {
#pragma unroll
                        for (int r = fused_group_start(RMAX, FUSED_W2, gi); r < fused_group_start(RMAX, FUSED_W2, gi) + fused_group_count(RMAX, FUSED_W2, gi); ++r) {
                            const int pk = W_[r];
                            const int key = pk & 127;
                            const int2 bd = basd[key];
                            const int p = bd.x + (pk >> 8);
                            if (key < 96 && key != kdef) {
                                a.dx[p] = X_[r]; a.dvx[p] = VX_[r]; a.dvy[p] = VY_[r]; a.dvz[p] = VZ_[r];
                                a.dcell[p] = bd.y;
                            }
                            if (r >= rdef && key == kdef) { // its rank inside the class is its place in the queue
                                const int q = (pk >> 8) - psRlast;
                                if (q < DEF) {
                                    qx[q] = X_[r]; qvx[q] = VX_[r]; qvy[q] = VY_[r]; qvz[q] = VZ_[r];
                                    qpos[q] = p;
                                }
                            }
                        }
                    }
                }
                ndef = min(nRlast, DEF);
            }
            // carry: this tile's last cell
            if (kind != FK_VIRTUAL) {
                const int nRR = ncell >= 2 ? __shfl_sync(FULL, Rc, ncell - 2) : pvR;
                pvL = __shfl_sync(FULL, Lc, ncell - 1);
                pvS = __shfl_sync(FULL, Sc, ncell - 1);
                pvR = __shfl_sync(FULL, Rc, ncell - 1);
                pvRR = nRR;
                pv_off = offs[cB - 1 - Cm];
                pv_real = kind == FK_REAL;
            }
            __syncwarp();
            I0 = I1;
            I1 = I2;
        }
    }

    // ---- CTA epilogue: report a decline and the largest new per-cell count.  No fence, no arrival counter: the step
    // is committed or rolled back by fused_commit_kernel, launched behind this kernel on the same stream.
    bad = (int)__reduce_or_sync(FULL, (unsigned)bad);
    mc = __reduce_max_sync(FULL, mc);
    if (lane == 0) {
        if (bad) {
            atomicExch(&st->abort, 1);
            atomicOr(&st->abort_reason, bad);
        }
        if (mc > *(volatile int *)&st->maxcount_next) atomicMax(&st->maxcount_next, mc);
    }
}

// Commit or roll back one fused step (one thread, launched behind fused_kernel; the kernel boundary orders it
// after every CTA's stores and atomics).
__global__ void fused_commit_kernel(DevState *st, int step_id, int *frozen)
{
    // launched programmatically behind fused_kernel: wait for that grid to complete (no early trigger there, so this
    // kernel runs after every CTA has exited; and none here, so the next step's edge kernel -- and with it the next
    // streaming kernel's prologue -- starts only after this step is complete)
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    if (!st->abort) {
        st->n = st->n_next;
        st->wall[0] += st->wall_pend[0];
        st->wall[1] += st->wall_pend[1];
        st->wall_arr = st->wall[0] + st->wall[1];
        st->vmax2 = 0x7f800000u; // speed bound unknown after a fused step (+inf): the split path, should it
                                 // take over, enqueues its general arranger until its mover has measured one
        st->maxcount = st->maxcount_next;
        st->w_acc = 0;
        st->step_max = 0;
        st->need_general = 0;
        st->used_general = 0;
    } else {
        // declined: nothing of the state was touched (outputs went to the other buffer set); remember which
        // step it was, every later fused launch exits at once, the host redoes the steps (pic.cu: verify_fused)
        if (!st->fused_disabled) st->fail_step = step_id;
        st->fused_disabled = 1;
        if (frozen) *frozen = 1;
    }
    st->n_next = 0;
    st->wall_pend[0] = st->wall_pend[1] = 0;
    st->vmax2_next = 0;
    st->maxcount_next = 0;
    st->abort = 0;
}

// Largest per-cell count of an offset array (sizes the fused tiles; only ever raises the bound).
__global__ void maxcount_kernel(const int *__restrict__ off, int nc, DevState *st)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int cn = c < nc ? off[c + 1] - off[c] : 0;
    cn = __reduce_max_sync(FULL, cn);
    if ((threadIdx.x & 31) == 0 && cn > *(volatile int *)&st->maxcount) atomicMax(&st->maxcount, cn);
}

} // namespace pic
