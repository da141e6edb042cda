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
// CTA owns a contiguous chunk of cell-aligned tiles (~T particles each), stages tile after tile in
// a two-stage shared-memory ring with TMA bulk copies (x, vx, vy, vz and the E nodes of the
// tile's cells; cp.async.bulk + mbarrier), pushes in place, ranks with ballot/popc prefix counts,
// and stores every particle straight to its final slot.  Across tiles it carries the counts of the
// previous cell; right-movers of a tile's last cell wait (a few particles, in shared memory) for
// the next tile's first-cell count.  Chunk ends push one halo cell redundantly instead of talking
// to the neighbour CTA.  Anything unexpected (a particle moving two cells, a tile larger than the
// shared-memory stage) aborts the whole step: the source buffers are untouched, and the guarded
// split kernels launched right behind (mover / scan / scatter) redo it.
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int FUSED_MIN_NC = 16;
constexpr int FUSED_T_DEFAULT = 128;   // target particles per tile
constexpr int FUSED_T_MIN = 64;
constexpr int FUSED_TPC_DEFAULT = 64;  // tiles per chunk (per CTA)
constexpr int FUSED_TPC_MAX = 256;
constexpr int FUSED_KMAX = 63;         // cells per tile
constexpr int FUSED_DEF = 32;          // deferred right-movers of a tile's last cell
constexpr int FUSED_XCAP = 256;        // edge kernel: leavers per edge cell
constexpr int FUSED_SMEM_SM = 233472;  // shared memory per SM (228 KB), 1 KB reserved per CTA
constexpr int FUSED_SMEM_CTA = 232448; // 227 KB

constexpr int FA_BAD_PARTICLE = 1; // moved more than one cell / left the gather range / broke the grouping
constexpr int FA_TILE_OVERFLOW = 2; // a tile does not fit the stage (CAP slots, KMAX cells)
constexpr int FA_DEFER_OVERFLOW = 4;
constexpr int FA_EDGE_OVERFLOW = 8;

struct FusedArgs {
    const double *sx, *svx, *svy, *svz;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const double *E;
    const int *off_old;  // nc+1
    const int2 *td_old;  // tile k covers cells [td[k].x, td[k+1].x), slots [td[k].y, td[k+1].y)
    int *count_new, *off_new;
    int2 *td_new;
    DevState *st;
    PushConst k;
    long long capacity; // slots allocated in every particle array
    int T, CAP, TPC, td_cap;
};

// Dynamic shared memory of one fused_kernel CTA (one warp).
struct FusedLayout {
    int stage_bytes; // x, vx, vy, vz [CAP] + E window
    int off_code, off_start, off_ps, off_pe, off_cnt, off_base, off_q, off_items, off_kind, off_mbar, total;
};

__host__ __device__ inline FusedLayout fused_layout(int CAP, int TPC)
{
    FusedLayout L;
    L.stage_bytes = 32 * CAP + 8 * (FUSED_KMAX + 3);
    int o = 2 * L.stage_bytes;
    L.off_code = o;  o += 4 * CAP;
    L.off_start = o; o += 4 * (FUSED_KMAX + 1);
    L.off_ps = o;    o += 2 * 3 * (FUSED_KMAX + 1);
    L.off_pe = o;    o += 2 * 3 * (FUSED_KMAX + 1);
    L.off_cnt = o;   o += 4 * 3 * (FUSED_KMAX + 1);
    L.off_base = o;  o += 4 * 3 * (FUSED_KMAX + 1);
    L.off_q = o;     o += FUSED_DEF * 40;
    L.off_items = o; o += 16 * (TPC + 2);
    L.off_kind = o;  o += 4 * (TPC + 2);
    o = (o + 15) & ~15;
    L.off_mbar = o;  o += 16;
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
    __shared__ int cL[4], cS[4], cR[4], cX[4];
    __shared__ int s_bad;
    DevState *st = a.st;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = (1u << lane) - 1u;
    const int nc = a.k.nc;
    if (threadIdx.x == 0) s_bad = 0;
    __syncthreads();
    if (st->fused_disabled) {
        if (threadIdx.x == 0) st->abort = 1;
        return;
    }
    const int cell = warp == 0 ? 0 : warp == 1 ? 1 : warp == 2 ? nc - 2 : nc - 1;
    const int s0 = a.off_old[cell], s1 = a.off_old[cell + 1];
    const int ql = warp == 0 ? 0 : 1; // list of this warp (only warps 0 and 3 can see class X)
    int nL = 0, nS = 0, nR = 0, nX = 0, bad = 0;
    for (int i0 = s0; i0 < s1; i0 += 32) {
        const int i = i0 + lane;
        int g = -1;
        PushOut o;
        if (i < s1) {
            const double x = a.sx[i], vx = a.svx[i], vy = a.svy[i], vz = a.svz[i];
            double xs, jf;
            int j;
            if (gather_cell(a.k, x, xs, jf, j) && j == cell) {
                const double E0 = __ldg(a.E + j), E1 = __ldg(a.E + j + 1);
                push_core(a.k, x, vx, vy, vz, xs, jf, j, E0, E1, o);
                g = fused_classify(a.k, j, o, bad);
            } else {
                bad = 1;
            }
        }
        const unsigned mL = __ballot_sync(FULL, g == 0), mS = __ballot_sync(FULL, g == 1);
        const unsigned mR = __ballot_sync(FULL, g == 2), mX = __ballot_sync(FULL, g == 3);
        if (g == 3) {
            const int r = nX + __popc(mX & lt);
            if (r < FUSED_XCAP && (warp == 0 || warp == 3)) {
                qx[ql][r] = o.x; qvx[ql][r] = o.vx; qvy[ql][r] = o.vy; qvz[ql][r] = o.vz;
            } else {
                bad = 2;
            }
        }
        nL += __popc(mL); nS += __popc(mS); nR += __popc(mR); nX += __popc(mX);
    }
    bad = (int)__reduce_or_sync(FULL, (unsigned)bad);
    if (lane == 0) {
        cL[warp] = nL; cS[warp] = nS; cR[warp] = nR; cX[warp] = nX;
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
enum { FK_REAL = 0, FK_HALO = 1, FK_VIRTUAL = 2 };

struct FusedSmem {
    unsigned char *base;
    FusedLayout L;
    int CAP;
    __device__ __forceinline__ double *sx(int s) const { return reinterpret_cast<double *>(base + s * L.stage_bytes); }
    __device__ __forceinline__ double *svx(int s) const { return sx(s) + CAP; }
    __device__ __forceinline__ double *svy(int s) const { return sx(s) + 2 * CAP; }
    __device__ __forceinline__ double *svz(int s) const { return sx(s) + 3 * CAP; }
    __device__ __forceinline__ double *sE(int s) const { return sx(s) + 4 * CAP; }
    __device__ __forceinline__ unsigned *code() const { return reinterpret_cast<unsigned *>(base + L.off_code); }
    __device__ __forceinline__ int *start() const { return reinterpret_cast<int *>(base + L.off_start); }
    __device__ __forceinline__ unsigned short *ps() const { return reinterpret_cast<unsigned short *>(base + L.off_ps); }
    __device__ __forceinline__ unsigned short *pe() const { return reinterpret_cast<unsigned short *>(base + L.off_pe); }
    __device__ __forceinline__ int *cnt() const { return reinterpret_cast<int *>(base + L.off_cnt); }
    __device__ __forceinline__ int *bas() const { return reinterpret_cast<int *>(base + L.off_base); }
    __device__ __forceinline__ double *q() const { return reinterpret_cast<double *>(base + L.off_q); }
    __device__ __forceinline__ int4 *items() const { return reinterpret_cast<int4 *>(base + L.off_items); }
    __device__ __forceinline__ int *kind() const { return reinterpret_cast<int *>(base + L.off_kind); }
    __device__ __forceinline__ unsigned mbar(int s) const { return smem_u32(base + L.off_mbar + 8 * s); }
};

// lane 0: start the bulk copies of one tile (item) into a stage
__device__ __forceinline__ void fused_issue(const FusedArgs &a, const FusedSmem &S, int4 it, int stage)
{
    const int cA = it.x, cB = it.y, sA = it.z, n = it.w - it.z;
    if (n <= 0) return;
    const int pad = sA & 1;
    const long long g0 = sA - pad;
    int cnt = round_up2(pad + n);
    bool tail = false;
    if (g0 + cnt > a.capacity) { cnt -= 2; tail = true; } // the array's last, odd, element
    const int ea = cA & ~1;
    const int ecount = round_up2(cB + 1 - ea);
    const unsigned mb = S.mbar(stage);
    const unsigned tx = 32u * (unsigned)cnt + 8u * (unsigned)ecount;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mb), "r"(tx) : "memory");
    if (cnt > 0) {
        const unsigned bytes = 8u * (unsigned)cnt;
        bulk_g2s(S.sx(stage), a.sx + g0, bytes, mb);
        bulk_g2s(S.svx(stage), a.svx + g0, bytes, mb);
        bulk_g2s(S.svy(stage), a.svy + g0, bytes, mb);
        bulk_g2s(S.svz(stage), a.svz + g0, bytes, mb);
    }
    bulk_g2s(S.sE(stage), a.E + ea, 8u * (unsigned)ecount, mb);
    if (tail) {
        const int li = pad + n - 1;
        const long long gi = (long long)sA + n - 1;
        S.sx(stage)[li] = a.sx[gi]; S.svx(stage)[li] = a.svx[gi]; S.svy(stage)[li] = a.svy[gi]; S.svz(stage)[li] = a.svz[gi];
    }
}

__device__ __forceinline__ int fused_table_fetch(const FusedArgs &a, int4 it, int idx)
{
    return idx <= it.y - it.x ? a.off_old[it.x + idx] : 0;
}

__global__ void __launch_bounds__(32) fused_kernel(FusedArgs a)
{
    extern __shared__ __align__(128) unsigned char fused_smem[];
    FusedSmem S;
    S.base = fused_smem;
    S.L = fused_layout(a.CAP, a.TPC);
    S.CAP = a.CAP;
    constexpr int K1 = FUSED_KMAX + 1; // row stride of the per-cell tables
    const int lane = threadIdx.x;
    const unsigned lt = (1u << lane) - 1u;
    DevState *st = a.st;
    const int nc = a.k.nc;
    int bad = 0; // FA_* bits
    int mc = 0;  // largest new per-cell count seen by this lane
    float vm2 = 0.f;
    int4 *items = S.items();
    int *kinds = S.kind();

    // ---- the chunk's work items: [halo cell] real tiles ... [halo cell | virtual end] --------------
    const int ntiles = st->ntiles;
    const int kA = blockIdx.x * a.TPC;
    bool active = kA < ntiles && !*(volatile int *)&st->abort;
    int nitems = 0;
    if (active) {
        const int kB = min(kA + a.TPC, ntiles);
        const int2 d0 = a.td_old[kA], dm = a.td_old[kB];
        const int cS = d0.x, cE = dm.x;
        if (cS >= cE) {
            active = false;
        } else {
            if (cS > 0) {
                if (lane == 0) {
                    items[0] = make_int4(cS - 1, cS, a.off_old[cS - 1], d0.y);
                    kinds[0] = FK_HALO;
                }
                nitems = 1;
            }
            for (int k0 = kA; k0 < kB; k0 += 32) {
                const int k = k0 + lane;
                int2 da = make_int2(0, 0), db = da;
                bool ne = false;
                if (k < kB) {
                    da = a.td_old[k];
                    db = a.td_old[k + 1];
                    ne = db.x > da.x;
                }
                const unsigned m = __ballot_sync(FULL, ne);
                if (ne) {
                    const int idx = nitems + __popc(m & lt);
                    items[idx] = make_int4(da.x, db.x, da.y, db.y);
                    kinds[idx] = FK_REAL;
                }
                nitems += __popc(m);
            }
            if (lane == 0) {
                if (cE < nc) {
                    items[nitems] = make_int4(cE, cE + 1, dm.y, a.off_old[cE + 1]);
                    kinds[nitems] = FK_HALO;
                } else {
                    items[nitems] = make_int4(nc, nc, dm.y, dm.y);
                    kinds[nitems] = FK_VIRTUAL;
                }
            }
            ++nitems;
            __syncwarp();
            for (int q = lane; q < nitems; q += 32) {
                const int4 I = items[q];
                if (round_up2((I.z & 1) + (I.w - I.z)) > a.CAP || I.y - I.x > FUSED_KMAX || I.w < I.z) bad |= FA_TILE_OVERFLOW;
            }
            if (__any_sync(FULL, bad != 0)) active = false;
        }
    }

    if (active) {
        if (lane == 0) {
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(S.mbar(0)) : "memory");
            asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(S.mbar(1)) : "memory");
            asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        }
        __syncwarp();
        const int OL = st->f_OL, AR = st->f_AR, shift = AR - OL;
        if (lane == 0) {
            fused_issue(a, S, items[0], 0);
            if (nitems > 1) fused_issue(a, S, items[1], 1);
        }
        int *start = S.start();
        unsigned short *ps = S.ps(), *pe = S.pe();
        int *cnt = S.cnt(), *bas = S.bas();
        unsigned *code = S.code();
        double *qx = S.q(), *qvx = qx + FUSED_DEF, *qvy = qx + 2 * FUSED_DEF, *qvz = qx + 3 * FUSED_DEF;
        int *qpos = reinterpret_cast<int *>(qx + 4 * FUSED_DEF);
        if (lane < 3) cnt[lane * K1] = 0;
        // carry across tiles: counts of the previous tile's last cell sit at table index 0
        int pvRR = 0;    // R of the cell before the carried one
        int pv_off = 0;  // off_old of the carried cell
        int pv_real = 0; // the carried cell belongs to this chunk (finalize it)
        int ndef = 0;    // deferred right-movers of the carried cell
        unsigned ph0 = 0, ph1 = 0;
        int4 itn = items[0];
        int t0 = fused_table_fetch(a, itn, lane), t1 = fused_table_fetch(a, itn, lane + 32);

        for (int it = 0; it < nitems; ++it) {
            const int stage = it & 1;
            const int4 I = itn;
            const int kind = kinds[it];
            const int cA = I.x, cB = I.y, sA = I.z, n = I.w - I.z, ncell = cB - cA, pad = sA & 1;
            if (lane <= ncell) start[lane] = t0 - sA + pad;
            if (lane + 32 <= ncell) start[lane + 32] = t1 - sA + pad;
            if (it + 1 < nitems) {
                itn = items[it + 1];
                t0 = fused_table_fetch(a, itn, lane);
                t1 = fused_table_fetch(a, itn, lane + 32);
            }
            __syncwarp();
            if (n > 0) {
                if (stage == 0) { mbar_wait(S.mbar(0), ph0); ph0 ^= 1u; }
                else            { mbar_wait(S.mbar(1), ph1); ph1 ^= 1u; }
            }
            double *px = S.sx(stage), *pvx = S.svx(stage), *pvy = S.svy(stage), *pvz = S.svz(stage);
            const double *pE = S.sE(stage);
            const int ea = cA & ~1;
            const int nrows = (pad + n + 31) >> 5;

            // ---- sweep 1: push in place, classify, prefix counts per class ------------------------
            int runL = 0, runS = 0, runR = 0;
            for (int r = 0; r < nrows; ++r) {
                const int i = (r << 5) + lane;
                int g = 3, cl = 0;
                bool first = false, last = false;
                if (i >= pad && i < pad + n) {
                    const double x = px[i], vx = pvx[i], vy = pvy[i], vz = pvz[i];
                    double xs, jf;
                    int j;
                    bool ok = gather_cell(a.k, x, xs, jf, j);
                    if (ok) {
                        const int c = j - cA;
                        ok = c >= 0 && c < ncell;
                        if (ok) {
                            const int s0 = start[c], s1 = start[c + 1];
                            ok = i >= s0 && i < s1;
                            if (ok) {
                                cl = c;
                                first = i == s0;
                                last = i == s1 - 1;
                                const double E0 = pE[j - ea], E1 = pE[j - ea + 1];
                                PushOut o;
                                push_core(a.k, x, vx, vy, vz, xs, jf, j, E0, E1, o);
                                int b = 0;
                                g = fused_classify(a.k, j, o, b);
                                if (b) { bad |= FA_BAD_PARTICLE; g = 3; }
                                px[i] = o.x; pvx[i] = o.vx; pvy[i] = o.vy; pvz[i] = o.vz;
                                vm2 = fmaxf(vm2, __double2float_ru(o.vx * o.vx + o.vy * o.vy + o.vz * o.vz));
                            }
                        }
                    }
                    if (!ok) bad |= FA_BAD_PARTICLE;
                }
                const unsigned mL = __ballot_sync(FULL, g == 0), mS = __ballot_sync(FULL, g == 1), mR = __ballot_sync(FULL, g == 2);
                const int bL = runL + __popc(mL & lt), bS = runS + __popc(mS & lt), bR = runR + __popc(mR & lt);
                if (first) {
                    ps[cl] = (unsigned short)bL; ps[K1 + cl] = (unsigned short)bS; ps[2 * K1 + cl] = (unsigned short)bR;
                }
                if (last) {
                    pe[cl] = (unsigned short)(bL + (g == 0)); pe[K1 + cl] = (unsigned short)(bS + (g == 1));
                    pe[2 * K1 + cl] = (unsigned short)(bR + (g == 2));
                }
                const int mine = g == 0 ? bL : (g == 1 ? bS : bR);
                code[i] = (unsigned)g | ((unsigned)cl << 2) | ((unsigned)mine << 8);
                runL += __popc(mL); runS += __popc(mS); runR += __popc(mR);
            }
            __syncwarp();

            // ---- per-cell phase: counts -> table index cl+1 -----------------------------------------
            if (kind == FK_VIRTUAL) {
                if (lane < 3) cnt[lane * K1 + 1] = 0;
            } else {
                for (int cl = lane; cl < ncell; cl += 32) {
                    const bool ne = start[cl + 1] > start[cl];
                    cnt[cl + 1] = ne ? (int)pe[cl] - (int)ps[cl] : 0;
                    cnt[K1 + cl + 1] = ne ? (int)pe[K1 + cl] - (int)ps[K1 + cl] : 0;
                    cnt[2 * K1 + cl + 1] = ne ? (int)pe[2 * K1 + cl] - (int)ps[2 * K1 + cl] : 0;
                }
            }
            __syncwarp();
            // destination bases of this tile's cells:  slot = base[class][cl] + prefix count
            if (kind == FK_REAL) {
                for (int cl = lane; cl < ncell; cl += 32) {
                    const int c = cA + cl, t = cl + 1;
                    const int oo = sA + start[cl] - pad, oo1 = sA + start[cl + 1] - pad;
                    const int Lc = cnt[t], Rc = cnt[2 * K1 + t], Rm1 = cnt[2 * K1 + t - 1];
                    const int Lp1 = cl < ncell - 1 ? cnt[t + 1] : 0; // last cell: added when the next tile knows it
                    const int pre_c = (a.k.periodic && c == nc - 1) ? OL : 0;
                    const int pre_c1 = (a.k.periodic && c + 1 == nc - 1) ? OL : 0;
                    bas[cl] = oo + (c == 1 ? -OL : shift) - Rm1 - (int)ps[cl];
                    bas[K1 + cl] = oo + (c >= 1 ? shift : 0) + Lc + pre_c - (int)ps[K1 + cl];
                    bas[2 * K1 + cl] = oo1 + shift - Rc + Lp1 + pre_c1 - (int)ps[2 * K1 + cl];
                }
            }
            // finalize cells cA-1 .. cB-2 (table index 0 .. ncell-1): count, offset, next partition
            {
                const int nfin = kind == FK_REAL ? ncell : 1;
                for (int t = lane; t < nfin; t += 32) {
                    if (t == 0 && !pv_real) continue;
                    const int c = cA - 1 + t;
                    const int Rm1 = t == 0 ? pvRR : cnt[2 * K1 + t - 1];
                    const int Lc = cnt[t], Sc = cnt[K1 + t], Lp1 = cnt[t + 1];
                    const int oo = t == 0 ? pv_off : sA + start[t - 1] - pad;
                    const int pre_c = (a.k.periodic && c == nc - 1) ? OL : 0;
                    const int post_c = c == 0 ? AR : 0;
                    const int cn = pre_c + Rm1 + Sc + Lp1 + post_c;
                    const int o0 = c == 0 ? 0 : oo + shift - Rm1 + Lc;
                    const int o1 = o0 + cn;
                    a.count_new[c] = cn;
                    a.off_new[c] = o0;
                    mc = max(mc, cn);
                    for (int kb = o0 / a.T + 1; kb <= o1 / a.T; ++kb)
                        if (kb < a.td_cap) a.td_new[kb] = make_int2(c + 1, o1);
                    if (c == 0) a.td_new[0] = make_int2(0, 0);
                    if (c == nc - 1) {
                        a.off_new[nc] = o1;
                        const int nt = o1 / a.T + 1;
                        if (nt < a.td_cap) a.td_new[nt] = make_int2(nc, o1);
                        st->ntiles_next = nt;
                    }
                }
            }
            // right-movers of the previous tile's last cell: their cell is cA, its L count is known now
            if (ndef) {
                if (lane < ndef) {
                    const long long p = (long long)qpos[lane] + cnt[1];
                    if (p < 0 || p >= a.capacity) bad |= FA_BAD_PARTICLE;
                    else {
                        a.dx[p] = qx[lane]; a.dvx[p] = qvx[lane]; a.dvy[p] = qvy[lane]; a.dvz[p] = qvz[lane];
                        a.dcell[p] = cA;
                    }
                }
                ndef = 0;
            }
            __syncwarp();

            // ---- sweep 2: every particle straight to its final slot ---------------------------------
            if (kind == FK_REAL) {
                for (int r = 0; r < nrows; ++r) {
                    const int i = (r << 5) + lane;
                    bool defer = false, store = false;
                    long long p = 0;
                    int cl = 0, g = 3;
                    if (i >= pad && i < pad + n) {
                        const unsigned cd = code[i];
                        g = (int)(cd & 3u);
                        if (g < 3) {
                            cl = (int)((cd >> 2) & 63u);
                            p = (long long)bas[g * K1 + cl] + (int)(cd >> 8);
                            defer = g == 2 && cl == ncell - 1;
                            store = !defer;
                        }
                    }
                    const unsigned md = __ballot_sync(FULL, defer);
                    if (store) {
                        if (p < 0 || p >= a.capacity) bad |= FA_BAD_PARTICLE;
                        else {
                            a.dx[p] = px[i]; a.dvx[p] = pvx[i]; a.dvy[p] = pvy[i]; a.dvz[p] = pvz[i];
                            a.dcell[p] = cA + cl + g - 1;
                        }
                    }
                    if (md) {
                        if (defer) {
                            const int q = ndef + __popc(md & lt);
                            if (q < FUSED_DEF) {
                                qx[q] = px[i]; qvx[q] = pvx[i]; qvy[q] = pvy[i]; qvz[q] = pvz[i];
                                qpos[q] = (int)p;
                            } else bad |= FA_DEFER_OVERFLOW;
                        }
                        ndef = min(ndef + __popc(md), FUSED_DEF);
                    }
                }
            }
            // carry: this tile's last cell becomes table index 0
            if (kind != FK_VIRTUAL) {
                const int nRR = cnt[2 * K1 + ncell - 1];
                const int cL_ = cnt[ncell], cS_ = cnt[K1 + ncell], cR_ = cnt[2 * K1 + ncell];
                const int po = sA + start[ncell - 1] - pad;
                __syncwarp();
                if (lane == 0) { cnt[0] = cL_; cnt[K1] = cS_; cnt[2 * K1] = cR_; }
                pvRR = nRR;
                pv_off = po;
                pv_real = kind == FK_REAL;
            }
            // refill this stage with the tile after next (generic writes above -> async proxy)
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            __syncwarp();
            if (lane == 0 && it + 2 < nitems) fused_issue(a, S, items[it + 2], stage);
        }
    }

    // ---- CTA epilogue; the last CTA commits or rolls back the step ----------------------------------
    bad = (int)__reduce_or_sync(FULL, (unsigned)bad);
    mc = __reduce_max_sync(FULL, mc);
    const unsigned vmw = __reduce_max_sync(FULL, __float_as_uint(vm2));
    if (lane == 0) {
        if (bad) {
            atomicExch(&st->abort, 1);
            atomicOr(&st->abort_reason, bad);
        }
        if (vmw > *(volatile unsigned *)&st->vmax2_next) atomicMax(&st->vmax2_next, vmw);
        if (mc > *(volatile int *)&st->maxcount_next) atomicMax(&st->maxcount_next, mc);
        __threadfence();
        const unsigned d = atomicAdd(&st->done, 1u);
        if (d == gridDim.x - 1u) {
            __threadfence();
            if (!*(volatile int *)&st->abort) {
                st->n = *(volatile int *)&st->n_next;
                st->wall[0] += *(volatile unsigned long long *)&st->wall_pend[0];
                st->wall[1] += *(volatile unsigned long long *)&st->wall_pend[1];
                st->vmax2 = *(volatile unsigned *)&st->vmax2_next;
                st->ntiles = *(volatile int *)&st->ntiles_next;
                st->maxcount = *(volatile int *)&st->maxcount_next;
                st->w_acc = 0;
                st->step_max = 0;
                st->need_general = 0;
                st->used_general = 0;
                st->run_split = 0;
            } else {
                st->run_split = 1;
                st->fused_disabled = 1;
            }
            st->n_next = 0;
            st->wall_pend[0] = st->wall_pend[1] = 0;
            st->vmax2_next = 0;
            st->maxcount_next = 0;
            st->done = 0;
            st->abort = 0;
        }
    }
}

// Tile partition of an offset array: td[k] = (first cell whose offset is >= k*T, that offset), for
// k = 0 .. ntiles with ntiles = n/T + 1 and td[ntiles] = (nc, n).  One thread per cell c settles
// cell c+1.  Used at pic_create and after every arrange of the split path; a fused step writes the
// next partition itself.
__global__ void bounds_kernel(const int *__restrict__ off, int nc, int T, int2 *__restrict__ td, int td_cap, DevState *st,
                              const int *guard)
{
    if (guard && !*guard) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    int cn = 0;
    if (c < nc) {
        const int o0 = off[c], o1 = off[c + 1];
        cn = o1 - o0;
        for (int kb = o0 / T + 1; kb <= o1 / T; ++kb)
            if (kb < td_cap) td[kb] = make_int2(c + 1, o1);
        if (c == 0) td[0] = make_int2(0, 0);
        if (c + 1 == nc) {
            const int nt = o1 / T + 1;
            if (nt < td_cap) td[nt] = make_int2(nc, o1);
            st->ntiles = nt;
        }
    }
    cn = __reduce_max_sync(FULL, cn);
    if ((threadIdx.x & 31) == 0 && cn > *(volatile int *)&st->maxcount) atomicMax(&st->maxcount, cn);
}

__global__ void zero_guarded_kernel(int *__restrict__ p, int n, const int *guard)
{
    if (guard && !*guard) return;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = 0;
}

} // namespace pic
