// fused.cuh -- single-pass push + arrange: one kernel per step when every
// step is followed by an arrange.  ~68 B of DRAM traffic per particle instead of 144 B.
//
// The source state is grouped by cell (offsets off_old).  Block b owns the DESTINATION cells
// [bound[b], bound[b+1]) (bound[] cuts the particle array every ~T particles at cell borders and
// is produced by the previous arrange).  A particle moves at most W cells per step (W from the
// device-side speed bound, verified per particle), so everything landing in the owned cells
// comes from the source cells [c0-W, c1+W): a contiguous slot range (plus a wrapped range at the
// ends of a periodic grid).  The block
//   1. stages that window of x, vx, vy, vz and the E nodes it covers into shared memory with
//      TMA bulk copies (cp.async.bulk + mbarrier),
//   2. pushes every window particle in shared memory (halo particles are pushed redundantly),
//      keeps those landing in an owned cell, and ranks them with ballot/popc prefix counts per
//      displacement group delta = -2..2: because the window is sorted by source cell, the stable
//      position of a particle inside its destination cell is
//         (# kept from earlier source cells into that cell) + (its rank inside its (cell, delta) group),
//      both of which follow from the group prefix counts sampled at the source-cell borders,
//   3. gets the slot of its first owned cell from a decoupled look-back chain over the blocks'
//      kept counts (this IS the device-wide exclusive scan of the per-cell histogram, coarsened),
//   4. writes count[], offset[], the next bound[] and the particles, in destination order, with
//      coalesced stores.
// Absorbed particles are dropped here (compaction), wall counters by ballot/popc.
// Anything the block cannot handle (window larger than the shared-memory budget, W > 2, a
// particle violating the bound) aborts the whole step: the source buffers are untouched, and the
// guarded split kernels launched right behind (mover / scan / scatter) redo it.
#pragma once
#include "pic_device.cuh"

namespace pic {

constexpr int FUSED_THREADS = 512;
constexpr int FUSED_WARPS = FUSED_THREADS / 32;
constexpr int FUSED_CAP = 2560;  // window slots per block (shared-memory budget)
constexpr int FUSED_KMAX = 320;  // window cells per block
constexpr int FUSED_WMAX = 2;    // largest per-step displacement (cells) the fused step handles
constexpr int FUSED_G = 2 * FUSED_WMAX + 1;
constexpr int FUSED_MIN_NC = 16;
constexpr int FUSED_T_DEFAULT = 1792; // target owned particles per block

struct FusedArgs {
    const double *sx, *svx, *svy, *svz;
    double *dx, *dvx, *dvy, *dvz;
    int *dcell;
    const double *E;
    const int *off_old;   // nc+1
    const int *bound_old; // nb_cap+1
    int *count_new, *off_new, *bound_new;
    unsigned long long *chain; // one look-back word per block: epoch<<34 | flag<<32 | value
    DevState *st;
    PushConst k;
    double vkick;       // 2*|h|*max|E|: bound on the growth of |v| in one step
    long long capacity; // slots allocated in every source array
    int T, nblocks, nb_cap;
    unsigned epoch;
};

struct FusedSeg {
    int ls, len;     // first local slot, number of particles
    int ua, ub;      // unwrapped cell range [ua, ub)
    int ushift;      // unwrapped cell = real cell + ushift
    int gshift;      // local slot = global slot - gshift
    int ebase;       // E node r sits at s_E[r + ebase]
    int pad;
};

struct FusedShared {
    double x[FUSED_CAP], vx[FUSED_CAP], vy[FUSED_CAP], vz[FUSED_CAP];
    double E[FUSED_KMAX + 16];
    unsigned code[FUSED_CAP];
    union {
        struct { unsigned short ps[FUSED_KMAX * FUSED_G], pe[FUSED_KMAX * FUSED_G]; } smp;
        unsigned short perm[FUSED_CAP];
    } u;
    int start[FUSED_KMAX], end[FUSED_KMAX];
    int cb[FUSED_KMAX];
    short gt[FUSED_KMAX * FUSED_G];
    unsigned char ws[FUSED_KMAX], we[FUSED_KMAX];
    int wtot[FUSED_WARPS][FUSED_G], wbase[FUSED_WARPS][FUSED_G];
    int wsum[FUSED_WARPS];
    FusedSeg seg[3];
    unsigned long long mbar;
    int b, c0, c1, W, nown, KW, uA0, ntot, nseg, abort, base, kept;
    unsigned vmax;
    int wall[2];
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, unsigned bytes, unsigned long long *mbar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(mbar))
                 : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long *mbar, unsigned parity)
{
    unsigned done = 0;
    const unsigned addr = smem_u32(mbar);
    while (!done) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done)
                     : "r"(addr), "r"(parity)
                     : "memory");
    }
}

__device__ __forceinline__ int round_up2(int v) { return (v + 1) & ~1; }

// Thread 0: take a ticket, find the owned cells and the window, start the bulk copies.
__device__ __forceinline__ void fused_setup(const FusedArgs &a, FusedShared &s)
{
    DevState *st = a.st;
    s.abort = 0;
    s.base = 0;
    s.kept = 0;
    s.vmax = 0;
    s.wall[0] = s.wall[1] = 0;
    s.nseg = 0;
    s.ntot = 0;
    s.nown = 0;
    s.KW = 0;
    const int b = (int)atomicAdd(&st->ticket, 1u);
    s.b = b;
    if (*(volatile int *)&st->abort || *(volatile int *)&st->fused_disabled) { s.abort = 1; return; }
    const int nc = a.k.nc;
    const double vm = sqrt((double)__uint_as_float(*(volatile unsigned *)&st->vmax2));
    const double reach = (vm * (1.0 + 1e-6) + a.vkick) * a.k.dt * a.k.inv_dx;
    if (!(reach < (double)FUSED_WMAX)) { s.abort = 1; return; }
    int W = (int)ceil(reach + 1e-9);
    if (W < 1) W = 1;
    if (W > FUSED_WMAX) { s.abort = 1; return; }
    const int c0 = a.bound_old[b], c1 = a.bound_old[b + 1];
    s.c0 = c0; s.c1 = c1; s.W = W;
    const int nown = c1 - c0;
    s.nown = nown;
    if (nown <= 0) return;
    const int KW = nown + 2 * W;
    if (KW > FUSED_KMAX) { s.abort = 1; return; }
    s.KW = KW;
    const int uA0 = c0 - W, uEnd = c1 + W;
    s.uA0 = uA0;
    // up to three contiguous source ranges, in unwrapped cell order
    int ua[3], ub[3], sh[3], ns = 0;
    if (a.k.periodic) {
        if (uA0 < 0) { ua[ns] = uA0; ub[ns] = min(0, uEnd); sh[ns] = -nc; ++ns; }
        if (max(uA0, 0) < min(uEnd, nc)) { ua[ns] = max(uA0, 0); ub[ns] = min(uEnd, nc); sh[ns] = 0; ++ns; }
        if (uEnd > nc) { ua[ns] = max(nc, uA0); ub[ns] = uEnd; sh[ns] = nc; ++ns; }
    } else {
        ua[0] = max(uA0, 0); ub[0] = min(uEnd, nc); sh[0] = 0; ns = 1;
    }
    int lcur = 0, ecur = 0;
    unsigned tx = 0;
    for (int q = 0; q < ns; ++q) {
        const int ra = ua[q] - sh[q], rb = ub[q] - sh[q]; // real cells [ra, rb)
        const int g0 = a.off_old[ra], g1 = a.off_old[rb];
        FusedSeg &sg = s.seg[q];
        sg.ua = ua[q]; sg.ub = ub[q]; sg.ushift = sh[q];
        sg.len = g1 - g0;
        sg.ls = lcur + (g0 & 1);
        sg.gshift = g0 - sg.ls;
        const int span = round_up2((g0 & 1) + sg.len);
        if (lcur + span > FUSED_CAP) { s.abort = 1; return; }
        const int ea = ra & ~1, eb = round_up2(rb + 1);
        sg.ebase = ecur - ea;
        if (ecur + (eb - ea) > FUSED_KMAX + 16) { s.abort = 1; return; }
        lcur += span;
        ecur += eb - ea;
    }
    s.nseg = ns;
    s.ntot = lcur;
    // bulk copies: particle window (16-byte aligned on both sides by construction) and E nodes
    const unsigned mb = smem_u32(&s.mbar);
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;\n" ::"r"(mb) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    // first pass: byte count; second pass: issue
    int l0[3], cntq[3], tail[3];
    for (int q = 0; q < ns; ++q) {
        const FusedSeg &sg = s.seg[q];
        const int g0 = sg.gshift + sg.ls;
        l0[q] = sg.ls - (g0 & 1);
        cntq[q] = round_up2((g0 & 1) + sg.len);
        tail[q] = 0;
        if ((long long)(g0 & ~1) + cntq[q] > a.capacity) { cntq[q] -= 2; tail[q] = 1; } // last slot is the array's last, odd, element
        tx += 4u * 8u * (unsigned)cntq[q];
        const int ra = sg.ua - sg.ushift, rb = sg.ub - sg.ushift;
        tx += 8u * (unsigned)(round_up2(rb + 1) - (ra & ~1));
    }
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(mb), "r"(tx) : "memory");
    for (int q = 0; q < ns; ++q) {
        const FusedSeg &sg = s.seg[q];
        const long long gsrc = (long long)l0[q] + sg.gshift;
        const unsigned bytes = 8u * (unsigned)cntq[q];
        if (bytes) {
            bulk_g2s(&s.x[l0[q]], a.sx + gsrc, bytes, &s.mbar);
            bulk_g2s(&s.vx[l0[q]], a.svx + gsrc, bytes, &s.mbar);
            bulk_g2s(&s.vy[l0[q]], a.svy + gsrc, bytes, &s.mbar);
            bulk_g2s(&s.vz[l0[q]], a.svz + gsrc, bytes, &s.mbar);
        }
        if (tail[q]) {
            const int li = sg.ls + sg.len - 1;
            const long long gi = (long long)li + sg.gshift;
            s.x[li] = a.sx[gi]; s.vx[li] = a.svx[gi]; s.vy[li] = a.svy[gi]; s.vz[li] = a.svz[gi];
        }
        const int ra = sg.ua - sg.ushift, rb = sg.ub - sg.ushift;
        const int ea = ra & ~1, eb = round_up2(rb + 1);
        bulk_g2s(&s.E[ea + sg.ebase], a.E + ea, 8u * (unsigned)(eb - ea), &s.mbar);
    }
}

// Decoupled look-back over the blocks' kept counts (warp 0).  Returns the exclusive prefix, or
// -1 if a predecessor aborted.
__device__ __forceinline__ int fused_lookback(const FusedArgs &a, int b, int lane)
{
    volatile unsigned long long *ch = a.chain;
    const unsigned long long ep = (unsigned long long)(a.epoch & 0x3fffffffu);
    int prefix = 0;
    int idx = b - 1;
    while (idx >= 0) {
        const int my = idx - lane;
        unsigned long long w;
        unsigned flag;
        do {
            w = my >= 0 ? ch[my] : ((ep << 34) | (2ull << 32));
            flag = ((w >> 34) == ep) ? (unsigned)(w >> 32) & 3u : 0u;
        } while (__any_sync(FULL, flag == 0));
        if (__any_sync(FULL, flag == 3)) return -1;
        const unsigned incl_mask = __ballot_sync(FULL, flag == 2);
        const int val = (int)(unsigned)w;
        if (incl_mask) {
            const int first = __ffs(incl_mask) - 1;
            prefix += __reduce_add_sync(FULL, lane <= first ? val : 0);
            break;
        }
        prefix += __reduce_add_sync(FULL, val);
        idx -= 32;
    }
    return prefix;
}

__global__ void __launch_bounds__(FUSED_THREADS, 2) fused_kernel(FusedArgs a)
{
    extern __shared__ __align__(128) unsigned char fused_smem[];
    FusedShared &s = *reinterpret_cast<FusedShared *>(fused_smem);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned lt = (1u << lane) - 1u;
    DevState *st = a.st;
    const unsigned long long ep = (unsigned long long)(a.epoch & 0x3fffffffu);

    if (tid == 0) fused_setup(a, s);
    __syncthreads();
    const int b = s.b, W = s.W, nown = s.nown, KW = s.KW, uA0 = s.uA0, ntot = s.ntot, nseg = s.nseg;
    const int nc = a.k.nc;
    bool work = !s.abort && nown > 0;

    // ---- tables: local slot range of every window cell -------------------------------------
    if (work) {
        for (int v = tid; v < KW; v += FUSED_THREADS) {
            const int u = uA0 + v;
            int st0 = 0, en0 = 0;
            for (int q = 0; q < nseg; ++q) {
                const FusedSeg &sg = s.seg[q];
                if (u >= sg.ua && u < sg.ub) {
                    const int r = u - sg.ushift;
                    st0 = a.off_old[r] - sg.gshift;
                    en0 = a.off_old[r + 1] - sg.gshift;
                }
            }
            s.start[v] = st0;
            s.end[v] = en0;
        }
    }
    __syncthreads();

    // ---- sweep 1: push in shared memory, classify, group prefix counts -----------------------
    int run[FUSED_G];
#pragma unroll
    for (int g = 0; g < FUSED_G; ++g) run[g] = 0;
    const int nr = (ntot + 31) >> 5;
    const int rb = (warp * nr) / FUSED_WARPS, re = ((warp + 1) * nr) / FUSED_WARPS;
    if (work) {
        mbar_wait(&s.mbar, 0);
        int nleft = 0, nright = 0, bad = 0;
        float vm2 = 0.f;
        for (int r = rb; r < re; ++r) {
            const int i = (r << 5) + lane;
            int q = -1;
#pragma unroll
            for (int t = 0; t < 3; ++t)
                if (t < nseg && i >= s.seg[t].ls && i < s.seg[t].ls + s.seg[t].len) q = t;
            bool kept = false;
            int g = 0, vs = 0, vd = 0;
            bool first = false, last = false;
            if (q >= 0) {
                const FusedSeg &sg = s.seg[q];
                const double x = s.x[i], vx = s.vx[i], vy = s.vy[i], vz = s.vz[i];
                double xs, jf;
                int j;
                if (gather_cell(a.k, x, xs, jf, j)) {
                    vs = j + sg.ushift - uA0;
                    if (vs >= 0 && vs < KW && i >= s.start[vs] && i < s.end[vs]) {
                        first = i == s.start[vs];
                        last = i == s.end[vs] - 1;
                        const double E0 = s.E[j + sg.ebase], E1 = s.E[j + sg.ebase + 1];
                        PushOut o;
                        push_core(a.k, x, vx, vy, vz, xs, jf, j, E0, E1, o);
                        s.x[i] = o.x; s.vx[i] = o.vx; s.vy[i] = o.vy; s.vz[i] = o.vz;
                        vm2 = fmaxf(vm2, __double2float_ru(o.vx * o.vx + o.vy * o.vy + o.vz * o.vz));
                        const bool owned_src = vs >= W && vs < W + nown;
                        if (o.wall) {
                            if (owned_src) { nleft += (o.wall == 1); nright += (o.wall == 2); }
                        } else {
                            int d = o.cell - j;
                            if (a.k.periodic) {
                                if (d > (nc >> 1)) d -= nc;
                                else if (d < -(nc >> 1)) d += nc;
                            }
                            if (d > W || d < -W) bad = 1;
                            else {
                                vd = vs + d;
                                g = d + FUSED_WMAX;
                                kept = vd >= W && vd < W + nown;
                            }
                        }
                    } else bad = 1;
                } else bad = 1;
            }
            // group prefix counts of this round
            int pre = 0;
            int cntg[FUSED_G], beforeg[FUSED_G];
#pragma unroll
            for (int gg = 0; gg < FUSED_G; ++gg) {
                const unsigned m = __ballot_sync(FULL, kept && g == gg);
                beforeg[gg] = run[gg] + __popc(m & lt);
                cntg[gg] = __popc(m);
                if (g == gg) pre = beforeg[gg];
            }
            if (first) {
#pragma unroll
                for (int gg = 0; gg < FUSED_G; ++gg) s.u.smp.ps[vs * FUSED_G + gg] = (unsigned short)beforeg[gg];
                s.ws[vs] = (unsigned char)warp;
            }
            if (last) {
#pragma unroll
                for (int gg = 0; gg < FUSED_G; ++gg)
                    s.u.smp.pe[vs * FUSED_G + gg] = (unsigned short)(beforeg[gg] + ((kept && g == gg) ? 1 : 0));
                s.we[vs] = (unsigned char)warp;
            }
#pragma unroll
            for (int gg = 0; gg < FUSED_G; ++gg) run[gg] += cntg[gg];
            if (q >= 0) s.code[i] = kept ? (0x80000000u | ((unsigned)g << 24) | ((unsigned)vd << 12) | (unsigned)pre) : 0u;
        }
        if (lane == 0) {
#pragma unroll
            for (int gg = 0; gg < FUSED_G; ++gg) s.wtot[warp][gg] = run[gg];
        }
        // per-warp reductions: walls, speed bound, violations
        const unsigned any = __ballot_sync(FULL, (nleft | nright | bad) != 0);
        if (any) {
            const int l = __reduce_add_sync(FULL, nleft), rr = __reduce_add_sync(FULL, nright);
            const unsigned bb = __reduce_or_sync(FULL, (unsigned)bad);
            if (lane == 0) {
                if (l) atomicAdd(&s.wall[0], l);
                if (rr) atomicAdd(&s.wall[1], rr);
                if (bb) s.abort = 1;
            }
        }
        const unsigned vmw = __reduce_max_sync(FULL, __float_as_uint(vm2));
        if (lane == 0 && vmw) atomicMax(&s.vmax, vmw);
    }
    __syncthreads();
    work = work && !s.abort;

    // ---- warp 0: exclusive scan of the warps' group totals, publish the block's kept count ----
    if (warp == 0) {
        int kept_total = 0;
        if (work) {
#pragma unroll
            for (int gg = 0; gg < FUSED_G; ++gg) {
                const int v = lane < FUSED_WARPS ? s.wtot[lane][gg] : 0;
                int incl = v;
#pragma unroll
                for (int o = 1; o < FUSED_WARPS; o <<= 1) {
                    const int t = __shfl_up_sync(FULL, incl, o);
                    if (lane >= o) incl += t;
                }
                if (lane < FUSED_WARPS) s.wbase[lane][gg] = incl - v;
                kept_total += __shfl_sync(FULL, incl, FUSED_WARPS - 1);
            }
        }
        if (lane == 0) {
            s.kept = kept_total;
            const unsigned flag = s.abort ? 3u : (b == 0 ? 2u : 1u);
            if (s.abort) atomicExch(&st->abort, 1);
            *(volatile unsigned long long *)&a.chain[b] = (ep << 34) | ((unsigned long long)flag << 32) | (unsigned)kept_total;
        }
    }
    __syncthreads();

    // ---- warp 0: look-back; other warps: per-destination-cell group bases ---------------------
    int cell_cnt = 0; // particles landing in this thread's destination cell (thread tid-32 <-> cell c0+tid-32)
    if (warp == 0) {
        if (!s.abort && b > 0) {
            const int prefix = fused_lookback(a, b, lane);
            if (lane == 0) {
                if (prefix < 0) {
                    s.abort = 1;
                    *(volatile unsigned long long *)&a.chain[b] = (ep << 34) | (3ull << 32);
                } else {
                    s.base = prefix;
                    *(volatile unsigned long long *)&a.chain[b] = (ep << 34) | (2ull << 32) | (unsigned)(prefix + s.kept);
                }
            }
        }
    } else if (work) {
        const int t = tid - 32;
        int acc = 0;
        if (t < nown) {
            const int vd = W + t;
            // sources of this destination cell in ascending real-cell (= source slot) order:
            // unwrapped cells >= nc first (they wrapped to the low end), then in-range, then < 0
#pragma unroll
            for (int cls = 0; cls < 3; ++cls) {
                for (int v = vd - W; v <= vd + W; ++v) {
                    const int u = uA0 + v;
                    const int c = a.k.periodic ? (u >= nc ? 0 : (u >= 0 ? 1 : 2)) : 1;
                    if (c != cls) continue;
                    const int gg = vd - v + FUSED_WMAX;
                    int M = 0, psabs = 0;
                    if (s.end[v] > s.start[v]) {
                        psabs = (int)s.u.smp.ps[v * FUSED_G + gg] + s.wbase[s.ws[v]][gg];
                        M = (int)s.u.smp.pe[v * FUSED_G + gg] + s.wbase[s.we[v]][gg] - psabs;
                    }
                    s.gt[vd * FUSED_G + gg] = (short)(acc - psabs);
                    acc += M;
                }
            }
        }
        cell_cnt = acc;
        // inclusive warp scan of the per-cell counts (warps 1.. hold the cells)
        int incl = acc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += v;
        }
        if (t < nown) s.cb[t] = incl - acc;
        if (lane == 31) s.wsum[warp] = incl;
    }
    __syncthreads();
    work = work && !s.abort;
    const int base = s.base;

    if (work) {
        // finish the block-wide exclusive scan of the per-cell counts
        if (tid >= 32 && tid - 32 < nown) {
            const int t = tid - 32;
            int add = 0;
            for (int w = 1; w < warp; ++w) add += s.wsum[w];
            const int cb = s.cb[t] + add;
            s.cb[t] = cb;
            const int cnt = cell_cnt;
            const int c = s.c0 + t;
            const int o0 = base + cb, o1 = o0 + cnt;
            a.count_new[c] = cnt;
            a.off_new[c] = o0;
            // next partition: bound[k] = first cell whose offset >= k*T; this thread settles cell c+1
            for (int kb = o0 / a.T + 1; kb <= o1 / a.T; ++kb)
                if (kb <= a.nb_cap) a.bound_new[kb] = c + 1;
            if (c == 0) a.bound_new[0] = 0;
            if (c + 1 == nc) {
                a.off_new[nc] = o1;
                for (int kb = o1 / a.T + 1; kb <= a.nb_cap; ++kb) a.bound_new[kb] = nc;
            }
        }
    }
    __syncthreads();

    // ---- sweep 2: destination slot of every kept particle -> inverse permutation --------------
    if (work) {
        for (int r = rb; r < re; ++r) {
            const int i = (r << 5) + lane;
            if (i < ntot) {
                bool in = false;
#pragma unroll
                for (int t = 0; t < 3; ++t)
                    if (t < nseg && i >= s.seg[t].ls && i < s.seg[t].ls + s.seg[t].len) in = true;
                if (in) {
                    const unsigned code = s.code[i];
                    if (code & 0x80000000u) {
                        const int g = (code >> 24) & 7, vd = (code >> 12) & 0xfff, pre = code & 0xfff;
                        const int d = s.cb[vd - W] + (int)s.gt[vd * FUSED_G + g] + s.wbase[warp][g] + pre;
                        s.u.perm[d] = (unsigned short)i;
                    }
                }
            }
        }
    }
    __syncthreads();

    // ---- sweep 3: coalesced stores in destination order ------------------------------------------
    if (work) {
        const int kept = s.kept;
        for (int k = tid; k < kept; k += FUSED_THREADS) {
            const int i = s.u.perm[k];
            const int vd = (s.code[i] >> 12) & 0xfff;
            int c = uA0 + vd;
            const long long gi = (long long)base + k;
            a.dx[gi] = s.x[i];
            a.dvx[gi] = s.vx[i];
            a.dvy[gi] = s.vy[i];
            a.dvz[gi] = s.vz[i];
            a.dcell[gi] = c;
        }
    }

    // ---- block epilogue; the last block commits or rolls back the step ------------------------------
    if (tid == 0) {
        if (work) {
            if (s.wall[0]) atomicAdd(&st->wall_pend[0], (unsigned long long)s.wall[0]);
            if (s.wall[1]) atomicAdd(&st->wall_pend[1], (unsigned long long)s.wall[1]);
            if (s.vmax) atomicMax(&st->vmax2_next, s.vmax);
            if (s.kept) atomicAdd(&st->n_next, s.kept);
        }
        __threadfence();
        const unsigned d = atomicAdd(&st->done, 1u);
        if (d == (unsigned)a.nblocks - 1u) {
            __threadfence();
            const int ab = *(volatile int *)&st->abort;
            if (!ab) {
                st->n = *(volatile int *)&st->n_next;
                st->wall[0] += *(volatile unsigned long long *)&st->wall_pend[0];
                st->wall[1] += *(volatile unsigned long long *)&st->wall_pend[1];
                st->vmax2 = *(volatile unsigned *)&st->vmax2_next;
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
            st->ticket = 0;
            st->done = 0;
            st->abort = 0;
        }
    }
}

// bound[k] = first cell whose offset is >= k*T (k = 0..nb_cap), from an offset array.  One thread
// per cell c settles cell c+1.  Used at pic_create and after every arrange of the split path.
__global__ void bounds_kernel(const int *__restrict__ off, int nc, int T, int *__restrict__ bound, int nb_cap,
                              const int *guard)
{
    if (guard && !*guard) return;
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= nc) return;
    const int o0 = off[c], o1 = off[c + 1];
    for (int kb = o0 / T + 1; kb <= o1 / T; ++kb)
        if (kb <= nb_cap) bound[kb] = c + 1;
    if (c == 0) bound[0] = 0;
    if (c + 1 == nc)
        for (int kb = o1 / T + 1; kb <= nb_cap; ++kb) bound[kb] = nc;
}

__global__ void zero_guarded_kernel(int *__restrict__ p, int n, const int *guard)
{
    if (guard && !*guard) return;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = 0;
}

} // namespace pic
