/*
 * oracle_omp.c -- the THREADED TWIN of the CPU oracle (oracle/oracle.c): the same mover and the
 * same arranger, run on all host cores with OpenMP.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT, exactly like oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it; it
 * shares no code, header, table or helper with the CUDA path under paper_2603_24508_b200/csrc/.
 *
 * Why it exists: "the same oracle source with `#pragma omp parallel
 * for` on the mover and a chunked (per-thread histogram -> scan across threads -> stable scatter)
 * arranger -- the design the paper itself used for `arrj`" ("Introducing OpenMP
 * thread parallelism to the arrj function"; PAPER.md:202 for the profile that motivates it).  It
 * is (a) the multi-core CPU baseline bench.py reports beside the single-thread oracle and (b) what
 * makes whole-run, element-by-element parity at BASELINE.json's full sizes affordable
 * (tests/test_gpu_fullsize.py).
 *
 * Authority: oracle.c stays the authority.  This file restates the arithmetic contract (SURVEY.md
 * section 8(c)) line by line -- every floating-point statement is ONE
 * IEEE-754 binary64 round-to-nearest-even operation, compiled with -ffp-contract=off -- and is
 * pinned BIT-IDENTICAL to oracle_push / oracle_arrange / oracle_run for 1, 2, 3 and nproc threads
 * (tests/test_oracle_omp.py, "-m not gpu"): the mover is independent per particle, and the stable
 * counting sort has a unique result, so neither depends on the number of threads.
 *
 *   mover    : particles split statically over the threads; wall counts by reduction.
 *   arranger : thread t owns the contiguous index range [n*t/T, n*(t+1)/T); it counts its range per
 *              cell (hist[t][c]); a scan over (cell, thread) turns the counts into the first slot of
 *              every (cell, thread) pair: offset[c] + sum_{t' < t} hist[t'][c]; each thread then
 *              walks its range in ascending order and copies particle i to first[t][cell_i]++.
 *              Lower threads hold lower indices, so equal cells keep their index order: stable.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

#define ORACLE_PERIODIC 0
#define ORACLE_ABSORBING 1

int oracle_omp_max_threads(void) { return omp_get_max_threads(); }

/* One mover step over slots [0,n): oracle_push (oracle.c) with the particle loop split over
 * `threads` OpenMP threads (0 = all).  Same return convention: 0, or -1 if any live particle's
 * gather cell is outside [0,nc-1] or differs from its stored cell (that particle is left
 * untouched; unlike the sequential oracle, particles behind it may already have been pushed). */
int oracle_omp_push(int64_t n, double *x, double *vx, double *vy, double *vz, int32_t *cell,
                    int32_t nc, double dx, double dt, int32_t boundary, const double *E,
                    double qm, const double *B, uint64_t *wall, int32_t threads)
{
    /* per-species constants (first block), one rounded operation per line */
    const double h = (qm * dt) * 0.5;
    const double tx = h * B[0];
    const double ty = h * B[1];
    const double tz = h * B[2];
    const double t2 = ((tx * tx) + (ty * ty)) + (tz * tz);
    const double f = 2.0 / (1.0 + t2);
    const double sx = f * tx;
    const double sy = f * ty;
    const double sz = f * tz;
    const double inv_dx = 1.0 / dx;
    const double L = (double)nc * dx;
    const int T = threads > 0 ? threads : omp_get_max_threads();
    uint64_t nleft = 0, nright = 0;
    int bad = 0;

#pragma omp parallel for num_threads(T) schedule(static) reduction(+ : nleft, nright) reduction(| : bad)
    for (int64_t i = 0; i < n; ++i) {
        if (cell[i] < 0)
            continue;
        /* (a-1) gather */
        double xs = x[i] * inv_dx;
        double jf = floor(xs);
        if (!(jf >= 0.0) || jf > (double)nc) {
            bad |= 1;
            continue;
        }
        int32_t j = (int32_t)jf;
        if (j > nc - 1) {
            j = nc - 1;
            jf = (double)j;
        }
        if (cell[i] != j) {
            bad |= 1;
            continue;
        }
        double w = xs - jf;
        double dE = E[j + 1] - E[j];
        double wdE = w * dE;
        double Ep = E[j] + wdE;
        /* (a-2) Boris */
        double hE = h * Ep;
        double ux = vx[i] + hE;
        double uy = vy[i];
        double uz = vz[i];
        double a1, a2;
        a1 = uy * tz; a2 = uz * ty; double px = ux + (a1 - a2);
        a1 = uz * tx; a2 = ux * tz; double py = uy + (a1 - a2);
        a1 = ux * ty; a2 = uy * tx; double pz = uz + (a1 - a2);
        a1 = py * sz; a2 = pz * sy; double wx = ux + (a1 - a2);
        a1 = pz * sx; a2 = px * sz; double wy = uy + (a1 - a2);
        a1 = px * sy; a2 = py * sx; double wz = uz + (a1 - a2);
        double nvx = wx + hE;
        /* (a-3) position advance */
        double dxp = nvx * dt;
        double xn = x[i] + dxp;
        /* (a-4) boundary and new cell */
        int dead = 0;
        if (boundary == ORACLE_PERIODIC) {
            if (xn >= L) {
                xn = xn - L;
            } else if (xn < 0.0) {
                xn = xn + L;
                if (xn >= L)
                    xn = 0.0;
            }
        } else {
            if (xn < 0.0) {
                dead = 1;
                nleft += 1;
            } else if (xn >= L) {
                dead = 1;
                nright += 1;
            }
        }
        int32_t cn = -1;
        if (!dead) {
            double cf = floor(xn * inv_dx);
            cn = (int32_t)cf;
            if (cn > nc - 1)
                cn = nc - 1;
        }
        x[i] = xn;
        vx[i] = nvx;
        vy[i] = wy;
        vz[i] = wz;
        cell[i] = cn;
    }
    wall[0] += nleft;
    wall[1] += nright;
    return bad ? -1 : 0;
}

/* Arranger: oracle_arrange (oracle.c) as a chunked counting sort.  Same outputs: count[nc],
 * offset[nc+1], the five arranged arrays; returns n_live or -1. */
int64_t oracle_omp_arrange(int64_t n, const double *x, const double *vx, const double *vy,
                           const double *vz, const int32_t *cell, double *xo, double *vxo,
                           double *vyo, double *vzo, int32_t *cello, int32_t nc,
                           int32_t *count, int32_t *offset, int32_t threads)
{
    int T = threads > 0 ? threads : omp_get_max_threads();
    if (T < 1) T = 1;
    /* hist[t*nc + c]: particles of cell c in thread t's index range; then their first slot */
    int32_t *hist = (int32_t *)calloc((size_t)T * (size_t)nc + 1, sizeof(int32_t));
    if (!hist)
        return -1;
    int bad = 0;

#pragma omp parallel num_threads(T) reduction(| : bad)
    {
        const int t = omp_get_thread_num();
        const int nt = omp_get_num_threads(); /* == T unless the runtime gave fewer */
        if (nt != T) {
            bad |= 2;
        } else {
            const int64_t i0 = n * t / T, i1 = n * (t + 1) / T;
            int32_t *h = hist + (size_t)t * (size_t)nc;
            for (int64_t i = i0; i < i1; ++i) {
                const int32_t c = cell[i];
                if (c < 0)
                    continue;
                if (c >= nc) {
                    bad |= 1;
                    continue;
                }
                h[c] += 1;
            }
        }
    }
    if (bad) {
        free(hist);
        if (bad & 2) /* fewer threads than asked for: fall back to one chunk, still the same result */
            return oracle_omp_arrange(n, x, vx, vy, vz, cell, xo, vxo, vyo, vzo, cello, nc, count, offset, 1);
        return -1;
    }
    /* per-cell totals, then the exclusive prefix sum over cells (sequential, nc terms) */
#pragma omp parallel for num_threads(T) schedule(static)
    for (int32_t c = 0; c < nc; ++c) {
        int32_t s = 0;
        for (int t = 0; t < T; ++t)
            s += hist[(size_t)t * (size_t)nc + c];
        count[c] = s;
    }
    offset[0] = 0;
    for (int32_t c = 0; c < nc; ++c)
        offset[c + 1] = offset[c] + count[c];
    /* first slot of every (cell, thread) pair */
#pragma omp parallel for num_threads(T) schedule(static)
    for (int32_t c = 0; c < nc; ++c) {
        int32_t run = offset[c];
        for (int t = 0; t < T; ++t) {
            const size_t k = (size_t)t * (size_t)nc + c;
            const int32_t cnt = hist[k];
            hist[k] = run;
            run += cnt;
        }
    }
    /* stable scatter: every thread walks its own range in ascending index order */
#pragma omp parallel num_threads(T)
    {
        const int t = omp_get_thread_num();
        const int64_t i0 = n * t / T, i1 = n * (t + 1) / T;
        int32_t *first = hist + (size_t)t * (size_t)nc;
        for (int64_t i = i0; i < i1; ++i) {
            const int32_t c = cell[i];
            if (c < 0)
                continue;
            const int64_t d = (int64_t)first[c];
            first[c] += 1;
            xo[d] = x[i];
            vxo[d] = vx[i];
            vyo[d] = vy[i];
            vzo[d] = vz[i];
            cello[d] = c;
        }
    }
    free(hist);
    return (int64_t)offset[nc];
}

/* The time loop of oracle_run (oracle.c; SURVEY 8(c) "Step counter") on the threaded routines.
 * The two buffer sets are swapped after an arrange instead of copied; if an odd number of
 * arranges ran, the final state is copied back so that it is in (x, vx, vy, vz, cell) on return,
 * as with oracle_run. */
int oracle_omp_run(int32_t nsteps, int32_t arrange_every, int64_t *step_count, int64_t *n,
                   double *x, double *vx, double *vy, double *vz, int32_t *cell, double *tx_,
                   double *tvx, double *tvy, double *tvz, int32_t *tcell, int32_t nc, double dx,
                   double dt, int32_t boundary, const double *E, double qm, const double *B,
                   uint64_t *wall, int32_t *count, int32_t *offset, int32_t threads)
{
    double *a[4] = {x, vx, vy, vz}, *b[4] = {tx_, tvx, tvy, tvz};
    int32_t *ac = cell, *bc = tcell;
    int swapped = 0, rc = 0;
    for (int32_t s = 0; s < nsteps && !rc; ++s) {
        rc = oracle_omp_push(*n, a[0], a[1], a[2], a[3], ac, nc, dx, dt, boundary, E, qm, B, wall, threads);
        if (rc)
            break;
        *step_count += 1;
        if (arrange_every > 0 && (*step_count % arrange_every) == 0) {
            int64_t nl = oracle_omp_arrange(*n, a[0], a[1], a[2], a[3], ac, b[0], b[1], b[2], b[3], bc, nc,
                                            count, offset, threads);
            if (nl < 0) {
                rc = -2;
                break;
            }
            for (int k = 0; k < 4; ++k) {
                double *t = a[k];
                a[k] = b[k];
                b[k] = t;
            }
            int32_t *tc = ac;
            ac = bc;
            bc = tc;
            swapped ^= 1;
            *n = nl;
        }
    }
    if (swapped) { /* the state sits in the caller's second buffer set: copy it home */
        const size_t m = (size_t)*n;
        memcpy(x, a[0], m * sizeof(double));
        memcpy(vx, a[1], m * sizeof(double));
        memcpy(vy, a[2], m * sizeof(double));
        memcpy(vz, a[3], m * sizeof(double));
        memcpy(cell, ac, m * sizeof(int32_t));
    }
    return rc;
}
