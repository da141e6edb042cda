/*
 * oracle.c -- plain, slow, obviously-correct CPU oracle for the BIT1-style particle
 * mover, arranger and charge deposition (the grey box of Fig. 1; phases (i)+(iv) of the PIC
 * cycle; `move0`/`moveb`, `arrj`, `rempar2`).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path under paper_2603_24508_b200/csrc/.
 *
 * The paper prints no equations for either routine (PAPER.md:89 names them only); the
 * concrete scheme is BASELINE.json's north_star (linear / cloud-in-cell gather of E_x,
 * Boris update in a uniform tilted B, x advance, absorbing-wall flag; stable per-cell
 * counting sort + compaction) in the operation order fixed by SURVEY.md section 8(c)
 * ("the arithmetic contract") and restated in DESIGN.md section 3.  Every floating
 * point statement below is ONE IEEE-754 binary64 round-to-nearest-even operation; the
 * file must be compiled with -ffp-contract=off (oracle/build.py does) so that no
 * multiply-add is fused.  Single thread, no blocking, no reordering.
 *
 * Parity pins (tests/test_oracle_*.py, all "-m not gpu"):
 *   oracle_boris_constants, oracle_push : P1 |v| conservation, P2 rotation angle
 *       2*atan(|t|) and sense, P3 constant acceleration closed form, P4 ExB fixed point,
 *       P5 implicit Boris identity, P6 theta=0 == unmagnetised leap-frog, P7 hex worked
 *       example (tests/golden/boris_worked_example.txt), P8 Rodrigues-rotation brute
 *       force in extended precision, gather vs numpy.interp, wall/wrap edge cases.
 *   oracle_arrange : P8 O(N^2) rank brute force and numpy stable argsort, P9 count /
 *       offset invariants, P10 idempotence, the tiny printed pin of SURVEY 8(c).
 *   oracle_deposit : single particle (exact 3/4, 1/4), total charge, first moment, one particle
 *       per cell centre, periodic fold, linearity, numpy add.at brute force, clamp (S8)
 *       (tests/test_oracle_deposit.py).
 *   Parity with BIT1's own output is UNPINNED (no code, no printed values in the paper).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_PERIODIC 0
#define ORACLE_ABSORBING 1

/* Per-species Boris constants, computed once on the host (first block):
 *   h = (qm*dt)*0.5;  t = h*B;  t2 = ((tx*tx)+(ty*ty))+(tz*tz);  f = 2/(1+t2);  s = f*t
 * t = (q/m) B dt/2 WITHOUT the tan() correction (reading S1; pinned by P2).
 * out[0..7] = h, tx, ty, tz, sx, sy, sz, inv_dx. */
void oracle_boris_constants(double qm, double dt, double dx, const double *B, double *out)
{
    double h = (qm * dt) * 0.5;
    double tx = h * B[0];
    double ty = h * B[1];
    double tz = h * B[2];
    double t2 = ((tx * tx) + (ty * ty)) + (tz * tz);
    double f = 2.0 / (1.0 + t2);
    out[0] = h;
    out[1] = tx;
    out[2] = ty;
    out[3] = tz;
    out[4] = f * tx;
    out[5] = f * ty;
    out[6] = f * tz;
    out[7] = 1.0 / dx;
}

/* One mover step over slots [0,n) (north_star: gather, Boris, x advance, wall flag).
 * Dead particles (cell < 0) are skipped and keep their final x', v'.
 * E has nc+1 node values, node j at x_j = j*dx.  wall[0] += absorbed at x<0,
 * wall[1] += absorbed at x>=L (half-open domain [0,L), reading S6).
 * Returns 0, or -1 if a live particle's gather cell falls outside [0,nc-1]
 * (precondition 0 <= x < L violated) or differs from its stored cell index (SURVEY 8(c):
 * "j == cell by invariant (oracle asserts)" -- a harness that hands over a stale cell array is
 * caught here; the state is left as it was up to that particle). */
int oracle_push(int64_t n, double *x, double *vx, double *vy, double *vz, int32_t *cell,
                int32_t nc, double dx, double dt, int32_t boundary, const double *E,
                double qm, const double *B, uint64_t *wall)
{
    double k[8];
    oracle_boris_constants(qm, dt, dx, B, k);
    const double h = k[0], tx = k[1], ty = k[2], tz = k[3];
    const double sx = k[4], sy = k[5], sz = k[6], inv_dx = k[7];
    const double L = (double)nc * dx;

    for (int64_t i = 0; i < n; ++i) {
        if (cell[i] < 0)
            continue;
        /* (a-1) field gather, linear weighting: E_p = E[j] + w*(E[j+1]-E[j])   (S5) */
        double xs = x[i] * inv_dx;
        double jf = floor(xs);
        if (!(jf >= 0.0) || jf > (double)nc)
            return -1;
        int32_t j = (int32_t)jf;
        if (j > nc - 1) { /* x*inv_dx rounded up to nc although x < L (dx != 1 only, S8) */
            j = nc - 1;
            jf = (double)j;
        }
        if (cell[i] != j)
            return -1; /* invariant cell == min(floor(x/dx), nc-1) broken */
        double w = xs - jf;
        double dE = E[j + 1] - E[j];
        double wdE = w * dE;
        double Ep = E[j] + wdE;
        /* (a-2) Boris: half kick, rotate by t then s, half kick; E = (Ex,0,0) */
        double hE = h * Ep;
        double ux = vx[i] + hE;
        double uy = vy[i];
        double uz = vz[i];
        double a1, a2;
        a1 = uy * tz; a2 = uz * ty; double px = ux + (a1 - a2);   /* v' = v- + v- x t */
        a1 = uz * tx; a2 = ux * tz; double py = uy + (a1 - a2);
        a1 = ux * ty; a2 = uy * tx; double pz = uz + (a1 - a2);
        a1 = py * sz; a2 = pz * sy; double wx = ux + (a1 - a2);   /* v+ = v- + v' x s */
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
                    xn = 0.0; /* tiny negative x' rounds to L: L == 0 on a ring (S7) */
            }
        } else {
            if (xn < 0.0) {
                dead = 1;
                wall[0] += 1;
            } else if (xn >= L) {
                dead = 1;
                wall[1] += 1;
            }
        }
        int32_t cn = -1;
        if (!dead) {
            double cf = floor(xn * inv_dx);
            cn = (int32_t)cf;
            if (cn > nc - 1)
                cn = nc - 1; /* S8 */
        }
        x[i] = xn;
        vx[i] = nvx;
        vy[i] = wy;
        vz[i] = wz;
        cell[i] = cn;
    }
    return 0;
}

/* Arranger: the stable sort of the live particles by cell, written out as a counting
 * sort (north_star; `arrj` "a sorting function" PAPER.md:200; natural sorting = grouped
 * per cell with counts np[species][cell]; `rempar2` removal
 * PAPER.md:202).  count[nc], offset[nc+1] (exclusive prefix, offset[nc] = n_live).
 * Particle i (ascending) with cell >= 0 goes to slot offset[cell] + next[cell]++.
 * Returns n_live, or -1 on a cell index >= nc / allocation failure. */
int64_t oracle_arrange(int64_t n, const double *x, const double *vx, const double *vy,
                       const double *vz, const int32_t *cell, double *xo, double *vxo,
                       double *vyo, double *vzo, int32_t *cello, int32_t nc,
                       int32_t *count, int32_t *offset)
{
    int64_t *next = (int64_t *)calloc((size_t)nc + 1, sizeof(int64_t));
    if (!next)
        return -1;
    for (int32_t c = 0; c < nc; ++c)
        count[c] = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (cell[i] < 0)
            continue;
        if (cell[i] >= nc) {
            free(next);
            return -1;
        }
        count[cell[i]] += 1;
    }
    offset[0] = 0;
    for (int32_t c = 0; c < nc; ++c)
        offset[c + 1] = offset[c] + count[c];
    for (int64_t i = 0; i < n; ++i) {
        int32_t c = cell[i];
        if (c < 0)
            continue;
        int64_t d = (int64_t)offset[c] + next[c];
        next[c] += 1;
        xo[d] = x[i];
        vxo[d] = vx[i];
        vyo[d] = vy[i];
        vzo[d] = vz[i];
        cello[d] = c;
    }
    free(next);
    return (int64_t)offset[nc];
}

/* The time loop the library's pic_push implements (SURVEY 8(c) "Step counter"): each
 * mover step increments *step_count; with arrange_every = k > 0 an arrange runs right
 * after every step whose new count is a multiple of k.  buf[0..4] are the five arrays
 * of the state, tmp[0..4] a second set of the same capacity; on return the state is in
 * buf (copied back after each arrange, keeping this loop free of pointer juggling).
 * *n is updated to n_live after each arrange.  Returns 0 or a negative error. */
int oracle_run(int32_t nsteps, int32_t arrange_every, int64_t *step_count, int64_t *n,
               double *x, double *vx, double *vy, double *vz, int32_t *cell, double *tx_,
               double *tvx, double *tvy, double *tvz, int32_t *tcell, int32_t nc, double dx,
               double dt, int32_t boundary, const double *E, double qm, const double *B,
               uint64_t *wall, int32_t *count, int32_t *offset)
{
    for (int32_t s = 0; s < nsteps; ++s) {
        int rc = oracle_push(*n, x, vx, vy, vz, cell, nc, dx, dt, boundary, E, qm, B, wall);
        if (rc)
            return rc;
        *step_count += 1;
        if (arrange_every > 0 && (*step_count % arrange_every) == 0) {
            int64_t nl = oracle_arrange(*n, x, vx, vy, vz, cell, tx_, tvx, tvy, tvz, tcell,
                                        nc, count, offset);
            if (nl < 0)
                return -2;
            memcpy(x, tx_, (size_t)nl * sizeof(double));
            memcpy(vx, tvx, (size_t)nl * sizeof(double));
            memcpy(vy, tvy, (size_t)nl * sizeof(double));
            memcpy(vz, tvz, (size_t)nl * sizeof(double));
            memcpy(cell, tcell, (size_t)nl * sizeof(int32_t));
            *n = nl;
        }
    }
    return 0;
}

/* Charge deposition, phase (ii) of the PIC cycle ("deposition to the grid, which maps particle
 * charges and currents to the mesh"), with the same linear (cloud-in-cell) weighting
 * as the gather (BASELINE.json north_star).  The paper prints no
 * formula; the reading (S20-S22): node j of nc+1 nodes receives
 *     rho[j] = weight * ( sum over live particles in cell j   of (1 - w_i)
 *                       + sum over live particles in cell j-1 of  w_i     ),
 * with xs = x*inv_dx, jf = floor(xs) (clamped to nc-1 as in the mover, reading S8), w = xs - jf;
 * `weight` (charge per macro-particle over dx, sign included) is the caller's business; on a
 * periodic grid nodes 0 and nc are the same point and both carry the sum of the two; at
 * absorbing walls the boundary nodes keep their half-cell sums (no correction).  Particles are
 * visited in index order, each adding (1-w) to node j and then w to node j+1; the node sums are
 * multiplied by weight at the end.  Flagged-dead particles (cell < 0) are skipped.
 * Pins (tests/test_oracle_deposit.py): single particle, total charge, first moment (dipole),
 * one particle per cell centre, linearity, periodic fold, numpy.add.at brute force. */
int oracle_deposit(int64_t n, const double *x, const int32_t *cell, int32_t nc, double dx,
                   int32_t boundary, double weight, double *rho)
{
    if (n < 0 || nc < 1 || !(dx > 0.0)) return -1;
    const double inv_dx = 1.0 / dx;
    for (int32_t j = 0; j <= nc; ++j) rho[j] = 0.0;
    for (int64_t i = 0; i < n; ++i) {
        if (cell[i] < 0) continue;
        const double xs = x[i] * inv_dx;
        double jf = floor(xs);
        if (!(jf >= 0.0) || jf > (double)nc) return -2;
        int32_t j = (int32_t)jf;
        if (j > nc - 1) { j = nc - 1; jf = (double)j; }
        const double w = xs - jf;
        const double w0 = 1.0 - w;
        rho[j] = rho[j] + w0;
        rho[j + 1] = rho[j + 1] + w;
    }
    if (boundary == ORACLE_PERIODIC) {
        rho[0] = rho[0] + rho[nc];
        rho[nc] = rho[0];
    }
    for (int32_t j = 0; j <= nc; ++j) rho[j] = rho[j] * weight;
    return 0;
}
