/*
 * oracle_field.c -- plain, slow, obviously-correct CPU oracle for the FIELD SOLVE of the 1D
 * electrostatic PIC cycle: phase (iii), "the field solver, which computes the electric ... fields by
 * solving ... Poisson's equations", with the "native Poisson solver ... and smoothing
 * operators without external numerical libraries" the paper attributes to BIT1 (XPDP1
 * lineage, ref [19]).  SURVEY.md section 8(f) rank 2.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline leg may load it); it shares no code, header, table or helper with the CUDA path.
 *
 * The paper prints neither the discretisation nor the filter.  Readings taken (DESIGN.md section 12,
 * S23-S28; normalised units, epsilon_0 = 1):
 *   S23  discrete Poisson equation on the nodes j = 0..nc of the mover's grid:
 *            (phi[j-1] - 2 phi[j] + phi[j+1]) / dx^2 = -rho[j]
 *   S24  absorbing (bounded) grid: both walls grounded, phi[0] = phi[nc] = 0 (Dirichlet); the unknowns
 *        are the nc-1 interior nodes; rho[0] and rho[nc] do not enter.
 *   S25  periodic grid: nodes 0 and nc are one point (rho[nc] mirrors rho[0], as pic_deposit writes it);
 *        the unknowns are nodes 0..nc-1; the operator is singular, so rho is neutralised first
 *        (rho~ = rho - mean over the nc distinct nodes: a uniform background) and the solution of zero
 *        mean is returned (sum over the nc distinct nodes = 0), phi[nc] = phi[0].
 *   S26  E on the nodes by centred difference, E[j] = -(phi[j+1] - phi[j-1]) / (2 dx); one-sided at the
 *        walls of a bounded grid, E[0] = -(phi[1] - phi[0])/dx, E[nc] = -(phi[nc] - phi[nc-1])/dx;
 *        periodic: the difference wraps and E[nc] = E[0] (reading S14 of the mover).
 *   S27  smoother = `passes` passes of the 1-2-1 binomial digital filter on rho,
 *            rho'[j] = (rho[j-1] + 2 rho[j] + rho[j+1]) / 4,
 *        periodic: indices wrap over the nc distinct nodes; bounded: the quarter that would leave the
 *        grid is reflected back into the wall node, rho'[0] = (3 rho[0] + rho[1])/4 (likewise at nc),
 *        so that every pass conserves the total charge and leaves a constant untouched.
 *   S28  precision and operation order.  Filter and E: binary64, each statement one rounded operation
 *        (-ffp-contract=off):
 *            filter  ((rho[j-1] + 2*rho[j]) + rho[j+1]) * 0.25   (the products by 2 and 0.25 are exact)
 *            E       (phi[j+1] - phi[j-1]) * (-0.5*inv_dx),  one-sided (phi[1] - phi[0]) * (-inv_dx)
 *        Solve: the textbook Thomas algorithm for  -phi[j-1] + 2 phi[j] - phi[j+1] = dx^2 rho[j], as written
 *        below, with its recurrences carried in binary128 (`xreal`: __float128 where the compiler has it, i.e.
 *        x86-64; `long double`, which is binary128, on aarch64) and phi rounded to binary64 at the end.  The
 *        solution of the linear system is what is defined, and a sequential elimination accumulates its own
 *        rounding error systematically: in binary64 3.7e-13 of max|phi| at nc = 1000 (uniform rho), and even in
 *        the 64-bit-mantissa x87 long double 1.8e-13 at nc = 10^5 and 8.7e-12 at nc = 10^6 (measured against an
 *        extended-precision double prefix sum, which the CUDA path matched to 1e-14).  At the 1e-12 parity bar the
 *        oracle, not the kernel, would be the larger error; in binary128 its own error is below 1e-25.
 *        Inputs and outputs are binary64.
 *
 * The solve reaches, up to rounding, a result with a plain definition (the solution of a linear system);
 * the oracle is the textbook sequential elimination.  Pins (tests/test_oracle_field.py, "-m not gpu";
 * none re-calls these routines): uniform rho -> the exact parabola rho dx^2 j (nc-j)/2; sine modes are
 * eigenvectors with eigenvalue (2 - 2 cos(k))/dx^2 on both grids; a point charge gives the
 * piecewise-linear Green's function; the residual of the discrete operator evaluated in extended
 * precision; the discrete Gauss law on the half nodes; numpy.linalg.solve / scipy solve_banded on small
 * grids; neutralisation and gauge on the periodic grid; E of linear and quadratic potentials incl. the
 * one-sided wall values; the filter's charge conservation, Nyquist annihilation, delta response at a
 * wall and in the interior, numpy.convolve in the interior, k passes = k single passes.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_PERIODIC 0
#define ORACLE_ABSORBING 1

/* the precision the elimination is carried in (S28) */
#if defined(__SIZEOF_FLOAT128__) && !defined(__aarch64__)
typedef __float128 xreal;
#define XABS(v) ((v) < 0 ? -(v) : (v))
#else
typedef long double xreal;
#define XABS(v) fabsl(v)
#endif

/* S27: `passes` passes of the 1-2-1 filter; in and out have nc+1 entries and may be the same array. */
int oracle_smooth(int32_t nc, int32_t boundary, int32_t passes, const double *rho_in, double *rho_out)
{
    if (nc < 2 || passes < 0) return -1;
    double *a = (double *)malloc(((size_t)nc + 1) * sizeof(double));
    double *b = (double *)malloc(((size_t)nc + 1) * sizeof(double));
    if (!a || !b) { free(a); free(b); return -2; }
    memcpy(a, rho_in, ((size_t)nc + 1) * sizeof(double));
    for (int32_t p = 0; p < passes; ++p) {
        for (int32_t j = 0; j <= nc; ++j) {
            double left, right;
            if (boundary == ORACLE_PERIODIC) {
                /* the nc distinct nodes are 0..nc-1; node nc is node 0 */
                int32_t jj = j == nc ? 0 : j;
                left = a[jj == 0 ? nc - 1 : jj - 1];
                right = a[jj == nc - 1 ? 0 : jj + 1];
            } else {
                left = j == 0 ? a[0] : a[j - 1];   /* reflected quarter */
                right = j == nc ? a[nc] : a[j + 1];
            }
            double centre = boundary == ORACLE_PERIODIC && j == nc ? a[0] : a[j];
            double t = 2.0 * centre;
            double s1 = left + t;
            double s2 = s1 + right;
            b[j] = s2 * 0.25;
        }
        double *sw = a; a = b; b = sw;
    }
    memcpy(rho_out, a, ((size_t)nc + 1) * sizeof(double));
    free(a);
    free(b);
    return 0;
}

/* Thomas algorithm for  -u[j-1] + 2 u[j] - u[j+1] = r[j],  j = 1..m,  u[0] = u[m+1] = 0.
 * r and u are indexed 1..m (arrays of m+2 entries); cp, dp scratch of m+2 entries.  binary128 (S28). */
static void thomas_121(int32_t m, const xreal *r, xreal *u, xreal *cp, xreal *dp)
{
    u[0] = (xreal)0.0;
    u[m + 1] = (xreal)0.0;
    if (m < 1) return;
    cp[1] = -(xreal)0.5;            /* c/b = -1/2 */
    dp[1] = r[1] * (xreal)0.5;      /* r/b */
    for (int32_t j = 2; j <= m; ++j) {
        xreal denom = (xreal)2.0 + cp[j - 1]; /* b - a*cp[j-1] with a = -1 */
        xreal num = r[j] + dp[j - 1];   /* r - a*dp[j-1] */
        cp[j] = -(xreal)1.0 / denom;
        dp[j] = num / denom;
    }
    u[m] = dp[m];
    for (int32_t j = m - 1; j >= 1; --j) {
        xreal t = cp[j] * u[j + 1];
        u[j] = dp[j] - t;
    }
}

/* Sum of n binary64 values in extended precision with Neumaier's compensation (the running error of every addition
 * is recovered exactly and added at the end): the result is the exact sum rounded once, for all practical n.
 * Needed for the mean that neutralises a periodic grid (S25): an error d in that mean leaves a uniform charge d
 * behind, i.e. a spurious parabola of height d dx^2 nc^2 / 8 in phi -- 1e11 d at the 10^6 nodes of config 4.  A
 * plain x87 long double loop is not enough: 65,536 equal terms already lose 12 bits (measured: phi = 1.7e-8 instead of
 * 0 for uniform rho = 0.37, dx = 0.5; pinned by test_uniform_rho_on_a_ring_gives_zero). */
static xreal sum_compensated(const double *v, int32_t n)
{
    xreal s = (xreal)0.0, c = (xreal)0.0;
    for (int32_t j = 0; j < n; ++j) {
        const xreal x = (xreal)v[j];
        const xreal t = s + x;
        if (XABS(s) >= XABS(x))
            c += (s - t) + x;
        else
            c += (x - t) + s;
        s = t;
    }
    return s + c;
}

static xreal sum_compensated_ld(const xreal *v, int32_t n)
{
    xreal s = (xreal)0.0, c = (xreal)0.0;
    for (int32_t j = 0; j < n; ++j) {
        const xreal x = v[j];
        const xreal t = s + x;
        if (XABS(s) >= XABS(x))
            c += (s - t) + x;
        else
            c += (x - t) + s;
        s = t;
    }
    return s + c;
}

/* S23-S25: phi on the nc+1 nodes from rho on the nc+1 nodes. */
int oracle_poisson(int32_t nc, double dx, int32_t boundary, const double *rho, double *phi)
{
    if (nc < 2 || !(dx > 0.0)) return -1;
    const size_t n1 = (size_t)nc + 2;
    xreal *r = (xreal *)malloc(n1 * sizeof(xreal));
    xreal *u = (xreal *)malloc(n1 * sizeof(xreal));
    xreal *cp = (xreal *)malloc(n1 * sizeof(xreal));
    xreal *dp = (xreal *)malloc(n1 * sizeof(xreal));
    if (!r || !u || !cp || !dp) { free(r); free(u); free(cp); free(dp); return -2; }
    const xreal dx2 = (xreal)dx * (xreal)dx;
    xreal mean = (xreal)0.0;
    if (boundary == ORACLE_PERIODIC)
        mean = sum_compensated(rho, nc) / (xreal)nc;
    for (int32_t j = 1; j <= nc - 1; ++j) {
        xreal rj = (xreal)rho[j] - mean; /* mean = 0 on a bounded grid */
        r[j] = dx2 * rj;
    }
    /* bounded: phi[0] = phi[nc] = 0.  periodic: the gauge phi[0] = 0 first (the equation at node 0 then holds
     * by itself because the neutralised rho sums to zero), the mean is removed below. */
    thomas_121(nc - 1, r, u, cp, dp);
    if (boundary == ORACLE_PERIODIC) {
        xreal pm = sum_compensated_ld(u, nc) / (xreal)nc;
        for (int32_t j = 0; j < nc; ++j) phi[j] = (double)(u[j] - pm);
        phi[nc] = phi[0];
    } else {
        for (int32_t j = 0; j <= nc; ++j) phi[j] = (double)u[j];
    }
    free(r);
    free(u);
    free(cp);
    free(dp);
    return 0;
}

/* S26: E on the nc+1 nodes from phi on the nc+1 nodes. */
int oracle_efield(int32_t nc, double dx, int32_t boundary, const double *phi, double *E)
{
    if (nc < 2 || !(dx > 0.0)) return -1;
    const double inv_dx = 1.0 / dx;
    const double mh = -0.5 * inv_dx; /* exact scaling of inv_dx */
    const double m1 = -inv_dx;
    for (int32_t j = 1; j <= nc - 1; ++j) {
        double d = phi[j + 1] - phi[j - 1];
        E[j] = d * mh;
    }
    if (boundary == ORACLE_PERIODIC) {
        double d = phi[1] - phi[nc - 1];
        E[0] = d * mh;
        E[nc] = E[0];
    } else {
        double d0 = phi[1] - phi[0];
        E[0] = d0 * m1;
        double d1 = phi[nc] - phi[nc - 1];
        E[nc] = d1 * m1;
    }
    return 0;
}

/* The field solve the library's pic_solve_field implements: smooth (passes >= 0) -> Poisson -> E.
 * rho_s (nc+1, the filtered density), phi (nc+1) and E (nc+1) are outputs. */
int oracle_field_solve(int32_t nc, double dx, int32_t boundary, int32_t passes, const double *rho,
                       double *rho_s, double *phi, double *E)
{
    int rc = oracle_smooth(nc, boundary, passes, rho, rho_s);
    if (rc) return rc;
    rc = oracle_poisson(nc, dx, boundary, rho_s, phi);
    if (rc) return rc;
    return oracle_efield(nc, dx, boundary, phi, E);
}
