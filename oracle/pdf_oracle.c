/*
 * oracle/pdf_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, scalar fp64 CPU implementation of what the CUDA library computes:
 * LHAPDF-style log-bicubic interpolation of xf(x,Q^2) on a Q^2-subgridded knot grid
 * (section 2.2), its continuation outside the grid, and log-cubic
 * interpolation of alpha_s(Q^2) with constant extrapolation (section 2.3).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call this file.  It shares no code, header, table or helper
 * with paper_2009_06635_b200/csrc/ and neither side includes the other.
 *
 * The paper prints no interpolation formula: it names "the prescription originally
 * implemented in LHAPDF6, namely a log-bicubic PDF interpolation in terms of x and Q^2"
 * and "a log-cubic interpolation with constant extrapolation".
 * The formulas below are the readings O1-O6 of SURVEY.md section 8(c), restated in
 * DESIGN.md ("Readings of the paper").  Each function cites the reading it follows, and
 * is written in that reading's order and notation: no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): knot reproduction, bilinear
 * exactness, brute-force separable-weight evaluation on tiny grids, quadratic exactness
 * in interior cells only, scipy CubicHermiteSpline special case, threshold side rule,
 * continuity and power-law exactness of the continuation, one-loop alpha_s closed form.
 * PARITY UNPINNED (no source in the paper, no LHAPDF here to compare with): the
 * continuation constants of O4/O5 (1e-3, 1e-5, -2.5, 1.01, 0.01, gamma = 1 for |y0| < 1e-5)
 * and reading Q10
 * (alpha_s frozen below the first node).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC pdf_oracle.c -lquadmath -lm
 */
#include <math.h>
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Reading R-ln: "ln" of a coordinate (x, Q^2, or a knot) is the natural
 * logarithm correctly rounded to fp64.  Computed in binary128 and rounded once, so the
 * definition does not depend on a libm version.  ("log-bicubic ... in terms
 * of x and Q^2"; natural log per reading Q4 -- the base cancels in t, tau and r.) */
static double ln_cr(double a) { return (double)logq((__float128)a); }

/* ------------------------------------------------------------------ grid storage */
typedef struct {
    int n_sub, nx, n_pid, nq_tot;
    int *x_off;     /* [n_sub+1] subgrid s owns x knots x_off[s] .. x_off[s+1]-1 (LHAPDF lets every subgrid
                       carry its own x-knot array; with one shared array all subgrids point at it) */
    double *x;      /* x knots, per subgrid */
    double *U;      /* ln x knots */
    int *q_off;     /* [n_sub+1] */
    double *q2;     /* [nq_tot] Q^2 knots, q2 = Q*Q */
    double *V;      /* [nq_tot] ln Q^2 knots */
    int *pids;      /* [n_pid] */
    long *v_off;    /* [n_sub] offset of subgrid s in val */
    double *val;    /* values [s][ix][iq][ipid] */
    long n_invalid; /* points that had no value (x > xmax, x <= 0, Q^2 <= 0, NaN) */
} ogrid;

static int nq_of(const ogrid *g, int s) { return g->q_off[s + 1] - g->q_off[s]; }
static int nx_of(const ogrid *g, int s) { return g->x_off[s + 1] - g->x_off[s]; }
static const double *x_of(const ogrid *g, int s) { return g->x + g->x_off[s]; }
static const double *U_of(const ogrid *g, int s) { return g->U + g->x_off[s]; }

/* f[i][m][k] of subgrid s */
static double fval(const ogrid *g, int s, int i, int m, int k)
{
    return g->val[g->v_off[s] + ((long)i * nq_of(g, s) + m) * g->n_pid + k];
}

/* x_offsets: [n_sub+1] into x_knots (per-subgrid x-knot arrays, values [s][ix_s][iq_s][ipid]), or NULL:
 * one array of nx knots shared by all subgrids.  All subgrids must span the same [x_0, x_max]. */
void *oracle_pdf_grid_create_xs(int n_sub, int nx, const int *x_offsets, const double *x_knots, const int *q_offsets,
                                const double *q_knots, int n_pid, const int *pids,
                                const double *values)
{
    ogrid *g = (ogrid *)calloc(1, sizeof(ogrid));
    g->n_sub = n_sub; g->n_pid = n_pid; g->nq_tot = q_offsets[n_sub];
    g->x_off = (int *)malloc(sizeof(int) * (n_sub + 1));
    int nxt = x_offsets ? x_offsets[n_sub] : nx;
    g->nx = nxt;
    g->x = (double *)malloc(sizeof(double) * nxt * (x_offsets ? 1 : n_sub));
    g->U = (double *)malloc(sizeof(double) * nxt * (x_offsets ? 1 : n_sub));
    for (int s = 0; s <= n_sub; s++) g->x_off[s] = x_offsets ? x_offsets[s] : s * nx;
    for (int s = 0; s < n_sub; s++)
        for (int i = 0; i < nx_of(g, s); i++) {
            double xv = x_offsets ? x_knots[x_offsets[s] + i] : x_knots[i];
            g->x[g->x_off[s] + i] = xv; g->U[g->x_off[s] + i] = ln_cr(xv);
        }
    g->q_off = (int *)malloc(sizeof(int) * (n_sub + 1));
    memcpy(g->q_off, q_offsets, sizeof(int) * (n_sub + 1));
    g->q2 = (double *)malloc(sizeof(double) * g->nq_tot);
    g->V = (double *)malloc(sizeof(double) * g->nq_tot);
    for (int j = 0; j < g->nq_tot; j++) {
        g->q2[j] = q_knots[j] * q_knots[j];  /* q_j = Q_j * Q_j */
        g->V[j] = ln_cr(g->q2[j]);           /* V_j = ln(Q_j * Q_j) */
    }
    g->pids = (int *)malloc(sizeof(int) * n_pid);
    memcpy(g->pids, pids, sizeof(int) * n_pid);
    g->v_off = (long *)malloc(sizeof(long) * n_sub);
    long tot = 0;
    for (int s = 0; s < n_sub; s++) { g->v_off[s] = tot; tot += (long)nx_of(g, s) * nq_of(g, s) * n_pid; }
    g->val = (double *)malloc(sizeof(double) * tot);
    memcpy(g->val, values, sizeof(double) * tot);
    return g;
}

void *oracle_pdf_grid_create(int n_sub, int nx, const double *x_knots, const int *q_offsets,
                             const double *q_knots, int n_pid, const int *pids,
                             const double *values)
{
    return oracle_pdf_grid_create_xs(n_sub, nx, NULL, x_knots, q_offsets, q_knots, n_pid, pids, values);
}

void oracle_pdf_grid_free(void *h)
{
    ogrid *g = (ogrid *)h;
    if (!g) return;
    free(g->x); free(g->U); free(g->x_off); free(g->q_off); free(g->q2); free(g->V);
    free(g->pids); free(g->v_off); free(g->val); free(g);
}

long oracle_pdf_grid_invalid(void *h) { return ((ogrid *)h)->n_invalid; }

/* ------------------------------------------------------------------ O1, O2 */

/* O1 -- cubic Hermite on the unit interval; dL, dH are derivatives already multiplied
 * by the interval length. */
static double hermite(double t, double yL, double dL, double yH, double dH)
{
    double t2 = t * t, t3 = t2 * t;
    double h00 = 2.0 * t3 - 3.0 * t2 + 1.0;
    double h10 = t3 - 2.0 * t2 + t;
    double h01 = -2.0 * t3 + 3.0 * t2;
    double h11 = t3 - t2;
    return h00 * yL + h10 * dL + h01 * yH + h11 * dH;
}

/* O2 -- finite-difference derivative at knot m of the sequence (z_m, y_m), m = 0..M-1:
 * one-sided at both ends, the plain mean of the two one-sided slopes inside.  "End"
 * means the end of the SUBGRID along Q^2 and of the x-knot array along x: this is the
 * "special care ... close to quark mass thresholds and grids x edges" of PAPER.md:67-69. */
static double fd_slope(double yL, double yH, double zL, double zH) { return (yH - yL) / (zH - zL); }

/* ------------------------------------------------------------------ O3 */
typedef struct { int s, i, j; double t, tau, dU, dV; } cell;

/* O3 steps 1-3: subgrid, cell and in-cell coordinates of an in-range point. */
static cell locate(const ogrid *g, double x, double q2)
{
    cell c;
    /* 1. subgrid: the last one whose first Q^2 knot <= Q^2 (threshold -> upper subgrid) */
    c.s = 0;
    for (int s = 1; s < g->n_sub; s++)
        if (g->q2[g->q_off[s]] <= q2) c.s = s;
    /* 2. cell: largest knot index <= the coordinate, clamped to the last interval;
     *    comparisons on raw x and Q^2, never on logs */
    const double *xs = x_of(g, c.s), *Us = U_of(g, c.s);  /* the x knots of the point's own subgrid */
    c.i = 0;
    for (int m = 1; m <= nx_of(g, c.s) - 2; m++)
        if (xs[m] <= x) c.i = m;
    const double *q2s = g->q2 + g->q_off[c.s];
    int nq = nq_of(g, c.s);
    c.j = 0;
    for (int m = 1; m <= nq - 2; m++)
        if (q2s[m] <= q2) c.j = m;
    /* 3. u = ln x, v = ln Q^2 */
    const double *Vs = g->V + g->q_off[c.s];
    double u = ln_cr(x), v = ln_cr(q2);
    c.dU = Us[c.i + 1] - Us[c.i];
    c.t = (u - Us[c.i]) / c.dU;
    c.dV = Vs[c.j + 1] - Vs[c.j];
    c.tau = (v - Vs[c.j]) / c.dV;
    return c;
}

/* O2 along x at fixed Q row m of subgrid s, for PID column k */
static double du_at(const ogrid *g, int s, int i, int m, int k)
{
    const double *U = U_of(g, s);
    int nx = nx_of(g, s);
    if (i == 0) return fd_slope(fval(g, s, 0, m, k), fval(g, s, 1, m, k), U[0], U[1]);
    if (i == nx - 1) return fd_slope(fval(g, s, nx - 2, m, k), fval(g, s, nx - 1, m, k), U[nx - 2], U[nx - 1]);
    return 0.5 * (fd_slope(fval(g, s, i, m, k), fval(g, s, i + 1, m, k), U[i], U[i + 1]) +
                  fd_slope(fval(g, s, i - 1, m, k), fval(g, s, i, m, k), U[i - 1], U[i]));
}

/* O3 step 4: row value R_m = Hermite in u along Q row m */
static double row_value(const ogrid *g, const cell *c, int m, int k)
{
    return hermite(c->t, fval(g, c->s, c->i, m, k), c->dU * du_at(g, c->s, c->i, m, k),
                   fval(g, c->s, c->i + 1, m, k), c->dU * du_at(g, c->s, c->i + 1, m, k));
}

/* O3 steps 4-6 for PID column k */
static double o3_column(const ogrid *g, const cell *c, int k)
{
    const double *Vs = g->V + g->q_off[c->s];
    int nq = nq_of(g, c->s), j = c->j;
    double Rj = row_value(g, c, j, k), Rj1 = row_value(g, c, j + 1, k);
    /* 5. derivatives of the row values along v, O2 inside the subgrid */
    double s1 = (Rj1 - Rj) / c->dV;
    double dL, dH;
    if (j == 0) dL = s1;
    else dL = 0.5 * (s1 + (Rj - row_value(g, c, j - 1, k)) / (Vs[j] - Vs[j - 1]));
    if (j + 1 == nq - 1) dH = s1;
    else dH = 0.5 * (s1 + (row_value(g, c, j + 2, k) - Rj1) / (Vs[j + 2] - Vs[j + 1]));
    /* 6. Hermite in v */
    return hermite(c->tau, Rj, c->dV * dL, Rj1, c->dV * dH);
}

/* O3 -- in-range value: x_0 <= x <= x_max and q_min <= Q^2 <= q_max, ends inclusive */
static double o3(const ogrid *g, int k, double x, double q2)
{
    cell c = locate(g, x, q2);
    return o3_column(g, &c, k);
}

/* ------------------------------------------------------------------ O4, O5 */
#define CONT_LOGLOG_MIN 1e-3 /* O4: both values above this -> linear in log-log      */
#define LOWQ_Y0_MIN 1e-5     /* O5-C: |y0| below this -> gamma = LOWQ_GAMMA_SMALL     */
#define LOWQ_GAMMA_SMALL 1.0 /* O5-C: then xf = y0 * rho, linear in Q^2 (reading Q9) */
#define LOWQ_GAMMA_MIN -2.5  /* O5-C: gamma clamp                                    */
#define LOWQ_PROBE 1.01      /* O5-C: second probe at 1.01 q_min                     */
#define LOWQ_PROBE_STEP 0.01

/* O4 -- continuation E(z; zL, zH, yL, yH), z arguments already logs */
static double continuation(double z, double zL, double zH, double yL, double yH)
{
    double r = (z - zL) / (zH - zL);
    if (yL > CONT_LOGLOG_MIN && yH > CONT_LOGLOG_MIN)
        return exp(log(yL) + r * (log(yH) - log(yL)));
    return yL + r * (yH - yL);
}

/* O5-A: x < x_0, Q^2 in range */
/* subgrid of an in-range scale (O3 step 1) */
static int subgrid_of(const ogrid *g, double q2)
{
    int s0 = 0;
    for (int s = 1; s < g->n_sub; s++)
        if (g->q2[g->q_off[s]] <= q2) s0 = s;
    return s0;
}

static double rule_a(const ogrid *g, int k, double x, double q2)
{
    int s = subgrid_of(g, q2);  /* the first two x knots of the subgrid the scale falls in */
    double yL = o3(g, k, x_of(g, s)[0], q2), yH = o3(g, k, x_of(g, s)[1], q2);
    return continuation(ln_cr(x), U_of(g, s)[0], U_of(g, s)[1], yL, yH);
}

/* G(x, q): O3 if x >= x_0, rule A otherwise (q in range) */
static double G(const ogrid *g, int k, double x, double q2)
{
    return (x >= g->x[0]) ? o3(g, k, x, q2) : rule_a(g, k, x, q2);
}

/* O5-B: Q^2 > q_max */
static double rule_b(const ogrid *g, int k, double x, double q2)
{
    double qa = g->q2[g->nq_tot - 2], qb = g->q2[g->nq_tot - 1];
    double ya = G(g, k, x, qa), yb = G(g, k, x, qb);
    return continuation(ln_cr(q2), ln_cr(qa), ln_cr(qb), ya, yb);
}

/* O5-C: Q^2 < q_min */
static double rule_c(const ogrid *g, int k, double x, double q2)
{
    double qmin = g->q2[0];
    double y0 = G(g, k, x, qmin), y1 = G(g, k, x, LOWQ_PROBE * qmin);
    double gamma = LOWQ_GAMMA_SMALL;
    if (fabs(y0) >= LOWQ_Y0_MIN) gamma = fmax(LOWQ_GAMMA_MIN, (y1 - y0) / y0 / LOWQ_PROBE_STEP);
    double rho = q2 / qmin;
    return y0 * pow(rho, gamma * rho + 1.0 - rho);
}

/* xf of PID column k at any (x, Q^2); NaN (and *bad = 1) where no value is defined */
static double xf_any(const ogrid *g, int k, double x, double q2, int *bad)
{
    double xmax = x_of(g, 0)[nx_of(g, 0) - 1], qmin = g->q2[0], qmax = g->q2[g->nq_tot - 1];
    if (!(x > 0.0) || !(q2 > 0.0) || !(x <= xmax) || isinf(q2)) { *bad = 1; return NAN; }
    if (q2 > qmax) return rule_b(g, k, x, q2);
    if (q2 < qmin) return rule_c(g, k, x, q2);
    return G(g, k, x, q2);
}

/* PID -> column; 0 is an alias of 21 (gluon); -1 if absent */
static int pid_column(const ogrid *g, int pid)
{
    if (pid == 0) pid = 21;
    for (int k = 0; k < g->n_pid; k++)
        if (g->pids[k] == pid) return k;
    return -1;
}

/* ==================================================================================
 * Conditioning scale -- a helper for the parity TOLERANCE only, not part of the method.
 * For one output it returns S ~ sum |d result / d f_knot| |f_knot|: the same steps as
 * above with every table value and every coefficient replaced by its magnitude, and the
 * continuation rules propagated by their partial derivatives.  eps*S is the size of the
 * rounding noise any fp64 evaluation order carries at that point (Tolerance).
 * ================================================================================== */
static double habs(double t, double yL, double dL, double yH, double dH)
{
    double t2 = t * t, t3 = t2 * t;
    return fabs(2.0 * t3 - 3.0 * t2 + 1.0) * yL + fabs(t3 - 2.0 * t2 + t) * dL +
           fabs(-2.0 * t3 + 3.0 * t2) * yH + fabs(t3 - t2) * dH;
}
static double aslope(double yL, double yH, double zL, double zH) { return (fabs(yH) + fabs(yL)) / (zH - zL); }
static double du_abs(const ogrid *g, int s, int i, int m, int k)
{
    const double *U = U_of(g, s);
    int nx = nx_of(g, s);
    if (i == 0) return aslope(fval(g, s, 0, m, k), fval(g, s, 1, m, k), U[0], U[1]);
    if (i == nx - 1) return aslope(fval(g, s, nx - 2, m, k), fval(g, s, nx - 1, m, k), U[nx - 2], U[nx - 1]);
    return 0.5 * (aslope(fval(g, s, i, m, k), fval(g, s, i + 1, m, k), U[i], U[i + 1]) +
                  aslope(fval(g, s, i - 1, m, k), fval(g, s, i, m, k), U[i - 1], U[i]));
}
static double row_abs(const ogrid *g, const cell *c, int m, int k)
{
    return habs(c->t, fabs(fval(g, c->s, c->i, m, k)), c->dU * du_abs(g, c->s, c->i, m, k),
                fabs(fval(g, c->s, c->i + 1, m, k)), c->dU * du_abs(g, c->s, c->i + 1, m, k));
}
static double o3_scale(const ogrid *g, int k, double x, double q2)
{
    cell c = locate(g, x, q2);
    const double *Vs = g->V + g->q_off[c.s];
    int nq = nq_of(g, c.s), j = c.j;
    double Rj = row_abs(g, &c, j, k), Rj1 = row_abs(g, &c, j + 1, k);
    double s1 = (Rj1 + Rj) / c.dV, dL, dH;
    if (j == 0) dL = s1;
    else dL = 0.5 * (s1 + (Rj + row_abs(g, &c, j - 1, k)) / (Vs[j] - Vs[j - 1]));
    if (j + 1 == nq - 1) dH = s1;
    else dH = 0.5 * (s1 + (row_abs(g, &c, j + 2, k) + Rj1) / (Vs[j + 2] - Vs[j + 1]));
    return habs(c.tau, Rj, c.dV * dL, Rj1, c.dV * dH);
}
/* scale of E(z; zL, zH, yL, yH) given the scales sL, sH of yL, yH */
static double cont_scale(double z, double zL, double zH, double yL, double yH, double sL, double sH)
{
    double r = (z - zL) / (zH - zL);
    if (yL > CONT_LOGLOG_MIN && yH > CONT_LOGLOG_MIN) {
        double e = exp(log(yL) + r * (log(yH) - log(yL)));
        return e * (fabs(1.0 - r) * sL / yL + fabs(r) * sH / yH);
    }
    return fabs(1.0 - r) * sL + fabs(r) * sH;
}
static double G_scale(const ogrid *g, int k, double x, double q2)
{
    if (x >= g->x[0]) return o3_scale(g, k, x, q2);
    int s = subgrid_of(g, q2);
    const double *xs = x_of(g, s), *Us = U_of(g, s);
    return cont_scale(ln_cr(x), Us[0], Us[1], o3(g, k, xs[0], q2), o3(g, k, xs[1], q2),
                      o3_scale(g, k, xs[0], q2), o3_scale(g, k, xs[1], q2));
}
static double xf_scale(const ogrid *g, int k, double x, double q2)
{
    double xmax = x_of(g, 0)[nx_of(g, 0) - 1], qmin = g->q2[0], qmax = g->q2[g->nq_tot - 1];
    if (!(x > 0.0) || !(q2 > 0.0) || !(x <= xmax) || isinf(q2)) return NAN;
    if (q2 > qmax) {
        double qa = g->q2[g->nq_tot - 2], qb = qmax;
        return cont_scale(ln_cr(q2), ln_cr(qa), ln_cr(qb), G(g, k, x, qa), G(g, k, x, qb),
                          G_scale(g, k, x, qa), G_scale(g, k, x, qb));
    }
    if (q2 < qmin) {
        double y0 = G(g, k, x, qmin), y1 = G(g, k, x, LOWQ_PROBE * qmin);
        double s0 = G_scale(g, k, x, qmin), s1 = G_scale(g, k, x, LOWQ_PROBE * qmin);
        double rho = q2 / qmin, gamma = LOWQ_GAMMA_SMALL, dg0 = 0.0, dg1 = 0.0;
        if (fabs(y0) >= LOWQ_Y0_MIN) {
            double graw = (y1 - y0) / y0 / LOWQ_PROBE_STEP;
            gamma = fmax(LOWQ_GAMMA_MIN, graw);
            if (graw > LOWQ_GAMMA_MIN) {
                dg0 = fabs(y1 / (y0 * y0)) / LOWQ_PROBE_STEP;
                dg1 = fabs(1.0 / y0) / LOWQ_PROBE_STEP;
            }
        }
        double res = fabs(y0 * pow(rho, gamma * rho + 1.0 - rho));
        double lr = fabs(rho * log(rho));
        double rel0 = (y0 != 0.0) ? s0 / fabs(y0) : 0.0;
        return res * (rel0 + lr * (dg0 * s0 + dg1 * s1)) + ((y0 == 0.0) ? s0 : 0.0);
    }
    return G_scale(g, k, x, q2);
}

/* ------------------------------------------------------------------ batch entry points */

/* out[kr * n + p] = xf of requested PID kr at point p (flavour-major).  scale may be
 * NULL; otherwise scale[kr * n + p] = conditioning scale (tolerance helper).  Returns 0,
 * or -1 if a requested PID is not in the grid. */
int oracle_pdf_xfxq2(void *h, int n_req, const int *pids, long n, const double *x,
                     const double *q2, double *out, double *scale)
{
    ogrid *g = (ogrid *)h;
    int cols[64];
    if (n_req > 64) return -2;
    for (int r = 0; r < n_req; r++) {
        cols[r] = pid_column(g, pids[r]);
        if (cols[r] < 0) return -1;
    }
    long n_bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : n_bad)
    for (long p = 0; p < n; p++) {
        int bad = 0;
        for (int r = 0; r < n_req; r++) {
            out[(long)r * n + p] = xf_any(g, cols[r], x[p], q2[p], &bad);
            if (scale) scale[(long)r * n + p] = xf_scale(g, cols[r], x[p], q2[p]);
        }
        n_bad += bad;
    }
    g->n_invalid += n_bad;
    return 0;
}

/* ------------------------------------------------------------------ O6: alpha_s */
typedef struct {
    int K;
    double *q2; /* Q_k * Q_k */
    double *Z;  /* ln(Q_k * Q_k) */
    double *a;  /* alpha_s(Q_k) */
} oalphas;

void *oracle_alphas_create(int n_knots, const double *q_knots, const double *alphas)
{
    oalphas *A = (oalphas *)calloc(1, sizeof(oalphas));
    A->K = n_knots;
    A->q2 = (double *)malloc(sizeof(double) * n_knots);
    A->Z = (double *)malloc(sizeof(double) * n_knots);
    A->a = (double *)malloc(sizeof(double) * n_knots);
    for (int k = 0; k < n_knots; k++) {
        A->q2[k] = q_knots[k] * q_knots[k];
        A->Z[k] = ln_cr(A->q2[k]);
        A->a[k] = alphas[k];
    }
    return A;
}

void oracle_alphas_free(void *h)
{
    oalphas *A = (oalphas *)h;
    if (!A) return;
    free(A->q2); free(A->Z); free(A->a); free(A);
}

/* O6 -- alpha_s(Q^2): constant outside the nodes ("constant extrapolation",
 * PAPER.md:73; reading Q10: on both sides); inside, cubic Hermite in ln Q^2 with O2
 * derivatives taken inside the subgrid ("improved treatment of the sub-grids mechanism
 * ... flavour thresholds").  A repeated Q value splits the node list. */
static double alphas_point(const oalphas *A, double q2)
{
    int K = A->K;
    if (!(q2 > 0.0)) return NAN;
    if (q2 < A->q2[0]) return A->a[0];
    if (q2 > A->q2[K - 1]) return A->a[K - 1];
    /* subgrid [lo, hi] = the last one whose first knot <= Q^2 (upper on a threshold) */
    int lo = 0;
    for (int k = 1; k < K; k++)
        if (A->q2[k] == A->q2[k - 1] && A->q2[k] <= q2) lo = k;
    int hi = K - 1;
    for (int k = lo + 1; k < K; k++)
        if (A->q2[k] == A->q2[k - 1]) { hi = k - 1; break; }
    int M = hi - lo + 1;
    const double *z = A->Z + lo, *y = A->a + lo, *qq = A->q2 + lo;
    int m = 0;
    for (int c = 1; c <= M - 2; c++)
        if (qq[c] <= q2) m = c;
    double dZ = z[m + 1] - z[m];
    double tau = (ln_cr(q2) - z[m]) / dZ;
    double s1 = fd_slope(y[m], y[m + 1], z[m], z[m + 1]);
    double dL = (m == 0) ? s1 : 0.5 * (s1 + fd_slope(y[m - 1], y[m], z[m - 1], z[m]));
    double dH = (m + 1 == M - 1) ? s1 : 0.5 * (s1 + fd_slope(y[m + 1], y[m + 2], z[m + 1], z[m + 2]));
    return hermite(tau, y[m], dZ * dL, y[m + 1], dZ * dH);
}

int oracle_alphas_q2(void *h, long n, const double *q2, double *out)
{
    const oalphas *A = (const oalphas *)h;
#pragma omp parallel for schedule(static)
    for (long p = 0; p < n; p++) out[p] = alphas_point(A, q2[p]);
    return 0;
}

/* ------------------------------------------------------------------ misc */
double oracle_ln(double a) { return ln_cr(a); }

int oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
