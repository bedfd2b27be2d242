/*
 * oracle/orc_react.c -- CPU ORACLE (test infrastructure, NOT the product): the reactive half of Eq. (1)-(2).
 *
 * "We describe a new time integration method ... spectral deferred corrections ... with implicit
 * reaction updates"; L31-33, Eq. (1): U_t = A(U) + R(U), "R(U) ... the reactive source"; L35-40, Eq. (2):
 *   U^{m+1,(k+1)} = U^{m,(k+1)} + dt_m [A(U^{m,(k+1)}) - A(U^{m,(k)})]
 *                               + dt_m [R(U^{m+1,(k+1)}) - R(U^{m+1,(k)})] + I_m^{m+1}(A(U^(k)) + R(U^(k)))
 * which is implicit in U^{m+1,(k+1)} through R only (L42: "implicit in the reactions").  SURVEY 8(f) NEXT-3.
 *
 * The paper's 13-isotope network needs rate tables that are not available, so R is a SYNTHETIC stiff network with
 * the same structure (readings R1-R4):
 *   R1  a linear chain X_0 -> X_1 -> ... -> X_{ns-1} with temperature-dependent rates
 *         lambda_k(T) = rate[k] * (T / T0)^nu,   lambda_{ns-1} = 0 (the last species is stable);
 *         R(rho X_k) = rho (lambda_{k-1} X_{k-1} - lambda_k X_k);  R(rho) = R(rho v) = 0;
 *         R(rho E) = rho sum_k q[k] lambda_k X_k   (q[k] = specific energy released by the reaction of species k);
 *   R2  T from the gamma-law state with a constant c_v:  e = E/rho - |v|^2/2,  T = e / c_v;
 *   R3  the node solve is Newton's method on the ns+1 unknowns y = (rho X_0 .. rho X_{ns-1}, rho E) of one zone
 *         (rho and rho v are explicit because their R vanishes), analytic Jacobian, Gaussian elimination with
 *         partial pivoting, first iterate = the explicit part c of Eq. (2); it stops when the last correction is
 *         <= tol relative to (rho for species, |rho E| for energy) or after max_iter iterations;
 *   R4  the quadrature term integrates A + R of the previous iteration with the same node weights.
 * Pins (tests/test_oracle_react.py): backward-Euler closed form of the linear chain (nu = 0), species and energy
 * bookkeeping to roundoff, residual of the converged nonlinear solve, analytic Jacobian against finite differences,
 * and the order of the whole SDC iteration with R != 0 (2 for trapezoid, 4 for Simpson) against a tight-tolerance
 * ODE reference on a uniform state (where <A(U)> = 0 bitwise).
 * Unpinned by the paper itself: the network (R1-R2 are synthetic stand-ins), the Newton controls of R3.
 * Shares no code with paper_1910_12578_b200/csrc.  Build: -O2 -ffp-contract=off (oracle/build.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int nx, ny, nz, ng, nbx, nby, nbz, nspec;
    double dx, dy, dz, gamma, grav[3];
    int bc_lo[3], bc_hi[3];
    double small_dens, small_pres;
} orc_params;                                  /* same layout as in orc.c */

#define ORC_MAX_REACT 15
typedef struct {
    double cv, T0, nu;
    double rate[ORC_MAX_REACT];                /* rate[k] of species k -> k+1 at T = T0 (the last one is ignored)  */
    double q[ORC_MAX_REACT];                   /* specific energy release of that reaction                         */
    int max_iter;
    double tol;
} orc_react;

enum { ORC_OK = 0, ORC_EINVAL = -1 };

/* R and (optionally) dR/dy of one zone.  y = (rho X_0 .. rho X_{ns-1}, rho E), n = ns + 1 unknowns;
 * rho and ke = |rho v|^2 / (2 rho) are fixed.  J is row-major n x n. */
void orc_react_zone(const orc_react *r, int ns, double rho, double ke, const double *y, double *R, double *J)
{
    const int n = ns + 1;
    const double e = (y[ns] - ke) / rho;                     /* R2 */
    const double T = e / r->cv;
    const double f = pow(T / r->T0, r->nu);
    double lam[ORC_MAX_REACT], dlam[ORC_MAX_REACT];
    for (int k = 0; k < ns; ++k) {
        lam[k] = (k < ns - 1) ? r->rate[k] * f : 0.0;        /* R1 */
        dlam[k] = r->nu * lam[k] / T;                        /* d lambda_k / dT */
    }
    const double dTdE = 1.0 / (rho * r->cv);                 /* dT / d(rho E) */
    double RE = 0.0;
    for (int k = 0; k < ns; ++k) {
        const double in = (k > 0) ? lam[k - 1] * y[k - 1] : 0.0;
        R[k] = in - lam[k] * y[k];
        RE += r->q[k] * lam[k] * y[k];
    }
    R[ns] = RE;
    if (!J) return;
    memset(J, 0, sizeof(double) * n * n);
    double dRE = 0.0;
    for (int k = 0; k < ns; ++k) {
        if (k > 0) J[k * n + (k - 1)] = lam[k - 1];
        J[k * n + k] = -lam[k];
        const double din = (k > 0) ? dlam[k - 1] * y[k - 1] : 0.0;
        J[k * n + ns] = (din - dlam[k] * y[k]) * dTdE;
        J[ns * n + k] = r->q[k] * lam[k];
        dRE += r->q[k] * dlam[k] * y[k];
    }
    J[ns * n + ns] = dRE * dTdE;
}

/* Gaussian elimination with partial pivoting: solves M x = b in place (M row-major n x n, destroyed). */
static void solve_dense(int n, double *M, double *b)
{
    for (int c = 0; c < n; ++c) {
        int piv = c;
        for (int r = c + 1; r < n; ++r) if (fabs(M[r * n + c]) > fabs(M[piv * n + c])) piv = r;
        if (piv != c) {
            for (int k = 0; k < n; ++k) { const double t = M[c * n + k]; M[c * n + k] = M[piv * n + k]; M[piv * n + k] = t; }
            const double t = b[c]; b[c] = b[piv]; b[piv] = t;
        }
        for (int r = c + 1; r < n; ++r) {
            const double f = M[r * n + c] / M[c * n + c];
            for (int k = c; k < n; ++k) M[r * n + k] -= f * M[c * n + k];
            b[r] -= f * b[c];
        }
    }
    for (int r = n - 1; r >= 0; --r) {
        double s = b[r];
        for (int k = r + 1; k < n; ++k) s -= M[r * n + k] * b[k];
        b[r] = s / M[r * n + r];
    }
}

/* R3: solves y = c + dt R(y) for one zone; returns the number of Newton iterations (max_iter + 1 = not converged) */
int orc_react_solve_zone(const orc_react *r, int ns, double rho, double ke, double dt, const double *c, double *y)
{
    const int n = ns + 1;
    double R[ORC_MAX_REACT + 1], J[(ORC_MAX_REACT + 1) * (ORC_MAX_REACT + 1)], M[(ORC_MAX_REACT + 1) * (ORC_MAX_REACT + 1)];
    double d[ORC_MAX_REACT + 1];
    for (int i = 0; i < n; ++i) y[i] = c[i];
    for (int it = 1; it <= r->max_iter; ++it) {
        orc_react_zone(r, ns, rho, ke, y, R, J);
        for (int i = 0; i < n; ++i) {
            d[i] = -(y[i] - c[i] - dt * R[i]);
            for (int j = 0; j < n; ++j) M[i * n + j] = ((i == j) ? 1.0 : 0.0) - dt * J[i * n + j];
        }
        solve_dense(n, M, d);
        double worst = 0.0;
        for (int i = 0; i < n; ++i) {
            y[i] += d[i];
            const double scale = (i < ns) ? rho : fabs(y[ns]);
            const double rel = fabs(d[i]) / scale;
            if (rel > worst) worst = rel;
        }
        if (worst <= r->tol) return it;
    }
    return r->max_iter + 1;
}

static int check(const orc_params *p, const orc_react *r)
{
    if (!p || !r || p->ng != 4 || p->nspec < 1 || p->nspec > ORC_MAX_REACT) return ORC_EINVAL;
    if (!(r->cv > 0) || !(r->T0 > 0) || r->max_iter < 1 || !(r->tol > 0)) return ORC_EINVAL;
    return ORC_OK;
}

/* R(U) on the interior zones, A-like layout [b][c][k][j][i]; components 0..3 are zero. */
int orc_react_R(const orc_params *p, const orc_react *r, const double *U, double *Rout)
{
    if (check(p, r) || !U || !Rout) return ORC_EINVAL;
    const int ng = p->ng, ns = p->nspec, N = 5 + ns;
    const long nx = p->nx, ny = p->ny, nz = p->nz, ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nbox = (long)p->nbx * p->nby * p->nbz, ca = nx * ny * nz, cg = ex * ey * ez;
    for (long b = 0; b < nbox; ++b)
    for (long k = 0; k < nz; ++k)
    for (long j = 0; j < ny; ++j)
    for (long i = 0; i < nx; ++i) {
        const long za = b * N * ca + (k * ny + j) * nx + i;
        const long zu = b * N * cg + ((k + ng) * ey + j + ng) * ex + i + ng;
        const double rho = U[zu], mx = U[zu + cg], my = U[zu + 2 * cg], mz = U[zu + 3 * cg];
        const double ke = 0.5 * (mx * mx + my * my + mz * mz) / rho;
        double y[ORC_MAX_REACT + 1], R[ORC_MAX_REACT + 1];
        for (int s = 0; s < ns; ++s) y[s] = U[zu + (5 + s) * cg];
        y[ns] = U[zu + 4 * cg];
        orc_react_zone(r, ns, rho, ke, y, R, NULL);
        for (int c = 0; c < 4; ++c) Rout[za + c * ca] = 0.0;
        Rout[za + 4 * ca] = R[ns];
        for (int s = 0; s < ns; ++s) Rout[za + (5 + s) * ca] = R[s];
    }
    return ORC_OK;
}

/* Eq. (2) with R != 0 on the interior zones:
 *   c = U_m + dt_m (A_new_m - A_old_m) - dt_m R_old_next + sum_q w_q (A_quad[q] + R_quad[q]),
 *   U_next = c + dt_m R(U_next)    (Newton per zone, R3);  R_new_out <- R(U_next);
 * iters_out (interior zones, one int per zone, may be NULL) <- Newton iterations of the zone. */
int orc_sdc_update_react(const orc_params *p, const orc_react *r, double *U_next, const double *U_m, double dt_m,
                         const double *A_new_m, const double *A_old_m, const double *R_old_next,
                         int nquad, const double *const *A_quad, const double *const *R_quad, const double *w_quad,
                         double *R_new_out, int *iters_out)
{
    if (check(p, r) || !U_next || !U_m || !A_new_m || !A_old_m || !R_old_next || !R_new_out) return ORC_EINVAL;
    if (nquad < 0 || (nquad > 0 && (!A_quad || !R_quad || !w_quad))) return ORC_EINVAL;
    const int ng = p->ng, ns = p->nspec, N = 5 + ns;
    const long nx = p->nx, ny = p->ny, nz = p->nz, ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nbox = (long)p->nbx * p->nby * p->nbz, ca = nx * ny * nz, cg = ex * ey * ez;
    for (long b = 0; b < nbox; ++b)
    for (long k = 0; k < nz; ++k)
    for (long j = 0; j < ny; ++j)
    for (long i = 0; i < nx; ++i) {
        const long za = b * N * ca + (k * ny + j) * nx + i;
        const long zu = b * N * cg + ((k + ng) * ey + j + ng) * ex + i + ng;
        double cexp[5 + ORC_MAX_REACT] = { 0.0 };
        for (int c = 0; c < N; ++c) {
            double I = 0.0;
            for (int q = 0; q < nquad; ++q) I += w_quad[q] * (A_quad[q][za + c * ca] + R_quad[q][za + c * ca]);
            cexp[c] = ((U_m[zu + c * cg] + dt_m * (A_new_m[za + c * ca] - A_old_m[za + c * ca]))
                       - dt_m * R_old_next[za + c * ca]) + I;
        }
        const double rho = cexp[0];
        const double ke = 0.5 * (cexp[1] * cexp[1] + cexp[2] * cexp[2] + cexp[3] * cexp[3]) / rho;
        double cy[ORC_MAX_REACT + 1], y[ORC_MAX_REACT + 1], R[ORC_MAX_REACT + 1];
        for (int s = 0; s < ns; ++s) cy[s] = cexp[5 + s];
        cy[ns] = cexp[4];
        const int it = orc_react_solve_zone(r, ns, rho, ke, dt_m, cy, y);
        if (iters_out) iters_out[b * ca + (k * ny + j) * nx + i] = it;
        orc_react_zone(r, ns, rho, ke, y, R, NULL);
        for (int c = 0; c < 4; ++c) { U_next[zu + c * cg] = cexp[c]; R_new_out[za + c * ca] = 0.0; }
        U_next[zu + 4 * cg] = y[ns]; R_new_out[za + 4 * ca] = R[ns];
        for (int s = 0; s < ns; ++s) { U_next[zu + (5 + s) * cg] = y[s]; R_new_out[za + (5 + s) * ca] = R[s]; }
    }
    return ORC_OK;
}
