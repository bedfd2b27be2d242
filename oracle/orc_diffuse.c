/*
 * oracle/orc_diffuse.c -- CPU ORACLE (test infrastructure, NOT the product): explicit thermal diffusion as an extra
 * term of the advective operator ("thermal diffusion" among the solvers that run on the GPU; L62:
 * "hydrodynamics, explicit diffusion ..." in the XRB runs).
 *
 * The paper's conductivities need tables that are not available; the reading (D1-D3) is
 *   D1  constant conductivity k_th and a constant c_v:  d(rho E)/dt += div(k_th grad T) = k_th lap T;
 *   D2  T is the temperature of the gamma-law state that S1 produces:  T = p / ((gamma - 1) rho c_v) with
 *       p = max((gamma - 1)(rho E - rho |v|^2 / 2), small_pres);
 *   D3  second-order centred differences of the zone values, summed in the order ((x + y) + z):
 *       D = k_th [ (T_{i+1} - 2 T_i + T_{i-1}) / dx^2 + (...) / dy^2 + (...) / dz^2 ];
 *       only the +-1 star is read (face ghosts), only the energy component of A changes.
 * Pins (tests/test_oracle_diffuse.py): D of a uniform-temperature state is exactly zero; sum of D over a periodic
 * domain vanishes to roundoff; for T = T0 + a sin(2 pi m x / L) the result converges to -k_th (2 pi m / L)^2 (T - T0)
 * at second order; the discrete eigenvalue -k_th (2 - 2 cos(theta)) / dx^2 is met to roundoff.
 * Unpinned by the paper itself: constant k_th and c_v (D1-D2 stand in for its conductivity tables).
 */
#include <math.h>

typedef struct {
    int nx, ny, nz, ng, nbx, nby, nbz, nspec;
    double dx, dy, dz, gamma, grav[3];
    int bc_lo[3], bc_hi[3];
    double small_dens, small_pres;
} orc_params;                                  /* same layout as in orc.c */

static double temperature(const orc_params *p, double cv, const double *U, long z, long cg)
{
    const double rho = U[z], mx = U[z + cg], my = U[z + 2 * cg], mz = U[z + 3 * cg], E = U[z + 4 * cg];
    const double u = mx / rho, v = my / rho, w = mz / rho;
    double pr = (p->gamma - 1.0) * (E - 0.5 * rho * (u * u + v * v + w * w));
    if (pr < p->small_pres) pr = p->small_pres;
    return pr / ((p->gamma - 1.0) * rho * cv);              /* D2 */
}

/* D[b][k][j][i] (interior zones, one value per zone) <- k_th lap T;  U ghosts must be filled. */
int orc_diffusion(const orc_params *p, double kth, double cv, const double *U, double *D)
{
    if (!p || !U || !D || p->ng != 4 || !(cv > 0)) return -1;
    const int ng = p->ng, N = 5 + p->nspec;
    const long nx = p->nx, ny = p->ny, nz = p->nz, ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nbox = (long)p->nbx * p->nby * p->nbz, cg = ex * ey * ez;
    for (long b = 0; b < nbox; ++b)
    for (long k = 0; k < nz; ++k)
    for (long j = 0; j < ny; ++j)
    for (long i = 0; i < nx; ++i) {
        const long z = b * N * cg + ((k + ng) * ey + j + ng) * ex + i + ng;
        const double T0 = temperature(p, cv, U, z, cg);
        const double lx = (temperature(p, cv, U, z + 1, cg) - 2.0 * T0 + temperature(p, cv, U, z - 1, cg)) / (p->dx * p->dx);
        const double ly = (temperature(p, cv, U, z + ex, cg) - 2.0 * T0 + temperature(p, cv, U, z - ex, cg)) / (p->dy * p->dy);
        const double lz = (temperature(p, cv, U, z + ex * ey, cg) - 2.0 * T0 + temperature(p, cv, U, z - ex * ey, cg)) / (p->dz * p->dz);
        D[((b * nz + k) * ny + j) * nx + i] = kth * ((lx + ly) + lz);      /* D3 */
    }
    return 0;
}
