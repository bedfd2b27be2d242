/*
 * oracle/orc.c -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, step-by-step fp64 implementation of the hot path of
 * arXiv:1910.12578 (Zingale et al., "The Castro AMR Simulation Code"):
 * ghost fill, the finite-volume advective term <A(U)> of Eq. (1)
 * ("the divergence of the hydrodynamic fluxes along with
 * hydrodynamic sources"), the SDC node update Eq. (2) with
 * R = 0, and the CFL reduction.  The paper states only Eq. (1)-(2); every
 * formula below the level of those equations follows the readings listed in
 * DESIGN.md section 3 (Q1..Q29), each cited at the
 * function that implements it.
 *
 * Rules this file obeys:
 *  - only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 *    --impl reference legs may load it; the product path never does;
 *  - it shares no code, header, table or helper with paper_1910_12578_b200/csrc;
 *  - straight loops in the order the text states, no blocking, no fusion;
 *    build with -O2 -ffp-contract=off (no FMA contraction, no fast-math);
 *  - OpenMP (optional) only around outermost plane loops, so that the timed
 *    CPU baseline can use the host's cores; results do not depend on it.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): exact Sod Riemann solution
 * (P1,P2), conservation (P3), A(uniform)=0 (P4), HLLC special cases (P5,P6),
 * permutation/mirror invariance (P7), species identity (P8), cubic edge
 * exactness (P9), limiter bounds (P10), hydrostatic residual order (P11),
 * Heun / Simpson (P12), box-lattice equivalence + brute-force ghost map (P13),
 * CFL closed form (P14), 2nd-order convergence (P15); the M-node SDC driver of orc.py: order rises by one per
 * iteration up to the order of the quadrature on U' = lambda U; tests/golden/oracle_tiny_case.txt
 * freezes the arithmetic of this file (written by tests/golden/make_golden.py from the oracle only).
 * Round 2 (tests/test_oracle_pins2.py): the shock branch of the wave-speed estimate (orc_wave_speeds fed the
 * exact star pressure returns the exact shock speed: textbook Sod value and the Rankine-Hugoniot mass
 * condition on random shocks), orc_hllc against the textbook HLLC written out on those speeds, and the
 * interface floors of line_fluxes against a brute-force restatement with floors that bind.
 * Unpinned by the paper itself (conventions only): the CHOICE of the PVRS wave-speed estimate,
 * CW84-vs-other limiter, method-of-lines-vs-CTU -- see DESIGN.md.
 *
 * Data layout: U[b][c][k][j][i] on ghosted extents
 * (n+2*ng), i fastest; A[b][c][k][j][i] on interior extents.  Component order
 * c = 0 rho, 1 rho*u, 2 rho*v, 3 rho*w, 4 rho*E, 5+s rho*X_s.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int nx, ny, nz;          /* interior zones per box */
    int ng;                  /* ghost width (4) */
    int nbx, nby, nbz;       /* box lattice */
    int nspec;
    double dx, dy, dz;
    double gamma;
    double grav[3];
    int bc_lo[3], bc_hi[3];  /* 0 periodic, 1 outflow, 2 reflecting */
    double small_dens, small_pres;
} orc_params;

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2 };
enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_REFLECT = 2 };

static int check_params(const orc_params *p)
{
    if (!p) return ORC_EINVAL;
    if (p->ng != 4) return ORC_EINVAL;
    if (p->nx < p->ng || p->ny < p->ng || p->nz < p->ng) return ORC_EINVAL;
    if (p->nbx < 1 || p->nby < 1 || p->nbz < 1 || p->nspec < 0) return ORC_EINVAL;
    if (!(p->dx > 0) || !(p->dy > 0) || !(p->dz > 0) || !(p->gamma > 1)) return ORC_EINVAL;
    for (int d = 0; d < 3; ++d) {
        if (p->bc_lo[d] < 0 || p->bc_lo[d] > 2 || p->bc_hi[d] < 0 || p->bc_hi[d] > 2) return ORC_EINVAL;
        if ((p->bc_lo[d] == BC_PERIODIC) != (p->bc_hi[d] == BC_PERIODIC)) return ORC_EINVAL; /* Q29 */
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------ S0 --- */
/* Ghost fill ("grids"/"boxes"; BCs: DESIGN.md Q16).
 * For a ghost zone with GLOBAL index g along one direction of a domain of D
 * zones: periodic s = g mod D; outflow s = clamp(g,0,D-1); reflecting
 * s = -1-g (low) or 2D-1-g (high) and the momentum normal to that wall
 * changes sign.  The map is applied direction by direction, which fills
 * edges and corners consistently. */
static long map_index(long g, long D, int bc_lo, int bc_hi, int *flip)
{
    *flip = 0;
    if (g >= 0 && g < D) return g;
    if (g < 0) {
        if (bc_lo == BC_PERIODIC) return ((g % D) + D) % D;
        if (bc_lo == BC_OUTFLOW) return 0;
        *flip = 1;
        return -1 - g;
    }
    if (bc_hi == BC_PERIODIC) return g % D;
    if (bc_hi == BC_OUTFLOW) return D - 1;
    *flip = 1;
    return 2 * D - 1 - g;
}

int orc_fill_ghosts(const orc_params *p, double *U)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!U) return ORC_EINVAL;
    const int ng = p->ng, N = 5 + p->nspec;
    const long ex = p->nx + 2 * ng, ey = p->ny + 2 * ng, ez = p->nz + 2 * ng;
    const long Dx = (long)p->nbx * p->nx, Dy = (long)p->nby * p->ny, Dz = (long)p->nbz * p->nz;
    const long box_stride = (long)N * ez * ey * ex;
    for (int bk = 0; bk < p->nbz; ++bk)
    for (int bj = 0; bj < p->nby; ++bj)
    for (int bi = 0; bi < p->nbx; ++bi) {
        const long b = bi + (long)p->nbx * (bj + (long)p->nby * bk);
        for (int c = 0; c < N; ++c)
        for (long k = 0; k < ez; ++k)
        for (long j = 0; j < ey; ++j)
        for (long i = 0; i < ex; ++i) {
            const long li = i - ng, lj = j - ng, lk = k - ng;  /* local interior index */
            if (li >= 0 && li < p->nx && lj >= 0 && lj < p->ny && lk >= 0 && lk < p->nz) continue;
            int fx, fy, fz;
            const long sx = map_index((long)bi * p->nx + li, Dx, p->bc_lo[0], p->bc_hi[0], &fx);
            const long sy = map_index((long)bj * p->ny + lj, Dy, p->bc_lo[1], p->bc_hi[1], &fy);
            const long sz = map_index((long)bk * p->nz + lk, Dz, p->bc_lo[2], p->bc_hi[2], &fz);
            const long sb = (sx / p->nx) + (long)p->nbx * ((sy / p->ny) + (long)p->nby * (sz / p->nz));
            const long si = sx % p->nx + ng, sj = sy % p->ny + ng, sk = sz % p->nz + ng;
            double v = U[sb * box_stride + ((c * ez + sk) * ey + sj) * ex + si];
            if ((c == 1 && fx) || (c == 2 && fy) || (c == 3 && fz)) v = -v;
            U[b * box_stride + ((c * ez + k) * ey + j) * ex + i] = v;
        }
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------ S1 --- */
/* Conserved -> primitive with a gamma-law EOS (BASELINE north_star; Q10-Q12).
 * W = (rho, u, v, w, p, X_s);  p = (gamma-1)(rhoE - rho|v|^2/2), floored at
 * small_pres; rho is not floored at zone centres (Q11). */
void orc_cons_to_prim(int N, double gamma, double small_pres, const double *Uz, double *Wz)
{
    const double rho = Uz[0];
    const double r = 1.0 / rho;
    const double u = Uz[1] * r, v = Uz[2] * r, w = Uz[3] * r;
    double pr = (gamma - 1.0) * (Uz[4] - 0.5 * rho * (u * u + v * v + w * w));
    if (pr < small_pres) pr = small_pres;
    Wz[0] = rho; Wz[1] = u; Wz[2] = v; Wz[3] = w; Wz[4] = pr;
    for (int s = 5; s < N; ++s) Wz[s] = Uz[s] * r;
}

/* ------------------------------------------------------------------ S2 --- */
/* PPM reconstruction of one scalar along one line (PAPER.md L52 cites CW84 =
 * ref [15]; uniform-grid form of CW84 eqs (1.6)-(1.10); Q1-Q5: method of
 * lines, primitive variables, original CW84 limiter, no flattening, no
 * contact steepening).
 * Input q[0..n-1].  Output, for zones i = 2..n-3, the parabola edge values
 * qm[i] (at i-1/2) and qp[i] (at i+1/2).  Entries outside that range are
 * left untouched. */
static double limited_slope(double qm1, double q0, double qp1)
{
    /* CW84 (1.7)-(1.8) */
    const double dp = qp1 - q0, dm = q0 - qm1;
    const double dc = 0.5 * (dp + dm);
    if (dp * dm > 0.0) {
        double a = fabs(dc);
        const double b = 2.0 * fabs(dp), c = 2.0 * fabs(dm);
        if (b < a) a = b;
        if (c < a) a = c;
        return dc > 0.0 ? a : -a;
    }
    return 0.0;
}

void orc_ppm_line(int n, const double *q, double *qm, double *qp)
{
    if (n < 5) return;
    double *dq = (double *)malloc(sizeof(double) * (size_t)n);
    double *ed = (double *)malloc(sizeof(double) * (size_t)n);   /* ed[i] = q_{i+1/2} */
    for (int i = 1; i <= n - 2; ++i) dq[i] = limited_slope(q[i - 1], q[i], q[i + 1]);
    /* CW84 (1.6), uniform grid */
    for (int i = 1; i <= n - 3; ++i)
        ed[i] = 0.5 * (q[i] + q[i + 1]) - (1.0 / 6.0) * (dq[i + 1] - dq[i]);
    for (int i = 2; i <= n - 3; ++i) {
        double a = ed[i - 1], b = ed[i];       /* q-, q+ */
        const double qc = q[i];
        /* CW84 (1.10); both later tests use the pre-modification a, b */
        if ((b - qc) * (qc - a) <= 0.0) {
            a = qc; b = qc;
        } else {
            const double D = b - a;
            const double q6 = 6.0 * (qc - 0.5 * (a + b));
            if (D * q6 > D * D)       a = 3.0 * qc - 2.0 * b;
            else if (-(D * D) > D * q6) b = 3.0 * qc - 2.0 * a;
        }
        qm[i] = a; qp[i] = b;
    }
    free(dq); free(ed);
}

/* --------------------------------------------------- S2b (optional) --- */
/* Shock flattening (CW84 appendix; "[15, 16]").  OFF on the graded
 * path (orc_advance_A); orc_advance_A_flat switches it on.  Readings F1-F4:
 *  F1  along direction d, with u the velocity component along d:
 *        dp = p_{i+1} - p_{i-1},  dp2 = p_{i+2} - p_{i-2},  z = |dp| / max(|dp2|, small_pres),
 *        chi~_i = clamp(1 - (z - 0.75) / (0.85 - 0.75), 0, 1)   if the zone sits in a shock, i.e.
 *        u_{i-1} - u_{i+1} >= 0 (compression) and |dp| / min(p_{i+1}, p_{i-1}) > 1/3;  else chi~_i = 1;
 *  F2  chi^d_i = min(chi~_i, chi~_{i+s}),  s = -1 if dp > 0 else +1  (the neighbour on the low-pressure side);
 *  F3  chi_i = min over the three directions of chi^d_i;
 *  F4  every parabola of the zone, in every direction and for every variable:  q+- <- chi q+- + (1 - chi) q.
 * orc_flatten_tilde: chi~ for zones i = 2..n-3 of one line (others untouched);
 * orc_flatten_line : chi^d for zones i = 3..n-4 of one line. */
void orc_flatten_tilde(int n, const double *p, const double *u, double small_pres, double *ct)
{
    for (int i = 2; i <= n - 3; ++i) {
        const double dp = p[i + 1] - p[i - 1], dp2 = p[i + 2] - p[i - 2];
        const double den = fabs(dp2) > small_pres ? fabs(dp2) : small_pres;
        const double z = fabs(dp) / den;
        double zeta = 1.0 - (z - 0.75) / (0.85 - 0.75);
        if (zeta < 0.0) zeta = 0.0;
        if (zeta > 1.0) zeta = 1.0;
        const double pmin = p[i + 1] < p[i - 1] ? p[i + 1] : p[i - 1];
        const int shock = (u[i - 1] - u[i + 1] >= 0.0) && (fabs(dp) / pmin > 1.0 / 3.0);
        ct[i] = shock ? zeta : 1.0;
    }
}

void orc_flatten_line(int n, const double *p, const double *u, double small_pres, double *chi)
{
    double *ct = (double *)malloc(sizeof(double) * (size_t)n);
    orc_flatten_tilde(n, p, u, small_pres, ct);
    for (int i = 3; i <= n - 4; ++i) {
        const double dp = p[i + 1] - p[i - 1];
        const double nb = dp > 0.0 ? ct[i - 1] : ct[i + 1];
        chi[i] = ct[i] < nb ? ct[i] : nb;
    }
    free(ct);
}

/* ------------------------------------------------------------------ S3 --- */
/* HLLC flux through a face whose normal is direction d (0,1,2)
 * (BASELINE north_star names HLLC; construction: Toro ch. 10; pressure-based
 * PVRS wave speeds Q6; tie-breaks Q7; species as mass flux x upwind X, Q8).
 * WL, WR: N primitives (rho,u,v,w,p,X_s) already floored.  F: N fluxes.
 *
 * Star state written with the ratio r = (S_K - u_K)/(S_K - S*) so that a
 * stationary contact (S* = u_K = 0) gives r = 1 and U*_K = U_K exactly
 * (pin P6; Q7b):
 *   rho* = rho_K r,  (rho v)* = rho* (v with normal component -> S*),
 *   E*   = r [E_K + (S* - u_K)(rho_K S* + p_K/(S_K - u_K))]. */
/* Wave-speed estimate of the HLLC solver (Q6; Toro ch. 10, pressure-based): given the two normal
 * states and an estimate ps of the star pressure,
 *   S_L = u_L - c_L q_L,  S_R = u_R + c_R q_R,  q_K = 1 if ps <= p_K (rarefaction)
 *   else sqrt(1 + (gamma+1)/(2 gamma) (ps/p_K - 1)) (shock).
 * Exported on its own so that the shock branch can be pinned: fed the EXACT star pressure it
 * returns the exact shock speed (tests/test_oracle_pins.py, Sod: 1.752156). */
void orc_wave_speeds(double gamma, double rL, double uL, double pL, double rR, double uR, double pR,
                     double ps, double *SL_out, double *SR_out)
{
    const double cL = sqrt(gamma * pL / rL), cR = sqrt(gamma * pR / rR);
    const double gfac = (gamma + 1.0) / (2.0 * gamma);
    const double qL = (ps <= pL) ? 1.0 : sqrt(1.0 + gfac * (ps / pL - 1.0));
    const double qR = (ps <= pR) ? 1.0 : sqrt(1.0 + gfac * (ps / pR - 1.0));
    *SL_out = uL - cL * qL;
    *SR_out = uR + cR * qR;
}

/* PVRS estimate of the star pressure (Toro (9.20)/(10.67)), floored at 0. */
double orc_pvrs_pstar(double gamma, double rL, double uL, double pL, double rR, double uR, double pR)
{
    const double cL = sqrt(gamma * pL / rL), cR = sqrt(gamma * pR / rR);
    const double ppv = 0.5 * (pL + pR) - 0.5 * (uR - uL) * (0.5 * (rL + rR)) * (0.5 * (cL + cR));
    return ppv > 0.0 ? ppv : 0.0;
}

void orc_hllc(int N, int d, double gamma, const double *WL, const double *WR, double *F)
{
    const double rL = WL[0], rR = WR[0], pL = WL[4], pR = WR[4];
    const double uL = WL[1 + d], uR = WR[1 + d];
    const double ps = orc_pvrs_pstar(gamma, rL, uL, pL, rR, uR, pR);
    double SL, SR;
    orc_wave_speeds(gamma, rL, uL, pL, rR, uR, pR, ps, &SL, &SR);
    const double Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR))
                    / (rL * (SL - uL) - rR * (SR - uR));
    const double *W; double SK;
    if (Ss >= 0.0) { W = WL; SK = SL; } else { W = WR; SK = SR; }
    const double rho = W[0], un = W[1 + d], pr = W[4];
    const double vel[3] = { W[1], W[2], W[3] };
    const double E = pr / (gamma - 1.0) + 0.5 * rho * (vel[0] * vel[0] + vel[1] * vel[1] + vel[2] * vel[2]);
    double UK[5] = { rho, rho * vel[0], rho * vel[1], rho * vel[2], E };
    double FK[5];
    for (int c = 0; c < 5; ++c) FK[c] = un * UK[c];
    FK[1 + d] += pr;
    FK[4] += pr * un;
    const int pure = (W == WL) ? (SL >= 0.0) : (SR <= 0.0);
    if (pure) {
        for (int c = 0; c < 5; ++c) F[c] = FK[c];
    } else {
        const double r = (SK - un) / (SK - Ss);
        double vs[3] = { vel[0], vel[1], vel[2] };
        vs[d] = Ss;
        const double rs = rho * r;
        double US[5];
        US[0] = rs; US[1] = rs * vs[0]; US[2] = rs * vs[1]; US[3] = rs * vs[2];
        US[4] = r * (E + (Ss - un) * (rho * Ss + pr / (SK - un)));
        for (int c = 0; c < 5; ++c) F[c] = FK[c] + SK * (US[c] - UK[c]);
    }
    for (int s = 5; s < N; ++s) F[s] = F[0] * W[s];
}

/* -------------------------------------------------------------- S1-S4 --- */
/* <A(U)> on every box.  Per box, in the order of
 * DESIGN.md "oracle loop structure":
 *  (1) W on the whole ghosted box;
 *  (2) for each direction: every line through the box is reconstructed
 *      (orc_ppm_line on the ghosted line), interface states at face f
 *      (between zones f-1 and f, f = 0..n) are W_L = W+_{f-1}, W_R = W-_f,
 *      floored (rho >= small_dens, p >= small_pres), HLLC -> F^d_f;
 *  (3) A_c = -[(Fx_{i+1}-Fx_i)/dx + (Fy_{j+1}-Fy_j)/dy + (Fz_{k+1}-Fz_k)/dz] + S_c,
 *      summed ((x+y)+z) (Q13);  S[rho v_d] = rho g_d,
 *      S[rho E] = sum_d (rho v_d) g_d from the zone-centre U (Q14). */
static void line_fluxes(const orc_params *p, int d, int n, const double *Wline /* [N][n+2ng] */,
                        double *Fline /* [N][n+1] */, double *scr, const double *chiline /* [n+2ng] or NULL */)
{
    const int ng = p->ng, N = 5 + p->nspec, e = n + 2 * ng;
    double *qm = scr, *qp = scr + (size_t)N * e;
    for (int c = 0; c < N; ++c)
        orc_ppm_line(e, Wline + (size_t)c * e, qm + (size_t)c * e, qp + (size_t)c * e);
    if (chiline)                                     /* F4: zones -1 .. n carry the parabolas the faces use */
        for (int c = 0; c < N; ++c)
        for (int i = ng - 1; i <= n + ng; ++i) {
            const double x = chiline[i], q = Wline[(size_t)c * e + i];
            qm[(size_t)c * e + i] = x * qm[(size_t)c * e + i] + (1.0 - x) * q;
            qp[(size_t)c * e + i] = x * qp[(size_t)c * e + i] + (1.0 - x) * q;
        }
    double WL[64], WR[64], F[64];
    for (int f = 0; f <= n; ++f) {
        const int zl = f - 1 + ng, zr = f + ng;   /* ghosted indices of the two zones */
        for (int c = 0; c < N; ++c) { WL[c] = qp[(size_t)c * e + zl]; WR[c] = qm[(size_t)c * e + zr]; }
        if (WL[0] < p->small_dens) WL[0] = p->small_dens;
        if (WR[0] < p->small_dens) WR[0] = p->small_dens;
        if (WL[4] < p->small_pres) WL[4] = p->small_pres;
        if (WR[4] < p->small_pres) WR[4] = p->small_pres;
        orc_hllc(N, d, p->gamma, WL, WR, F);
        for (int c = 0; c < N; ++c) Fline[(size_t)c * (n + 1) + f] = F[c];
    }
}

static int advance_A_impl(const orc_params *p, const double *U, double *A, int flatten)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!U || !A) return ORC_EINVAL;
    const int ng = p->ng, N = 5 + p->nspec;
    if (N > 64) return ORC_EINVAL;
    const int nx = p->nx, ny = p->ny, nz = p->nz;
    const long ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nzone_g = ex * ey * ez, nzone = (long)nx * ny * nz;
    const long nbox = (long)p->nbx * p->nby * p->nbz;
    double *W  = (double *)malloc(sizeof(double) * (size_t)(N * nzone_g));
    double *Fx = (double *)malloc(sizeof(double) * (size_t)N * (nx + 1) * ny * nz);
    double *Fy = (double *)malloc(sizeof(double) * (size_t)N * nx * (ny + 1) * nz);
    double *Fz = (double *)malloc(sizeof(double) * (size_t)N * nx * ny * (nz + 1));
    double *chi = flatten ? (double *)malloc(sizeof(double) * (size_t)nzone_g) : NULL;
    if (!W || !Fx || !Fy || !Fz || (flatten && !chi)) { free(W); free(Fx); free(Fy); free(Fz); free(chi); return ORC_ENOMEM; }
    long emax = ex > ey ? ex : ey; if (ez > emax) emax = ez;

    for (long b = 0; b < nbox; ++b) {
        const double *Ub = U + b * N * nzone_g;
        double *Ab = A + b * N * nzone;
        /* (1) primitives everywhere */
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < ez; ++k) {
            double Uz[64], Wz[64];
            for (long j = 0; j < ey; ++j)
            for (long i = 0; i < ex; ++i) {
                const long z = (k * ey + j) * ex + i;
                for (int c = 0; c < N; ++c) Uz[c] = Ub[c * nzone_g + z];
                orc_cons_to_prim(N, p->gamma, p->small_pres, Uz, Wz);
                for (int c = 0; c < N; ++c) W[c * nzone_g + z] = Wz[c];
            }
        }
        /* (1b) optional flattening coefficient on zones -1 .. n of every direction (F1-F3); needs the whole shell */
        if (flatten) {
            for (long z = 0; z < nzone_g; ++z) chi[z] = 1.0;
            double *pl = (double *)malloc(sizeof(double) * (size_t)emax), *ul = (double *)malloc(sizeof(double) * (size_t)emax);
            double *cl = (double *)malloc(sizeof(double) * (size_t)emax);
            for (int d = 0; d < 3; ++d) {
                const long e_d = d == 0 ? ex : d == 1 ? ey : ez, st = d == 0 ? 1 : d == 1 ? ex : ex * ey;
                const long ea = d == 0 ? ey : ex, eb = d == 2 ? ey : ez;          /* the two other extents */
                const long sa = d == 0 ? ex : 1, sb = d == 2 ? ex : ex * ey;      /* and their strides */
                for (long bb = ng - 1; bb <= eb - ng; ++bb)
                for (long aa = ng - 1; aa <= ea - ng; ++aa) {
                    const long z0 = aa * sa + bb * sb;
                    for (long i = 0; i < e_d; ++i) { pl[i] = W[4 * nzone_g + z0 + i * st]; ul[i] = W[(1 + d) * nzone_g + z0 + i * st]; }
                    orc_flatten_line((int)e_d, pl, ul, p->small_pres, cl);
                    for (long i = ng - 1; i <= e_d - ng; ++i)
                        if (cl[i] < chi[z0 + i * st]) chi[z0 + i * st] = cl[i];        /* F3 */
                }
            }
            free(pl); free(ul); free(cl);
        }
        /* (2) fluxes, direction by direction */
        #pragma omp parallel
        {
            double *Wl = (double *)malloc(sizeof(double) * (size_t)N * emax);
            double *Cl = (double *)malloc(sizeof(double) * (size_t)emax);
            double *Fl = (double *)malloc(sizeof(double) * (size_t)N * emax);
            double *sc = (double *)malloc(sizeof(double) * (size_t)2 * N * emax);
            /* x lines */
            #pragma omp for schedule(static)
            for (long k = 0; k < nz; ++k)
            for (long j = 0; j < ny; ++j) {
                for (int c = 0; c < N; ++c)
                for (long i = 0; i < ex; ++i)
                    Wl[c * ex + i] = W[c * nzone_g + ((k + ng) * ey + (j + ng)) * ex + i];
                if (chi) for (long i = 0; i < ex; ++i) Cl[i] = chi[((k + ng) * ey + (j + ng)) * ex + i];
                line_fluxes(p, 0, nx, Wl, Fl, sc, chi ? Cl : NULL);
                for (int c = 0; c < N; ++c)
                for (long f = 0; f <= nx; ++f)
                    Fx[((c * (long)nz + k) * ny + j) * (nx + 1) + f] = Fl[c * (nx + 1) + f];
            }
            /* y lines */
            #pragma omp for schedule(static)
            for (long k = 0; k < nz; ++k)
            for (long i = 0; i < nx; ++i) {
                for (int c = 0; c < N; ++c)
                for (long j = 0; j < ey; ++j)
                    Wl[c * ey + j] = W[c * nzone_g + ((k + ng) * ey + j) * ex + (i + ng)];
                if (chi) for (long j = 0; j < ey; ++j) Cl[j] = chi[((k + ng) * ey + j) * ex + (i + ng)];
                line_fluxes(p, 1, ny, Wl, Fl, sc, chi ? Cl : NULL);
                for (int c = 0; c < N; ++c)
                for (long f = 0; f <= ny; ++f)
                    Fy[((c * (long)nz + k) * (ny + 1) + f) * nx + i] = Fl[c * (ny + 1) + f];
            }
            /* z lines */
            #pragma omp for schedule(static)
            for (long j = 0; j < ny; ++j)
            for (long i = 0; i < nx; ++i) {
                for (int c = 0; c < N; ++c)
                for (long k = 0; k < ez; ++k)
                    Wl[c * ez + k] = W[c * nzone_g + (k * ey + (j + ng)) * ex + (i + ng)];
                if (chi) for (long k = 0; k < ez; ++k) Cl[k] = chi[(k * ey + (j + ng)) * ex + (i + ng)];
                line_fluxes(p, 2, nz, Wl, Fl, sc, chi ? Cl : NULL);
                for (int c = 0; c < N; ++c)
                for (long f = 0; f <= nz; ++f)
                    Fz[((c * (long)(nz + 1) + f) * ny + j) * nx + i] = Fl[c * (nz + 1) + f];
            }
            free(Wl); free(Fl); free(sc); free(Cl);
        }
        /* (3) divergence + source */
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < nz; ++k)
        for (long j = 0; j < ny; ++j)
        for (long i = 0; i < nx; ++i) {
            const long zg = ((k + ng) * ey + (j + ng)) * ex + (i + ng);
            const double rho = Ub[zg];
            const double mx = Ub[1 * nzone_g + zg], my = Ub[2 * nzone_g + zg], mz = Ub[3 * nzone_g + zg];
            for (int c = 0; c < N; ++c) {
                const double fxl = Fx[((c * (long)nz + k) * ny + j) * (nx + 1) + i];
                const double fxh = Fx[((c * (long)nz + k) * ny + j) * (nx + 1) + i + 1];
                const double fyl = Fy[((c * (long)nz + k) * (ny + 1) + j) * nx + i];
                const double fyh = Fy[((c * (long)nz + k) * (ny + 1) + j + 1) * nx + i];
                const double fzl = Fz[((c * (long)(nz + 1) + k) * ny + j) * nx + i];
                const double fzh = Fz[((c * (long)(nz + 1) + k + 1) * ny + j) * nx + i];
                double S = 0.0;
                if (c == 1) S = rho * p->grav[0];
                else if (c == 2) S = rho * p->grav[1];
                else if (c == 3) S = rho * p->grav[2];
                else if (c == 4) S = (mx * p->grav[0] + my * p->grav[1]) + mz * p->grav[2];
                Ab[(c * (long)nz + k) * ny * nx + j * nx + i] =
                    -(((fxh - fxl) / p->dx + (fyh - fyl) / p->dy) + (fzh - fzl) / p->dz) + S;
            }
        }
    }
    free(W); free(Fx); free(Fy); free(Fz); free(chi);
    return ORC_OK;
}

int orc_advance_A(const orc_params *p, const double *U, double *A)
{
    return advance_A_impl(p, U, A, 0);
}

/* <A(U)> with CW84 shock flattening switched on (readings F1-F4 above); reads the WHOLE 4-deep shell (edges and
 * corners included: the coefficient of a face-ghost zone looks three zones sideways). */
int orc_advance_A_flat(const orc_params *p, const double *U, double *A)
{
    return advance_A_impl(p, U, A, 1);
}

/* ------------------------------------------------------------------ S5 --- */
/* SDC node update, Eq. (2) of the paper with R = 0:
 *   U^{m+1,(k+1)} = U^{m,(k+1)} + dt_m [A^{m,(k+1)} - A^{m,(k)}] + I_m^{(k)},
 *   I_m^{(k)} = sum_j w_quad[j] * A_quad[j]   (weights already times dt; Q17).
 * Interior zones only; ghosts of U_next are left untouched (Q28). */
int orc_sdc_update(const orc_params *p, double *U_next, const double *U_m, double dt_m,
                   const double *A_new_m, const double *A_old_m,
                   int nquad, const double *const *A_quad, const double *w_quad)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!U_next || !U_m || !A_new_m || !A_old_m || nquad < 0 || (nquad > 0 && (!A_quad || !w_quad)))
        return ORC_EINVAL;
    const int ng = p->ng, N = 5 + p->nspec;
    const long nx = p->nx, ny = p->ny, nz = p->nz;
    const long ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nbox = (long)p->nbx * p->nby * p->nbz;
    for (long b = 0; b < nbox; ++b)
    for (int c = 0; c < N; ++c) {
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < nz; ++k)
        for (long j = 0; j < ny; ++j)
        for (long i = 0; i < nx; ++i) {
            const long za = ((b * N + c) * nz + k) * ny * nx + j * nx + i;
            const long zu = (((b * N + c) * ez + k + ng) * ey + j + ng) * ex + i + ng;
            double I = 0.0;
            for (int q = 0; q < nquad; ++q) I += w_quad[q] * A_quad[q][za];
            U_next[zu] = (U_m[zu] + dt_m * (A_new_m[za] - A_old_m[za])) + I;
        }
    }
    return ORC_OK;
}

/* ------------------------------------------------------------------ S6 --- */
/* CFL time step (BASELINE north_star; sum form, Q20):
 *   dt = cfl / max_zones [ (|u|+c)/dx + (|v|+c)/dy + (|w|+c)/dz ],
 * c = sqrt(gamma p / rho), interior zones of all boxes. */
int orc_cfl_dt(const orc_params *p, const double *U, double cfl, double *dt_out)
{
    int rc = check_params(p);
    if (rc) return rc;
    if (!U || !dt_out) return ORC_EINVAL;
    const int ng = p->ng, N = 5 + p->nspec;
    const long nx = p->nx, ny = p->ny, nz = p->nz;
    const long ex = nx + 2 * ng, ey = ny + 2 * ng, ez = nz + 2 * ng;
    const long nzone_g = ex * ey * ez;
    const long nbox = (long)p->nbx * p->nby * p->nbz;
    double smax = 0.0;
    for (long b = 0; b < nbox; ++b) {
        const double *Ub = U + b * N * nzone_g;
        for (long k = 0; k < nz; ++k)
        for (long j = 0; j < ny; ++j)
        for (long i = 0; i < nx; ++i) {
            const long z = ((k + ng) * ey + (j + ng)) * ex + (i + ng);
            double Uz[5], Wz[5];
            for (int c = 0; c < 5; ++c) Uz[c] = Ub[c * nzone_g + z];
            orc_cons_to_prim(5, p->gamma, p->small_pres, Uz, Wz);
            const double cs = sqrt(p->gamma * Wz[4] / Wz[0]);
            const double s = ((fabs(Wz[1]) + cs) / p->dx + (fabs(Wz[2]) + cs) / p->dy)
                           + (fabs(Wz[3]) + cs) / p->dz;
            if (s > smax) smax = s;
        }
    }
    *dt_out = cfl / smax;
    return ORC_OK;
}

/* ------------------------------------------------- exact Riemann (pins) --- */
/* Exact solution of the 1-D Riemann problem for an ideal gas (Toro ch. 4):
 * Newton iteration on f(p) = f_L(p) + f_R(p) + (u_R - u_L) = 0, then sampling
 * at xi = x/t.  Used only as the closed-form pin P1/P2 and for the config[1]
 * physics check.  out5 = (p*, u*, rho*_L, rho*_R, iterations). */
static double f_K(double p, double rK, double pK, double g, double *df)
{
    const double cK = sqrt(g * pK / rK);
    if (p > pK) {             /* shock */
        const double AK = 2.0 / ((g + 1.0) * rK), BK = (g - 1.0) / (g + 1.0) * pK;
        const double s = sqrt(AK / (p + BK));
        *df = s * (1.0 - 0.5 * (p - pK) / (BK + p));
        return (p - pK) * s;
    }                         /* rarefaction */
    const double pr = p / pK;
    *df = pow(pr, -(g + 1.0) / (2.0 * g)) / (rK * cK);
    return 2.0 * cK / (g - 1.0) * (pow(pr, (g - 1.0) / (2.0 * g)) - 1.0);
}

int orc_exact_riemann_star(double g, double rL, double uL, double pL,
                           double rR, double uR, double pR, double *out5)
{
    const double cL = sqrt(g * pL / rL), cR = sqrt(g * pR / rR);
    double p = 0.5 * (pL + pR);
    /* two-rarefaction start, always positive */
    const double z = (g - 1.0) / (2.0 * g);
    p = pow((cL + cR - 0.5 * (g - 1.0) * (uR - uL)) / (cL / pow(pL, z) + cR / pow(pR, z)), 1.0 / z);
    int it = 0;
    for (; it < 100; ++it) {
        double dL, dR;
        const double f = f_K(p, rL, pL, g, &dL) + f_K(p, rR, pR, g, &dR) + (uR - uL);
        double pn = p - f / (dL + dR);
        if (pn <= 0.0) pn = 1e-14 * p + 1e-300;
        const double ch = 2.0 * fabs(pn - p) / (pn + p);
        p = pn;
        if (ch < 1e-15) break;
    }
    double dL, dR;
    const double fl = f_K(p, rL, pL, g, &dL), fr = f_K(p, rR, pR, g, &dR);
    const double us = 0.5 * (uL + uR) + 0.5 * (fr - fl);
    const double gm = (g - 1.0) / (g + 1.0);
    out5[0] = p; out5[1] = us;
    out5[2] = (p > pL) ? rL * ((p / pL + gm) / (gm * p / pL + 1.0)) : rL * pow(p / pL, 1.0 / g);
    out5[3] = (p > pR) ? rR * ((p / pR + gm) / (gm * p / pR + 1.0)) : rR * pow(p / pR, 1.0 / g);
    out5[4] = (double)it;
    return ORC_OK;
}

/* Sample (rho,u,p) of the exact solution at n similarity coordinates xi = x/t. */
int orc_exact_riemann_sample(double g, double rL, double uL, double pL,
                             double rR, double uR, double pR,
                             int n, const double *xi, double *rho, double *u, double *pr)
{
    double st[5];
    orc_exact_riemann_star(g, rL, uL, pL, rR, uR, pR, st);
    const double ps = st[0], us = st[1], rsL = st[2], rsR = st[3];
    const double cL = sqrt(g * pL / rL), cR = sqrt(g * pR / rR);
    for (int m = 0; m < n; ++m) {
        const double s = xi[m];
        double r_, u_, p_;
        if (s <= us) {                         /* left of the contact */
            if (ps > pL) {                     /* left shock */
                const double SL = uL - cL * sqrt((g + 1.0) / (2.0 * g) * ps / pL + (g - 1.0) / (2.0 * g));
                if (s <= SL) { r_ = rL; u_ = uL; p_ = pL; } else { r_ = rsL; u_ = us; p_ = ps; }
            } else {                           /* left rarefaction */
                const double head = uL - cL, csL = cL * pow(ps / pL, (g - 1.0) / (2.0 * g)), tail = us - csL;
                if (s <= head) { r_ = rL; u_ = uL; p_ = pL; }
                else if (s >= tail) { r_ = rsL; u_ = us; p_ = ps; }
                else {
                    const double c = 2.0 / (g + 1.0) * (cL + 0.5 * (g - 1.0) * (uL - s));
                    u_ = 2.0 / (g + 1.0) * (cL + 0.5 * (g - 1.0) * uL + s);
                    r_ = rL * pow(c / cL, 2.0 / (g - 1.0));
                    p_ = pL * pow(c / cL, 2.0 * g / (g - 1.0));
                }
            }
        } else {                               /* right of the contact */
            if (ps > pR) {
                const double SR = uR + cR * sqrt((g + 1.0) / (2.0 * g) * ps / pR + (g - 1.0) / (2.0 * g));
                if (s >= SR) { r_ = rR; u_ = uR; p_ = pR; } else { r_ = rsR; u_ = us; p_ = ps; }
            } else {
                const double head = uR + cR, csR = cR * pow(ps / pR, (g - 1.0) / (2.0 * g)), tail = us + csR;
                if (s >= head) { r_ = rR; u_ = uR; p_ = pR; }
                else if (s <= tail) { r_ = rsR; u_ = us; p_ = ps; }
                else {
                    const double c = 2.0 / (g + 1.0) * (cR - 0.5 * (g - 1.0) * (uR - s));
                    u_ = 2.0 / (g + 1.0) * (-cR + 0.5 * (g - 1.0) * uR + s);
                    r_ = rR * pow(c / cR, 2.0 / (g - 1.0));
                    p_ = pR * pow(c / cR, 2.0 * g / (g - 1.0));
                }
            }
        }
        rho[m] = r_; u[m] = u_; pr[m] = p_;
    }
    return ORC_OK;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
