/*
 * oracle/orc_ctu.c -- CPU ORACLE (test infrastructure, NOT the product): the unsplit CTU PPM advective operator.
 *
 * "the main unsplit PPM hydrodynamics scheme [15, 16]" -- the hydro solver the paper's GPU port runs on
 * the Strang path: PPM reconstruction with characteristic tracing to the half time (ref [15], Colella & Woodward
 * 1984) and corner-transport-upwind transverse corrections (ref [16], Miller & Colella 2002).  SURVEY 8(f) NEXT-2 (ii):
 * "a second A-like kernel".  Neither reference is available here; the scheme is restated as readings C1-C9.
 * Unlike <A(U)> of the SDC path it depends on the time step:  A_ctu(U, dt) = -div F^{n+1/2} + S,  U^{n+1} = U^n + dt A_ctu.
 *  C1  W = (rho, u, v, w, p, X_k) by S1 in every zone of the 4-deep shell; c = sqrt(gamma p / rho).
 *  C2  along each direction d the CW84 parabola (q-, q+) of every primitive (S2 steps 1-3; no flattening here).
 *  C3  characteristic tracing (CW84 (1.12); [16]).  With Dq = q+ - q-, q6 = 6 (q - (q- + q+)/2) and, for a wave of speed
 *      lambda, sigma = |lambda| dt / Delta_d:
 *        I+(sigma) = q+ - (sigma/2) (Dq - (1 - 2 sigma/3) q6)    average over the part of the zone the wave carries to face i+1/2,
 *        I-(sigma) = q- + (sigma/2) (Dq + (1 - 2 sigma/3) q6)    ... to face i-1/2.
 *      State the zone sends to its PLUS face (left state of face i+1/2), with u the velocity along d:
 *        reference state  q~ = I+(sigma_{u+c}) if u + c > 0 else q (zone average), for rho, u, p;
 *        a+ = (1/2)(dp/(rho c) + du) rho/c with (du, dp) = q~ - I+(sigma_{u+c}), kept only if u + c > 0;
 *        a- = (1/2)(dp/(rho c) - du) rho/c with (du, dp) = q~ - I+(sigma_{u-c}), kept only if u - c > 0;
 *        a0 = drho - dp/c^2           with (drho, dp) = q~ - I+(sigma_u),       kept only if u > 0;
 *        rho_L = rho~ - (a+ + a- + a0),  u_L = u~ - (a+ - a-) c/rho,  p_L = p~ - (a+ + a-) c^2
 *        (rho, c of the zone average); transverse velocities and X_k ride on the u wave: I+(sigma_u) if u > 0 else q.
 *      State it sends to its MINUS face (right state of face i-1/2): the mirror image -- q~ = I-(sigma_{u-c}) if u - c < 0
 *      else q; a-, a0, a+ from I-(sigma) of the waves with NEGATIVE speed (u - c < 0, u < 0, u + c < 0); passives I-(sigma_u)
 *      if u < 0 else q.
 *  C4  gravity enters the traced states as (dt/2) g added to the three velocity components.
 *  C5  F^d = HLLC(W_L, W_R) (S3) after the interface floors of S2 step 4, on every face whose two zones carry states.
 *  C6  first transverse correction, in conserved variables: for each ordered pair d != d',
 *        U^{d|d'} = cons(W^d) - (dt / (3 Delta_d')) (F^d'_{+1/2} - F^d'_{-1/2})   (the zone's own two d' faces),
 *      back to primitives by S1, floors, F^{d|d'} = HLLC.
 *  C7  final states: with d' < d'' the two other directions,
 *        U^{d,fin} = (cons(W^d) - (dt / (2 Delta_d')) (F^{d'|d''}_{+} - F^{d'|d''}_{-})) - (dt / (2 Delta_d'')) (F^{d''|d'}_{+} - F^{d''|d'}_{-}),
 *      back to primitives, floors, F^{d,fin} = HLLC.
 *  C8  A_ctu = -(((Fx_{i+1/2} - Fx_{i-1/2})/dx + (Fy ...)/dy) + (Fz ...)/dz) + S with the zone-centre gravity source of S4.
 *  C9  cons(W): rho, rho v, p/(gamma-1) + rho |v|^2 / 2, rho X_k.
 * Reads the whole 4-deep shell (edges and corners).  Pins (tests/test_oracle_ctu.py): pure advection with
 * dt = dx/u = dy/v = dz/w is an EXACT shift by one zone along the diagonal (every coefficient of C3, C6, C7 enters);
 * 1-D Sod against the exact Riemann solution at CFL 0.8 (the acoustic part of C3); second-order convergence in 3-D at
 * CFL 0.8 where the method-of-lines operator with one Euler stage is unstable; conservation, A(uniform) = 0,
 * permutation / mirror invariance, box-lattice equivalence.
 * Unpinned by the paper itself (it only names refs [15, 16]): the choice of reference state and of zone-centre
 * eigenvectors in C3, the passive treatment of transverse velocities, the source placement of C4 / C8 -- conventions,
 * fixed by the readings and pinned only through the properties above.
 * Shares no code with paper_1910_12578_b200/csrc.
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

void orc_cons_to_prim(int N, double gamma, double small_pres, const double *Uz, double *Wz);    /* orc.c, S1 */
void orc_ppm_line(int n, const double *q, double *qm, double *qp);                              /* orc.c, S2 */
void orc_hllc(int N, int d, double gamma, const double *WL, const double *WR, double *F);       /* orc.c, S3 */

static double Iplus(double qm, double qp, double q, double sigma)
{
    const double Dq = qp - qm, q6 = 6.0 * (q - 0.5 * (qm + qp));
    return qp - 0.5 * sigma * (Dq - (1.0 - (2.0 / 3.0) * sigma) * q6);
}
static double Iminus(double qm, double qp, double q, double sigma)
{
    const double Dq = qp - qm, q6 = 6.0 * (q - 0.5 * (qm + qp));
    return qm + 0.5 * sigma * (Dq + (1.0 - (2.0 / 3.0) * sigma) * q6);
}

/* C3 + C4 for one zone and one direction.  W, qm, qp: N values each (zone average and parabola edges);
 * Wp <- the state sent to the plus face, Wm <- the state sent to the minus face. */
void orc_ctu_trace_zone(int N, int d, double gamma, double dtdx, double hdt, const double *grav,
                        const double *W, const double *qm, const double *qp, double *Wm, double *Wp)
{
    const double rho = W[0], u = W[1 + d], p = W[4];
    const double c = sqrt(gamma * p / rho);
    const double lam[3] = { u - c, u, u + c };
    double sig[3];
    for (int k = 0; k < 3; ++k) sig[k] = fabs(lam[k]) * dtdx;
    const int iv[3] = { 0, 1 + d, 4 };                    /* rho, normal velocity, p */
    for (int side = 0; side < 2; ++side) {               /* 0: minus face, 1: plus face */
        double I[3][3];                                   /* [wave][rho, u, p] */
        for (int k = 0; k < 3; ++k)
            for (int v = 0; v < 3; ++v)
                I[k][v] = side ? Iplus(qm[iv[v]], qp[iv[v]], W[iv[v]], sig[k]) : Iminus(qm[iv[v]], qp[iv[v]], W[iv[v]], sig[k]);
        const int kref = side ? 2 : 0;                    /* the fastest wave towards the face */
        const int towards[3] = { side ? lam[0] > 0.0 : lam[0] < 0.0, side ? lam[1] > 0.0 : lam[1] < 0.0,
                                 side ? lam[2] > 0.0 : lam[2] < 0.0 };
        double ref[3];
        for (int v = 0; v < 3; ++v) ref[v] = towards[kref] ? I[kref][v] : W[iv[v]];
        double ap = 0.0, am = 0.0, a0 = 0.0;
        if (towards[2]) { const double du = ref[1] - I[2][1], dp = ref[2] - I[2][2]; ap = 0.5 * (dp / (rho * c) + du) * rho / c; }
        if (towards[0]) { const double du = ref[1] - I[0][1], dp = ref[2] - I[0][2]; am = 0.5 * (dp / (rho * c) - du) * rho / c; }
        if (towards[1]) { const double dr = ref[0] - I[1][0], dp = ref[2] - I[1][2]; a0 = dr - dp / (c * c); }
        double *out = side ? Wp : Wm;
        out[0] = ref[0] - ((ap + am) + a0);
        out[1 + d] = ref[1] - (ap - am) * c / rho;
        out[4] = ref[2] - (ap + am) * (c * c);
        for (int s = 1; s < N; ++s) {                      /* passives: transverse velocities and species */
            if (s == 1 + d || s == 4) continue;
            out[s] = towards[1] ? (side ? Iplus(qm[s], qp[s], W[s], sig[1]) : Iminus(qm[s], qp[s], W[s], sig[1])) : W[s];
        }
        for (int e = 0; e < 3; ++e) out[1 + e] += hdt * grav[e];                                  /* C4 */
    }
}

static void prim_to_cons(int N, double gamma, const double *W, double *U)                       /* C9 */
{
    const double rho = W[0];
    U[0] = rho; U[1] = rho * W[1]; U[2] = rho * W[2]; U[3] = rho * W[3];
    U[4] = W[4] / (gamma - 1.0) + 0.5 * rho * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
    for (int s = 5; s < N; ++s) U[s] = rho * W[s];
}

static void floor_state(const orc_params *p, double *W)
{
    if (W[0] < p->small_dens) W[0] = p->small_dens;
    if (W[4] < p->small_pres) W[4] = p->small_pres;
}

typedef struct { int lo[3], hi[3]; } range3;                 /* inclusive zone coordinates (-4 .. n+3) per direction */

/* flux at the LOW d-face of every zone in r from the zone states Sm (this zone) and Sp (its low neighbour) */
static void riemann_faces(const orc_params *p, int N, int d, const long *st, long cg, range3 r,
                          const double *Sm, const double *Sp, double *F)
{
    const int ng = p->ng;
    for (int k = r.lo[2]; k <= r.hi[2]; ++k)
    for (int j = r.lo[1]; j <= r.hi[1]; ++j)
    for (int i = r.lo[0]; i <= r.hi[0]; ++i) {
        const long z = (k + ng) * st[2] + (j + ng) * st[1] + (i + ng);
        double wl[64], wr[64], f[64];
        for (int c = 0; c < N; ++c) { wl[c] = Sp[c * cg + z - st[d]]; wr[c] = Sm[c * cg + z]; }
        floor_state(p, wl); floor_state(p, wr);                                                   /* C5 */
        orc_hllc(N, d, p->gamma, wl, wr, f);
        for (int c = 0; c < N; ++c) F[c * cg + z] = f[c];
    }
}

/* C6 / C7: out = prim(cons(S) - sum_t coef[t] (Ft[t](z + e_dt[t]) - Ft[t](z))) for both states of every zone in r */
static void correct_states(const orc_params *p, int N, const long *st, long cg, range3 r, int nt, const int *dt_, const double *coef,
                           const double *const *Ft, const double *Sm, const double *Sp, double *Om, double *Op)
{
    const int ng = p->ng;
    for (int k = r.lo[2]; k <= r.hi[2]; ++k)
    for (int j = r.lo[1]; j <= r.hi[1]; ++j)
    for (int i = r.lo[0]; i <= r.hi[0]; ++i) {
        const long z = (k + ng) * st[2] + (j + ng) * st[1] + (i + ng);
        for (int side = 0; side < 2; ++side) {
            const double *S = side ? Sp : Sm;
            double *O = side ? Op : Om;
            double W[64], U[64], Wn[64];
            for (int c = 0; c < N; ++c) W[c] = S[c * cg + z];
            prim_to_cons(N, p->gamma, W, U);
            for (int t = 0; t < nt; ++t)
                for (int c = 0; c < N; ++c)
                    U[c] = U[c] - coef[t] * (Ft[t][c * cg + z + st[dt_[t]]] - Ft[t][c * cg + z]);
            orc_cons_to_prim(N, p->gamma, p->small_pres, U, Wn);
            for (int c = 0; c < N; ++c) O[c * cg + z] = Wn[c];
        }
    }
}

int orc_advance_ctu(const orc_params *p, const double *U, double dt, double *A)
{
    if (!p || !U || !A || p->ng != 4 || p->nspec < 0 || 5 + p->nspec > 64 || !(dt >= 0.0)) return -1;
    const int ng = p->ng, N = 5 + p->nspec;
    const int n[3] = { p->nx, p->ny, p->nz };
    if (n[0] < ng || n[1] < ng || n[2] < ng) return -1;
    const long e[3] = { n[0] + 2 * ng, n[1] + 2 * ng, n[2] + 2 * ng };
    const long st[3] = { 1, e[0], e[0] * e[1] }, cg = e[0] * e[1] * e[2];
    const double h[3] = { p->dx, p->dy, p->dz };
    const long nzone = (long)n[0] * n[1] * n[2], nbox = (long)p->nbx * p->nby * p->nbz;
    const size_t sz = sizeof(double) * (size_t)(N * cg);
    double *W = (double *)malloc(sz);
    double *Sm[3], *Sp[3], *F1[3], *Tm[3][3], *Tp[3][3], *Ft[3][3], *Gm[3], *Gp[3], *Ff[3];
    for (int d = 0; d < 3; ++d) {
        Sm[d] = (double *)malloc(sz); Sp[d] = (double *)malloc(sz); F1[d] = (double *)malloc(sz);
        Gm[d] = (double *)malloc(sz); Gp[d] = (double *)malloc(sz); Ff[d] = (double *)malloc(sz);
        for (int t = 0; t < 3; ++t) {
            Tm[d][t] = Tp[d][t] = Ft[d][t] = NULL;
            if (t != d) { Tm[d][t] = (double *)malloc(sz); Tp[d][t] = (double *)malloc(sz); Ft[d][t] = (double *)malloc(sz); }
        }
    }
    long emax = e[0] > e[1] ? e[0] : e[1]; if (e[2] > emax) emax = e[2];
    double *ql = (double *)malloc(sizeof(double) * (size_t)(3 * N * emax));

    for (long b = 0; b < nbox; ++b) {
        const double *Ub = U + b * N * cg;
        double *Ab = A + b * N * nzone;
        for (long z = 0; z < cg; ++z) {                                                           /* C1 */
            double Uz[64], Wz[64];
            for (int c = 0; c < N; ++c) Uz[c] = Ub[c * cg + z];
            orc_cons_to_prim(N, p->gamma, p->small_pres, Uz, Wz);
            for (int c = 0; c < N; ++c) W[c * cg + z] = Wz[c];
        }
        /* C2-C4: traced states of zones -1 .. n in every coordinate, for every direction */
        for (int d = 0; d < 3; ++d) {
            const int a = (d + 1) % 3, bb = (d + 2) % 3;
            for (int ib = -1; ib <= n[bb]; ++ib)
            for (int ia = -1; ia <= n[a]; ++ia) {
                const long z0 = (ia + ng) * st[a] + (ib + ng) * st[bb];
                double *q = ql, *qm = ql + N * emax, *qp = ql + 2 * N * emax;
                for (int c = 0; c < N; ++c) {
                    for (long i = 0; i < e[d]; ++i) q[c * emax + i] = W[c * cg + z0 + i * st[d]];
                    orc_ppm_line((int)e[d], q + c * emax, qm + c * emax, qp + c * emax);
                }
                for (int i = -1; i <= n[d]; ++i) {
                    double Wz[64], qmz[64], qpz[64], wm[64], wp[64];
                    for (int c = 0; c < N; ++c) { Wz[c] = q[c * emax + i + ng]; qmz[c] = qm[c * emax + i + ng]; qpz[c] = qp[c * emax + i + ng]; }
                    orc_ctu_trace_zone(N, d, p->gamma, dt / h[d], 0.5 * dt, p->grav, Wz, qmz, qpz, wm, wp);
                    const long z = z0 + (i + ng) * st[d];
                    for (int c = 0; c < N; ++c) { Sm[d][c * cg + z] = wm[c]; Sp[d][c * cg + z] = wp[c]; }
                }
            }
        }
        /* C5: one-dimensional fluxes at the low d-face of zones 0 .. n along d, -1 .. n across */
        for (int d = 0; d < 3; ++d) {
            range3 r;
            for (int t = 0; t < 3; ++t) { r.lo[t] = (t == d) ? 0 : -1; r.hi[t] = n[t]; }
            riemann_faces(p, N, d, st, cg, r, Sm[d], Sp[d], F1[d]);
        }
        /* C6: states corrected by ONE transverse flux difference, and their fluxes */
        for (int d = 0; d < 3; ++d)
        for (int t = 0; t < 3; ++t) {
            if (t == d) continue;
            const int o = 3 - d - t;                          /* the third direction */
            range3 r;
            r.lo[d] = -1; r.hi[d] = n[d]; r.lo[t] = 0; r.hi[t] = n[t] - 1; r.lo[o] = -1; r.hi[o] = n[o];
            const double coef[1] = { dt / (3.0 * h[t]) };
            const double *Fs[1] = { F1[t] };
            const int dts[1] = { t };
            correct_states(p, N, st, cg, r, 1, dts, coef, Fs, Sm[d], Sp[d], Tm[d][t], Tp[d][t]);
            r.lo[d] = 0;
            riemann_faces(p, N, d, st, cg, r, Tm[d][t], Tp[d][t], Ft[d][t]);
        }
        /* C7: final states and fluxes */
        for (int d = 0; d < 3; ++d) {
            const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;       /* the two other directions, t1 < t2 */
            range3 r;
            r.lo[d] = -1; r.hi[d] = n[d]; r.lo[t1] = 0; r.hi[t1] = n[t1] - 1; r.lo[t2] = 0; r.hi[t2] = n[t2] - 1;
            const double coef[2] = { dt / (2.0 * h[t1]), dt / (2.0 * h[t2]) };
            const double *Fs[2] = { Ft[t1][t2], Ft[t2][t1] };
            const int dts[2] = { t1, t2 };
            correct_states(p, N, st, cg, r, 2, dts, coef, Fs, Sm[d], Sp[d], Gm[d], Gp[d]);
            r.lo[d] = 0;
            riemann_faces(p, N, d, st, cg, r, Gm[d], Gp[d], Ff[d]);
        }
        /* C8 */
        for (long k = 0; k < n[2]; ++k)
        for (long j = 0; j < n[1]; ++j)
        for (long i = 0; i < n[0]; ++i) {
            const long z = (k + ng) * st[2] + (j + ng) * st[1] + (i + ng);
            const double rho = Ub[z], mx = Ub[cg + z], my = Ub[2 * cg + z], mz = Ub[3 * cg + z];
            for (int c = 0; c < N; ++c) {
                const double *fx = Ff[0] + c * cg + z, *fy = Ff[1] + c * cg + z, *fz = Ff[2] + c * cg + z;
                double S = 0.0;
                if (c == 1) S = rho * p->grav[0];
                else if (c == 2) S = rho * p->grav[1];
                else if (c == 3) S = rho * p->grav[2];
                else if (c == 4) S = (mx * p->grav[0] + my * p->grav[1]) + mz * p->grav[2];
                Ab[(c * (long)n[2] + k) * n[1] * n[0] + j * n[0] + i] =
                    -(((fx[st[0]] - fx[0]) / h[0] + (fy[st[1]] - fy[0]) / h[1]) + (fz[st[2]] - fz[0]) / h[2]) + S;
            }
        }
    }
    free(W); free(ql);
    for (int d = 0; d < 3; ++d) {
        free(Sm[d]); free(Sp[d]); free(F1[d]); free(Gm[d]); free(Gp[d]); free(Ff[d]);
        for (int t = 0; t < 3; ++t) if (t != d) { free(Tm[d][t]); free(Tp[d][t]); free(Ft[d][t]); }
    }
    return 0;
}
