/*
 * oracle/orc_fourth.c -- CPU ORACLE (test infrastructure, NOT the product): the fourth-order finite-volume <A(U)>.
 *
 * "a fourth-order method in space and time (using a Simpsons rule for the integral and the spatial
 * reconstruction of [12])"; L60: "one less refinement level"; ref [12] (L91) = McCorquodale & Colella 2011.
 * SURVEY 8(f) NEXT-1.  [12] is not available here; the construction below is the standard fourth-order
 * finite-volume method of that line of work, restated as readings G1-G9, on cell AVERAGES <U> of a
 * uniform Cartesian grid (h_d = zone width along d; all second differences are undivided, so h^2/24 becomes 1/24):
 *  G1  cell-centre conserved state:  U^c = <U> - (1/24) sum_d (<U>_{+d} - 2 <U> + <U>_{-d});
 *  G2  q^c = prim(U^c) (point values);  qbar = prim(<U>) (a second-order stand-in for <q>), both by S1;
 *  G3  cell-average primitives:  <q> = q^c + (1/24) sum_d (qbar_{+d} - 2 qbar + qbar_{-d});
 *  G4  face averages along d:  <q>_{i+1/2} = (7/12)(<q>_i + <q>_{i+1}) - (1/12)(<q>_{i-1} + <q>_{i+2});
 *  G4b a face value that does not lie between its two zone averages, (q_{i+1/2} - q_i)(q_{i+1} - q_{i+1/2}) < 0, is
 *      rebuilt from a limited second difference (Colella & Sekora's first step, which the limiter of [12] builds on):
 *        D2 = 3 (q_i - 2 q_{i+1/2} + q_{i+1}),  D2L = q_{i-1} - 2 q_i + q_{i+1},  D2R = q_i - 2 q_{i+1} + q_{i+2};
 *        D2lim = s min(C |D2L|, C |D2R|, |D2|) if the three have one sign s, else 0;
 *        q_{i+1/2} = (q_i + q_{i+1}) / 2 - D2lim / 6      (D2lim = D2 gives the value back);
 *  G5  limiter of [12] section 2.4.1 (a variant of Colella & Sekora's extremum-preserving PPM limiter), zone by zone:
 *        d- = q_i - q_{i-1/2},  d+ = q_{i+1/2} - q_i;  the zone is an EXTREMUM if d- d+ <= 0 or
 *        (q_i - q_{i-2})(q_{i+2} - q_i) <= 0.
 *        extremum:  D2f = 6 (q_{i-1/2} - 2 q_i + q_{i+1/2}),  D2c_j = q_{j-1} - 2 q_j + q_{j+1} for j = i-1, i, i+1;
 *          if the four have one sign s:  D2lim = s min(C |D2c_{i-1}|, C |D2c_i|, C |D2c_{i+1}|, |D2f|), C = 1.25, else 0;
 *          rho = 0 if |D2f| <= 1e-12 max(|q_{i-2}| .. |q_{i+2}|), else D2lim / D2f;
 *          if rho < 1 - 1e-12:  if d- d+ < 0: d- <- rho d-, d+ <- rho d+;
 *                               else if |d-| >= 2 |d+|: d- <- 2 (1 - rho) d+ + rho d-;
 *                               else if |d+| >= 2 |d-|: d+ <- 2 (1 - rho) d- + rho d+;
 *        not an extremum:  if |d-| >= 2 |d+|: d- <- 2 d+;  else if |d+| >= 2 |d-|: d+ <- 2 d-;
 *        parabola edges  q_{i,-} = q_i - d-,  q_{i,+} = q_i + d+;  face states  W_L = q_{i,+},  W_R = q_{i+1,-}.
 *      [12] adds a test on third differences before limiting at an extremum; its stencil (q_{i-3} .. q_{i+3} for
 *      zones -1 .. n, i.e. <U> five zones outside the box) does not fit the 4-deep ghost shell of this build, so it
 *      is LEFT OUT -- a reading; smooth extrema keep their accuracy through rho (pin: fourth-order convergence);
 *  G6  face-centred states:  W^c = W - (1/24) sum_{d' != d} (W_{+d'} - 2 W + W_{-d'})   (each of W_L, W_R);
 *  G7  F^c = HLLC(W^c_L, W^c_R),  F^a = HLLC(W_L, W_R)  (S3, after the interface floors of S2 step 4 on both pairs);
 *      face-average flux:  <F> = F^c + (1/24) sum_{d' != d} (F^a_{+d'} - 2 F^a + F^a_{-d'});
 *  G8  <A> = -(((<F>x_{i+1/2} - <F>x_{i-1/2}) / dx + (y ...) / dy) + (z ...) / dz) + S,  S[rho v_d] = <rho> g_d,
 *      S[rho E] = sum_d <rho v_d> g_d  (exact cell averages for a constant g);
 *  G9  no flattening, no contact steepening on this path.
 * Transverse sums run in the order (lower direction + higher direction); everything reads at most the 4-deep shell,
 * edges and corners included (a face-ghost line needs <q> three zones out, and <q> needs <U> one zone further).
 * Pins (tests/test_oracle_fourth.py): fourth-order convergence of <A> to the exact finite-volume right-hand side of
 * an analytic smooth state (ratio -> 16 where the second-order path gives 4); A(uniform) = 0; conservation;
 * permutation / mirror invariance; box-lattice equivalence; limiter: smooth monotone data untouched, a step stays
 * monotone, smooth extremum keeps its height; the space-time scheme (3-node SDC, 4 iterations) at fourth order.
 * Unpinned by the paper itself (it only names ref [12]): G4b-G5 as recalled here, the omission of the third-difference
 * test, the flux form of G7 -- pinned only through the properties above.
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
void orc_hllc(int N, int d, double gamma, const double *WL, const double *WR, double *F);       /* orc.c, S3 */

/* G4 + G5 on one line: q[0..n-1] cell averages; for zones i = 2..n-3 the limited parabola edges qm[i] (at i-1/2)
 * and qp[i] (at i+1/2).  Entries outside that range are left untouched. */
void orc_ppm4_line(int n, const double *q, double *qm, double *qp)
{
    if (n < 5) return;
    double *qf = (double *)malloc(sizeof(double) * (size_t)n);        /* qf[i] = <q>_{i+1/2}, i = 1..n-3 */
    const double C = 1.25;
    for (int i = 1; i <= n - 3; ++i) {
        qf[i] = (7.0 / 12.0) * (q[i] + q[i + 1]) - (1.0 / 12.0) * (q[i - 1] + q[i + 2]);        /* G4 */
        if ((qf[i] - q[i]) * (q[i + 1] - qf[i]) < 0.0) {                                        /* G4b */
            const double D2 = 3.0 * ((q[i] - 2.0 * qf[i]) + q[i + 1]);
            const double D2L = (q[i - 1] - 2.0 * q[i]) + q[i + 1];
            const double D2R = (q[i] - 2.0 * q[i + 1]) + q[i + 2];
            double D2lim = 0.0;
            if (D2 > 0.0 && D2L > 0.0 && D2R > 0.0) {
                D2lim = C * D2L;
                if (C * D2R < D2lim) D2lim = C * D2R;
                if (D2 < D2lim) D2lim = D2;
            } else if (D2 < 0.0 && D2L < 0.0 && D2R < 0.0) {
                D2lim = C * D2L;
                if (C * D2R > D2lim) D2lim = C * D2R;
                if (D2 > D2lim) D2lim = D2;
            }
            qf[i] = 0.5 * (q[i] + q[i + 1]) - (1.0 / 6.0) * D2lim;
        }
    }
    for (int i = 2; i <= n - 3; ++i) {
        double dm = q[i] - qf[i - 1], dp = qf[i] - q[i];
        const int extremum = (dm * dp <= 0.0) || ((q[i] - q[i - 2]) * (q[i + 2] - q[i]) <= 0.0);
        if (extremum) {
            const double D2f = 6.0 * ((qf[i - 1] - 2.0 * q[i]) + qf[i]);
            const double D2l = (q[i - 2] - 2.0 * q[i - 1]) + q[i];
            const double D2c = (q[i - 1] - 2.0 * q[i]) + q[i + 1];
            const double D2r = (q[i] - 2.0 * q[i + 1]) + q[i + 2];
            double D2lim = 0.0;
            if (D2f > 0.0 && D2l > 0.0 && D2c > 0.0 && D2r > 0.0) {
                D2lim = C * D2l;
                if (C * D2c < D2lim) D2lim = C * D2c;
                if (C * D2r < D2lim) D2lim = C * D2r;
                if (D2f < D2lim) D2lim = D2f;
            } else if (D2f < 0.0 && D2l < 0.0 && D2c < 0.0 && D2r < 0.0) {
                D2lim = C * D2l;
                if (C * D2c > D2lim) D2lim = C * D2c;
                if (C * D2r > D2lim) D2lim = C * D2r;
                if (D2f > D2lim) D2lim = D2f;
            }
            double qmax = fabs(q[i - 2]);
            for (int j = i - 1; j <= i + 2; ++j) if (fabs(q[j]) > qmax) qmax = fabs(q[j]);
            const double rho = (fabs(D2f) <= 1e-12 * qmax) ? 0.0 : D2lim / D2f;
            if (rho < 1.0 - 1e-12) {
                if (dm * dp < 0.0) { dm = rho * dm; dp = rho * dp; }
                else if (fabs(dm) >= 2.0 * fabs(dp)) dm = 2.0 * (1.0 - rho) * dp + rho * dm;
                else if (fabs(dp) >= 2.0 * fabs(dm)) dp = 2.0 * (1.0 - rho) * dm + rho * dp;
            }
        } else {
            if (fabs(dm) >= 2.0 * fabs(dp)) dm = 2.0 * dp;
            else if (fabs(dp) >= 2.0 * fabs(dm)) dp = 2.0 * dm;
        }
        qm[i] = q[i] - dm;
        qp[i] = q[i] + dp;
    }
    free(qf);
}

static void floor_state(const orc_params *p, double *W)
{
    if (W[0] < p->small_dens) W[0] = p->small_dens;
    if (W[4] < p->small_pres) W[4] = p->small_pres;
}

/* <q> of every zone that has all six neighbours (G1-G3); qavg[c][z], ghosted layout of one box */
void orc_fourth_qavg(const orc_params *p, const double *Ub, double *qavg)
{
    const int ng = p->ng, N = 5 + p->nspec;
    const long ex = p->nx + 2 * ng, ey = p->ny + 2 * ng, ez = p->nz + 2 * ng, cg = ex * ey * ez;
    const long st[3] = { 1, ex, ex * ey };
    double *qbar = (double *)malloc(sizeof(double) * (size_t)(N * cg));
    #pragma omp parallel for schedule(static)
    for (long z = 0; z < cg; ++z) {
        double Uz[64], Wz[64];
        for (int c = 0; c < N; ++c) Uz[c] = Ub[c * cg + z];
        orc_cons_to_prim(N, p->gamma, p->small_pres, Uz, Wz);                                   /* G2: qbar */
        for (int c = 0; c < N; ++c) qbar[c * cg + z] = Wz[c];
    }
    #pragma omp parallel for schedule(static)
    for (long k = 1; k < ez - 1; ++k)
    for (long j = 1; j < ey - 1; ++j)
    for (long i = 1; i < ex - 1; ++i) {
        const long z = (k * ey + j) * ex + i;
        double Uc[64], qc[64];
        for (int c = 0; c < N; ++c) {
            const double *u = Ub + c * cg + z;
            const double lap = ((u[st[0]] - 2.0 * u[0] + u[-st[0]]) + (u[st[1]] - 2.0 * u[0] + u[-st[1]]))
                               + (u[st[2]] - 2.0 * u[0] + u[-st[2]]);
            Uc[c] = u[0] - (1.0 / 24.0) * lap;                                                  /* G1 */
        }
        orc_cons_to_prim(N, p->gamma, p->small_pres, Uc, qc);                                   /* G2: q^c */
        for (int c = 0; c < N; ++c) {
            const double *b = qbar + c * cg + z;
            const double lap = ((b[st[0]] - 2.0 * b[0] + b[-st[0]]) + (b[st[1]] - 2.0 * b[0] + b[-st[1]]))
                               + (b[st[2]] - 2.0 * b[0] + b[-st[2]]);
            qavg[c * cg + z] = qc[c] + (1.0 / 24.0) * lap;                                      /* G3 */
        }
    }
    free(qbar);
}

int orc_advance_A4(const orc_params *p, const double *U, double *A)
{
    if (!p || !U || !A || p->ng != 4 || p->nspec < 0 || 5 + p->nspec > 64) return -1;
    if (p->nx < p->ng || p->ny < p->ng || p->nz < p->ng) return -1;
    const int ng = p->ng, N = 5 + p->nspec;
    const int n[3] = { p->nx, p->ny, p->nz };
    const long ex = n[0] + 2 * ng, ey = n[1] + 2 * ng, ez = n[2] + 2 * ng, cg = ex * ey * ez;
    const long e[3] = { ex, ey, ez }, st[3] = { 1, ex, ex * ey };
    const double h[3] = { p->dx, p->dy, p->dz };
    const long nzone = (long)n[0] * n[1] * n[2];
    const long nbox = (long)p->nbx * p->nby * p->nbz;
    double *qavg = (double *)malloc(sizeof(double) * (size_t)(N * cg));
    /* per direction: states and F^a on faces f = 0..n_d of every line with transverse zones -1..n (m = n + 2 of them) */
    long fmax = 0;
    for (int d = 0; d < 3; ++d) {
        const int a = d == 0 ? 1 : 0, b = d == 2 ? 1 : 2;
        const long sz = (long)(n[d] + 1) * (n[a] + 2) * (n[b] + 2);
        if (sz > fmax) fmax = sz;
    }
    double *WL = (double *)malloc(sizeof(double) * (size_t)(N * fmax));
    double *WR = (double *)malloc(sizeof(double) * (size_t)(N * fmax));
    double *Fa = (double *)malloc(sizeof(double) * (size_t)(N * fmax));
    double *Fd[3];
    for (int d = 0; d < 3; ++d) Fd[d] = (double *)malloc(sizeof(double) * (size_t)N * (n[d] + 1) * (nzone / n[d]));
    if (!qavg || !WL || !WR || !Fa || !Fd[0] || !Fd[1] || !Fd[2]) return -2;

    for (long bx = 0; bx < nbox; ++bx) {
        const double *Ub = U + bx * N * cg;
        double *Ab = A + bx * N * nzone;
        orc_fourth_qavg(p, Ub, qavg);
        for (int d = 0; d < 3; ++d) {
            const int a = d == 0 ? 1 : 0, b = d == 2 ? 1 : 2;         /* transverse directions, a < b */
            const long nf = n[d] + 1, ma = n[a] + 2, mb = n[b] + 2;
            /* (i) limited face states on every line, transverse zones -1..n (index 0..m-1) */
            #pragma omp parallel
            {
                double *ql = (double *)malloc(sizeof(double) * (size_t)e[d]);
                double *qm = (double *)malloc(sizeof(double) * (size_t)e[d]);
                double *qp = (double *)malloc(sizeof(double) * (size_t)e[d]);
                #pragma omp for schedule(static)
                for (long ib = 0; ib < mb; ++ib)
                for (long ia = 0; ia < ma; ++ia) {
                    const long z0 = (ia + ng - 1) * st[a] + (ib + ng - 1) * st[b];
                    for (int c = 0; c < N; ++c) {
                        for (long i = 1; i < e[d] - 1; ++i) ql[i] = qavg[c * cg + z0 + i * st[d]];
                        ql[0] = ql[1]; ql[e[d] - 1] = ql[e[d] - 2];      /* never used: orc_ppm4_line reads 1 .. e-2 for zones 3 .. e-4 */
                        orc_ppm4_line((int)e[d] - 2, ql + 1, qm + 1, qp + 1);
                        for (long f = 0; f < nf; ++f) {
                            const long w = ((c * mb + ib) * ma + ia) * nf + f;
                            WL[w] = qp[f - 1 + ng];                    /* plus edge of zone f-1 */
                            WR[w] = qm[f + ng];                        /* minus edge of zone f  */
                        }
                    }
                }
                free(ql); free(qm); free(qp);
            }
            /* (ii) F^a on all those faces */
            #pragma omp parallel for schedule(static)
            for (long ib = 0; ib < mb; ++ib)
            for (long ia = 0; ia < ma; ++ia)
            for (long f = 0; f < nf; ++f) {
                double wl[64], wr[64], F[64];
                for (int c = 0; c < N; ++c) { const long w = ((c * mb + ib) * ma + ia) * nf + f; wl[c] = WL[w]; wr[c] = WR[w]; }
                floor_state(p, wl); floor_state(p, wr);
                orc_hllc(N, d, p->gamma, wl, wr, F);
                for (int c = 0; c < N; ++c) Fa[((c * mb + ib) * ma + ia) * nf + f] = F[c];
            }
            /* (iii) face-centred states, F^c, face-average flux on the faces of interior lines */
            #pragma omp parallel for schedule(static)
            for (long ib = 1; ib < mb - 1; ++ib)
            for (long ia = 1; ia < ma - 1; ++ia)
            for (long f = 0; f < nf; ++f) {
                double wl[64], wr[64], Fc[64];
                const long sa = nf, sb = ma * nf;
                for (int c = 0; c < N; ++c) {
                    const long w = ((c * mb + ib) * ma + ia) * nf + f;
                    wl[c] = WL[w] - (1.0 / 24.0) * ((WL[w + sa] - 2.0 * WL[w] + WL[w - sa]) + (WL[w + sb] - 2.0 * WL[w] + WL[w - sb]));
                    wr[c] = WR[w] - (1.0 / 24.0) * ((WR[w + sa] - 2.0 * WR[w] + WR[w - sa]) + (WR[w + sb] - 2.0 * WR[w] + WR[w - sb]));   /* G6 */
                }
                floor_state(p, wl); floor_state(p, wr);
                orc_hllc(N, d, p->gamma, wl, wr, Fc);
                for (int c = 0; c < N; ++c) {
                    const long w = ((c * mb + ib) * ma + ia) * nf + f;
                    const double lap = (Fa[w + sa] - 2.0 * Fa[w] + Fa[w - sa]) + (Fa[w + sb] - 2.0 * Fa[w] + Fa[w - sb]);
                    Fd[d][((c * (long)n[b] + (ib - 1)) * n[a] + (ia - 1)) * nf + f] = Fc[c] + (1.0 / 24.0) * lap;                        /* G7 */
                }
            }
        }
        /* (iv) divergence + source (G8) */
        #pragma omp parallel for schedule(static)
        for (long k = 0; k < n[2]; ++k)
        for (long j = 0; j < n[1]; ++j)
        for (long i = 0; i < n[0]; ++i) {
            const long zg = ((k + ng) * ey + (j + ng)) * ex + (i + ng);
            const double rho = Ub[zg], mx = Ub[cg + zg], my = Ub[2 * cg + zg], mz = Ub[3 * cg + zg];
            for (int c = 0; c < N; ++c) {
                const double *fx = Fd[0] + ((c * (long)n[2] + k) * n[1] + j) * (n[0] + 1) + i;      /* a = y, b = z */
                const double *fy = Fd[1] + ((c * (long)n[2] + k) * n[0] + i) * (n[1] + 1) + j;      /* a = x, b = z */
                const double *fz = Fd[2] + ((c * (long)n[1] + j) * n[0] + i) * (n[2] + 1) + k;      /* a = x, b = y */
                double S = 0.0;
                if (c == 1) S = rho * p->grav[0];
                else if (c == 2) S = rho * p->grav[1];
                else if (c == 3) S = rho * p->grav[2];
                else if (c == 4) S = (mx * p->grav[0] + my * p->grav[1]) + mz * p->grav[2];
                Ab[(c * (long)n[2] + k) * n[1] * n[0] + j * n[0] + i] =
                    -(((fx[1] - fx[0]) / h[0] + (fy[1] - fy[0]) / h[1]) + (fz[1] - fz[0]) / h[2]) + S;
            }
        }
    }
    free(qavg); free(WL); free(WR); free(Fa);
    for (int d = 0; d < 3; ++d) free(Fd[d]);
    return 0;
}
