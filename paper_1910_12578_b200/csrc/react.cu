// react.cu -- the reactive half of Eq. (1)-(2) ("implicit reaction updates", L31-40; SURVEY 8(f)
// NEXT-3; include/cst.h cst_set_reactions, cst_react_R, cst_sdc_update_react).
//
// Eq. (2) is implicit in U^{m+1,(k+1)} through R only:   U' = c + dt_m R(U'),
//   c = U_m + dt_m (A_new_m - A_old_m) - dt_m R^{m+1,(k)} + sum_q w_q (A_q + R_q).
// R is the synthetic stiff chain of DESIGN.md readings R1-R4 (the paper's 13-isotope network needs rate tables that
// are not available): X_0 -> X_1 -> ... with lambda_k(T) = rate_k (T/T0)^nu, T = e / c_v, energy release q_k.
// rho and rho v have no reactive source, so they are explicit; the ns + 1 unknowns y = (rho X_k, rho E) of a zone are
// found by Newton's method, one thread per zone, everything in registers:
//   the Newton matrix I - dt dR/dy is lower BIDIAGONAL in the species (each reaction feeds the next species) plus a
//   last column (the rates' temperature dependence) and a last row (the energy release).  Writing the species
//   corrections as d_k = alpha_k + beta_k d_E turns the elimination into two forward recurrences and one scalar
//   division for d_E: O(ns) operations and registers instead of a dense (ns+1)^2 factorisation in local memory.
//   (The diagonal 1 + dt lambda_k >= 1 dominates, so no pivoting is needed.)
// Convergence test and first iterate are those of the readings: start from c, stop when the last correction is
// <= tol relative to (rho | |rho E|), at most max_iter iterations; zones that do not converge are counted.
#include "common.cuh"

struct ReactDev {
    double cv, T0, nu, tol;
    int max_iter, ns;
    double rate[CST_MAX_REACT], q[CST_MAX_REACT];
};

// rates and their temperature derivative at the state (y_E, rho, ke)
__device__ __forceinline__ void react_rates(const ReactDev& r, double rho, double ke, double yE,
                                            double (&lam)[CST_MAX_REACT], double& dlnlam_dE)
{
    const double rcv = 1.0 / (rho * r.cv);
    const double T = (yE - ke) * rcv;
    const double f = pow(T / r.T0, r.nu);
#pragma unroll
    for (int k = 0; k < CST_MAX_REACT; ++k) lam[k] = (k < r.ns - 1) ? r.rate[k] * f : 0.0;
    dlnlam_dE = r.nu / T * rcv;                          // (d lambda / d(rho E)) / lambda
}

__device__ __forceinline__ void react_rhs(const ReactDev& r, const double (&lam)[CST_MAX_REACT],
                                          const double (&y)[CST_MAX_REACT], double (&R)[CST_MAX_REACT], double& RE)
{
    RE = 0.0;
#pragma unroll
    for (int k = 0; k < CST_MAX_REACT; ++k) {
        if (k < r.ns) {
            const double out = lam[k] * y[k];
            R[k] = ((k > 0) ? lam[k > 0 ? k - 1 : 0] * y[k > 0 ? k - 1 : 0] : 0.0) - out;
            RE = fma(r.q[k], out, RE);
        } else {
            R[k] = 0.0;
        }
    }
}

__global__ void __launch_bounds__(128)
k_react_R(Geom g, ReactDev r, const double* __restrict__ U, double* __restrict__ Rout)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long b = r2 / g.nz;
        const long long zu = b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const long long za = b * g.box_a + ((long long)k * g.ny + j) * g.nx + i;
        const double rho = U[zu], mx = U[zu + g.comp_g], my = U[zu + 2 * g.comp_g], mz = U[zu + 3 * g.comp_g];
        const double ke = 0.5 * (mx * mx + my * my + mz * mz) / rho;
        double y[CST_MAX_REACT], lam[CST_MAX_REACT], R[CST_MAX_REACT], RE, dl;
#pragma unroll
        for (int s = 0; s < CST_MAX_REACT; ++s) y[s] = (s < r.ns) ? U[zu + (5 + s) * g.comp_g] : 0.0;
        react_rates(r, rho, ke, U[zu + 4 * g.comp_g], lam, dl);
        react_rhs(r, lam, y, R, RE);
#pragma unroll
        for (int c = 0; c < 4; ++c) Rout[za + c * g.comp_a] = 0.0;
        Rout[za + 4 * g.comp_a] = RE;
#pragma unroll
        for (int s = 0; s < CST_MAX_REACT; ++s) if (s < r.ns) Rout[za + (5 + s) * g.comp_a] = R[s];
    }
}

struct ReactQuad {           // quadrature arrays of A and R, passed by value
    int nquad;
    const double* A[CST_MAX_QUAD];
    const double* R[CST_MAX_QUAD];
    double w[CST_MAX_QUAD];
};

__global__ void __launch_bounds__(128)
k_sdc_update_react(Geom g, ReactDev r, double* U_next, const double* U_m, double dt,
                   const double* __restrict__ A_new, const double* __restrict__ A_old,
                   const double* R_old_next, ReactQuad q, double* R_new,      // may be the same array (cst.h)
                   unsigned long long* __restrict__ n_fail)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long b = r2 / g.nz;
        const long long zu = b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const long long za = b * g.box_a + ((long long)k * g.ny + j) * g.nx + i;
        // the explicit part c of Eq. (2), component by component
        auto explicit_part = [&](int c) -> double {
            const long long ia = za + c * g.comp_a;
            double I = 0.0;
            for (int n = 0; n < q.nquad; ++n) I = fma(q.w[n], q.A[n][ia] + q.R[n][ia], I);
            return fma(-dt, R_old_next[ia], fma(dt, A_new[ia] - A_old[ia], U_m[zu + c * g.comp_g])) + I;
        };
        const double rho = explicit_part(0), mx = explicit_part(1), my = explicit_part(2), mz = explicit_part(3);
        const double cE = explicit_part(4);
        double cy[CST_MAX_REACT], y[CST_MAX_REACT];
#pragma unroll
        for (int s = 0; s < CST_MAX_REACT; ++s) { cy[s] = (s < r.ns) ? explicit_part(5 + s) : 0.0; y[s] = cy[s]; }
        const double ke = 0.5 * (mx * mx + my * my + mz * mz) / rho;
        double yE = cE;
        double lam[CST_MAX_REACT], R[CST_MAX_REACT], RE, dl;
        bool converged = false;
        for (int it = 0; it < r.max_iter && !converged; ++it) {
            react_rates(r, rho, ke, yE, lam, dl);
            react_rhs(r, lam, y, R, RE);
            // Newton matrix I - dt J:  species row k:  -dt lam_{k-1} d_{k-1} + (1 + dt lam_k) d_k + a_k d_E = res_k,
            // a_k = -dt dR_k/dy_E = -dt dl R_k (every rate has the same logarithmic derivative);  energy row:
            // sum_k (-dt q_k lam_k) d_k + (1 - dt dl R_E) d_E = res_E.   d_k = alpha_k + beta_k d_E.
            double al_prev = 0.0, be_prev = 0.0, sum_a = 0.0, sum_b = 0.0;
            double al[CST_MAX_REACT], be[CST_MAX_REACT];
#pragma unroll
            for (int s = 0; s < CST_MAX_REACT; ++s) {
                if (s < r.ns) {
                    const double res = -(y[s] - cy[s] - dt * R[s]);
                    const double sub = (s > 0) ? dt * lam[s > 0 ? s - 1 : 0] : 0.0;
                    const double rd = 1.0 / fma(dt, lam[s], 1.0);
                    al[s] = fma(sub, al_prev, res) * rd;
                    be[s] = fma(sub, be_prev, dt * dl * R[s]) * rd;
                    al_prev = al[s]; be_prev = be[s];
                    const double brow = -dt * r.q[s] * lam[s];
                    sum_a = fma(brow, al[s], sum_a);
                    sum_b = fma(brow, be[s], sum_b);
                } else { al[s] = 0.0; be[s] = 0.0; }
            }
            const double resE = -(yE - cE - dt * RE);
            const double dE = (resE - sum_a) / (fma(-dt * dl, RE, 1.0) + sum_b);
            yE += dE;
            double worst = fabs(dE) / fabs(yE);
            const double rrho = 1.0 / rho;
#pragma unroll
            for (int s = 0; s < CST_MAX_REACT; ++s) {
                if (s < r.ns) {
                    const double d = fma(be[s], dE, al[s]);
                    y[s] += d;
                    worst = fmax(worst, fabs(d) * rrho);
                }
            }
            converged = worst <= r.tol;
        }
        if (!converged) atomicAdd(n_fail, 1ull);
        react_rates(r, rho, ke, yE, lam, dl);
        react_rhs(r, lam, y, R, RE);
        const long long ub = zu;
        U_next[ub] = rho; U_next[ub + g.comp_g] = mx; U_next[ub + 2 * g.comp_g] = my; U_next[ub + 3 * g.comp_g] = mz;
        U_next[ub + 4 * g.comp_g] = yE;
#pragma unroll
        for (int c = 0; c < 4; ++c) R_new[za + c * g.comp_a] = 0.0;
        R_new[za + 4 * g.comp_a] = RE;
#pragma unroll
        for (int s = 0; s < CST_MAX_REACT; ++s)
            if (s < r.ns) { U_next[ub + (5 + s) * g.comp_g] = y[s]; R_new[za + (5 + s) * g.comp_a] = R[s]; }
    }
}

static ReactDev to_dev(const cst_ctx* ctx)
{
    ReactDev r;
    const cst_react_params& p = ctx->react;
    r.cv = p.cv; r.T0 = p.T0; r.nu = p.nu; r.tol = p.tol; r.max_iter = p.max_iter; r.ns = ctx->g.nspec;
    for (int k = 0; k < CST_MAX_REACT; ++k) { r.rate[k] = p.rate[k]; r.q[k] = p.q[k]; }
    return r;
}

static unsigned react_grid(const cst_ctx* ctx)
{
    const long long total = (long long)ctx->g.nbox * ctx->g.comp_a;
    long long nb = (total + 127) / 128;
    const long long cap = (long long)ctx->sm_count * 32;
    return (unsigned)(nb > cap ? cap : (nb < 1 ? 1 : nb));
}

int launch_react_R(cst_ctx* ctx, const double* U, double* R, cudaStream_t st)
{
    if (!ctx->has_react) return CST_EINVAL;
    k_react_R<<<react_grid(ctx), 128, 0, st>>>(ctx->g, to_dev(ctx), U, R);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

int launch_sdc_update_react(cst_ctx* ctx, double* U_next, const double* U_m, double dt_m, const double* A_new_m,
                            const double* A_old_m, const double* R_old_next, int nquad, const double* const* A_quad,
                            const double* const* R_quad, const double* w_quad, double* R_new, cudaStream_t st)
{
    if (!ctx->has_react) return CST_EINVAL;
    ReactQuad q{};
    q.nquad = nquad;
    for (int n = 0; n < nquad; ++n) { q.A[n] = A_quad[n]; q.R[n] = R_quad[n]; q.w[n] = w_quad[n]; }
    k_sdc_update_react<<<react_grid(ctx), 128, 0, st>>>(ctx->g, to_dev(ctx), U_next, U_m, dt_m, A_new_m, A_old_m, R_old_next,
                                                        q, R_new, reinterpret_cast<unsigned long long*>(ctx->d_scratch + 3));
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
