// advect.cu -- launcher of <A(U)> (S1-S4) and of the fused A + node update (S1-S5)
// (include/cst.h cst_advance_A, cst_advance_A_update).  Two kernels on the caller's stream:
//   k_advect_hydro   (advect_hydro.cu)   the five hydrodynamic components, + workspace rinv, Fm
//   k_advect_species (advect_species.cu) the nspec passively advected components
// Both tile every box into 16^3 tiles and sweep pencils with the PPM stencil in registers
// (tile.cuh, sweep.cuh); DESIGN.md section 6 has the design and its roofline.
#include "tile.cuh"

long long workspace_bytes(const Geom& g)
{
    return (ws_rinv_doubles(g) + ws_fm_doubles(g)) * (long long)sizeof(double);
}

int launch_advance_A(cst_ctx* ctx, const double* U, double* A, double* U_next, double dt_m,
                     const double* A_old_m, const QuadArgs& q, bool fused, cudaStream_t st)
{
    if (!ctx->ws || ctx->ws_bytes < workspace_bytes(ctx->g)) return CST_ENOWORKSPACE;
    UpdArgs up{};
    up.fused = fused;
    up.U_next = U_next;
    up.dt_m = dt_m;
    up.A_old = (A_old_m == A) ? nullptr : A_old_m;
    up.nquad = fused ? q.nquad : 0;
    for (int n = 0; n < up.nquad; ++n) { up.Aq[n] = (q.A[n] == A) ? nullptr : q.A[n]; up.w[n] = q.w[n]; }
    int rc = launch_advect_hydro(ctx, U, A, up, st);
    if (rc) return rc;
    return launch_advect_species(ctx, U, A, up, st);
}
