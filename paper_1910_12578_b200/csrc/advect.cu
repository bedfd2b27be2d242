// advect.cu -- launcher of <A(U)> (S1-S4) and of the fused A + node update (S1-S5)
// (include/cst.h cst_advance_A, cst_advance_A_update).  Two kernels on the caller's stream:
//   k_advect_hydro   (advect_hydro.cu)   the five hydrodynamic components, + workspace rinv, Fm
//   k_advect_species (advect_species.cu) the nspec passively advected components
// Both tile every box into 16^3 tiles and sweep pencils with the PPM stencil in registers
// (tile.cuh, sweep.cuh); DESIGN.md section 6 has the design and its roofline.
#include "tile.cuh"

long long workspace_bytes(const cst_ctx* ctx)
{   // [rinv][Fm] and, with flattening switched on, [chi] (one double per ghosted zone); order 4: fourth.cu's arrays
    const Geom& g = ctx->g;
    if (ctx->order == 4) return fourth_workspace_doubles(g) * (long long)sizeof(double);
    return (ws_rinv_doubles(g) + ws_fm_doubles(g) + (ctx->flatten ? ws_rinv_doubles(g) : 0)) * (long long)sizeof(double);
}

// Eq. (2) with R = 0 -> coefficient list (tile.cuh UpdArgs).  Returns false when more than
// UPD_MAX_EXT distinct external arrays are involved.
static bool make_upd(UpdArgs& up, const double* U, double* A, double* U_next, double dt_m,
                     const double* A_old_m, const QuadArgs& q)
{
    up.nr = 0; up.U_m = U; up.U_next = U_next; up.ca = 0.0; up.A_base = A;
    for (int r = 0; r < UPD_MAX_EXT; ++r) { up.P[r] = nullptr; up.c[r] = 0.0; }
    auto add = [&](const double* ptr, double coef) -> bool {
        if (ptr == A) { up.ca += coef; return true; }
        for (int r = 0; r < up.nr; ++r) if (up.P[r] == ptr) { up.c[r] += coef; return true; }
        if (up.nr == UPD_MAX_EXT) return false;
        up.P[up.nr] = ptr; up.c[up.nr] = coef; up.nr++;
        return true;
    };
    bool ok = add(A, dt_m) && add(A_old_m, -dt_m);
    for (int n = 0; ok && n < q.nquad; ++n) ok = add(q.A[n], q.w[n]);
    return ok;
}

int launch_advance_A(cst_ctx* ctx, const double* U, double* A, double* U_next, double dt_m,
                     const double* A_old_m, const QuadArgs& q, bool fused, cudaStream_t st, double* cfl_scratch)
{
    if (!ctx->ws || ctx->ws_bytes < workspace_bytes(ctx)) return CST_ENOWORKSPACE;
    UpdArgs up{};
    up.nr = -1; up.U_m = U; up.A_base = A;
    bool split = false;
    if (fused && !make_upd(up, U, A, U_next, dt_m, A_old_m, q)) { up.nr = -1; split = true; }
    int rc = CST_OK;
    if (ctx->order == 4) {             // fourth-order <A(U)> (fourth.cu), then the optional extra term and the plain node update
        rc = launch_advance_A4(ctx, U, A, st);
        if (!rc && ctx->diff_kth != 0.0) rc = launch_diffuse_add(ctx, U, A, nullptr, 0.0, st);
        if (rc || !fused) return rc;
        return launch_sdc_update(ctx, U_next, U, dt_m, A, A_old_m, q, st);
    }
    if (ctx->flatten && (rc = launch_flatten(ctx, U, st)) != CST_OK) return rc;
    if (ctx->timing) cudaEventRecord(ctx->ev[0], st);
    rc = cfl_scratch ? launch_advect_hydro_cfl(ctx, U, A, up, cfl_scratch, st) : launch_advect_hydro(ctx, U, A, up, st);
    if (rc) return rc;
    if (ctx->timing) cudaEventRecord(ctx->ev[1], st);
    rc = launch_advect_species(ctx, U, A, up, st);
    if (ctx->timing) cudaEventRecord(ctx->ev[2], st);
    if (!rc && ctx->diff_kth != 0.0)     // optional extra term of A (cst_set_diffusion); the fused update is completed too
        rc = launch_diffuse_add(ctx, U, A, (up.nr >= 0) ? U_next : nullptr, up.ca, st);
    if (rc || !split) return rc;
    // too many distinct arrays for the fused epilogue: A first, then the plain update kernel
    return launch_sdc_update(ctx, U_next, U, dt_m, A, A_old_m, q, st);
}

// S1-S6 in one call: the advance above and the CFL step of the SAME state.  On lattices of full tiles (second-order
// path) the max signal rate is gathered inside the hydro kernel's z sweep, which has every zone's primitives at hand --
// the separate pass over the five hydro components (k_cfl_max) is then not needed; otherwise it runs after the advance.
int launch_advance_A_cfl(cst_ctx* ctx, const double* U, double* A, double* U_next, double dt_m, const double* A_old_m,
                         const QuadArgs& q, bool fused, double cfl, double* dt_out_dev, cudaStream_t st)
{
    if (ctx->order == 2 && hydro_cfl_eligible(ctx, U)) {
        int rc = launch_cfl_reset(ctx, st);
        if (!rc) rc = launch_advance_A(ctx, U, A, U_next, dt_m, A_old_m, q, fused, st, ctx->d_scratch);
        if (!rc) rc = launch_cfl_final(ctx, cfl, dt_out_dev, st);
        return rc;
    }
    int rc = launch_advance_A(ctx, U, A, U_next, dt_m, A_old_m, q, fused, st);
    if (!rc) rc = launch_cfl(ctx, U, cfl, dt_out_dev, st);
    return rc;
}
