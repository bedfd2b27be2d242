// common.cuh -- geometry shared by the CUDA kernels of libcst (product code; shares nothing
// with oracle/).  Layout and index conventions: include/cst.h, DESIGN.md section 4.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/cst.h"

#define CST_NG 4

struct Geom {
    int nx, ny, nz;          // interior zones per box
    int ex, ey, ez;          // ghosted extents
    int nbx, nby, nbz, nbox;
    int gnbx, gnby, gnbz;    // global box lattice this context's boxes are a brick of (cst_set_sublattice; default = local)
    int obx, oby, obz;       // lattice coordinates of local box (0, 0, 0) in the global lattice
    int nspec, nvar;
    int bc_lo[3], bc_hi[3];
    double dx, dy, dz;
    double rdx, rdy, rdz;    // reciprocals
    double gamma, gm1, rgm1, gfac;   // gamma, gamma-1, 1/(gamma-1), (gamma+1)/(2 gamma)
    double grav[3];
    double small_dens, small_pres;
    long long plane_g;       // ex*ey
    long long comp_g;        // ex*ey*ez   (stride between components of U)
    long long box_g;         // nvar*comp_g
    long long comp_a;        // nx*ny*nz   (stride between components of A)
    long long box_a;         // nvar*comp_a
};

struct cst_ctx {
    cst_params p;
    Geom g;
    double* d_scratch;       // [0] = max signal rate bits, [1] = dt
    double* ws;              // caller-owned workspace (cst_set_workspace): [rinv][Fm], tile.cuh
    long long ws_bytes;
    long long launches;
    int sm_count;
    int timing;              // cst_set_timing: record events around the kernels of the advance calls
    cudaEvent_t ev[3];       // before hydro, between hydro and species, after species
    struct XPlan* xplan;     // cst_set_sublattice: ghost-exchange plan with the neighbouring ranks (exchange.cu)
    cst_react_params react;  // cst_set_reactions (react.cu)
    int has_react;
    int species_split;       // CTAs that share one tile in the species kernel (each a contiguous share of the species); 0 = default
    int species_variant;     // cst_set_variant / cst_tune_advance: 0 measured kernel, 1 / 2 variant kernels (species_tma.cuh)
    int order;               // cst_set_order: 2 (PPM path, default) or 4 (fourth.cu)
    int flatten;             // cst_set_flattening (flatten.cu): chi array behind rinv and Fm in the workspace
    double diff_kth, diff_cv;  // cst_set_diffusion (diffuse.cu); kth = 0: no diffusion term
};

struct UpdArgs;
struct QuadArgs {            // passed by value to the update kernels
    int nquad;
    const double* A[CST_MAX_QUAD];
    double w[CST_MAX_QUAD];
};

__host__ __device__ inline long long uidx(const Geom& g, int b, int c, int k, int j, int i)
{   // ghosted index; k, j, i in [0, e*)
    return (long long)b * g.box_g + (long long)c * g.comp_g + ((long long)k * g.ey + j) * g.ex + i;
}
__host__ __device__ inline long long aidx(const Geom& g, int b, int c, int k, int j, int i)
{   // interior index; k, j, i in [0, n*)
    return (long long)b * g.box_a + (long long)c * g.comp_a + ((long long)k * g.ny + j) * g.nx + i;
}

// launchers (one per source file)
int launch_fill_ghosts(cst_ctx*, double* U, cudaStream_t);
int launch_advance_A(cst_ctx*, const double* U, double* A, double* U_next, double dt_m,
                     const double* A_old_m, const QuadArgs& q, bool fused, cudaStream_t, double* cfl_scratch = nullptr);
int launch_advance_A_cfl(cst_ctx*, const double* U, double* A, double* U_next, double dt_m, const double* A_old_m,
                         const QuadArgs& q, bool fused, double cfl, double* dt_out_dev, cudaStream_t);
int launch_advect_hydro_cfl(cst_ctx*, const double* U, double* A, const UpdArgs& up, double* cfl_scratch, cudaStream_t);
bool hydro_cfl_eligible(const cst_ctx*, const double* U);
int launch_cfl_reset(cst_ctx*, cudaStream_t);
int launch_cfl_final(cst_ctx*, double cfl, double* dt_out_dev, cudaStream_t);
int launch_advect_hydro(cst_ctx*, const double* U, double* A, const UpdArgs& up, cudaStream_t);
int launch_advect_species(cst_ctx*, const double* U, double* A, const UpdArgs& up, cudaStream_t);
long long workspace_bytes(const cst_ctx* ctx);
int launch_sdc_update(cst_ctx*, double* U_next, const double* U_m, double dt_m,
                      const double* A_new_m, const double* A_old_m, const QuadArgs& q, cudaStream_t);
int launch_cfl(cst_ctx*, const double* U, double cfl, double* dt_out_dev, cudaStream_t);
int launch_validate(cst_ctx*, const double* U, cudaStream_t);   // count left in d_scratch[2]
int launch_advance_A4(cst_ctx*, const double* U, double* A, cudaStream_t);   // fourth.cu: fourth-order <A(U)>
long long fourth_workspace_doubles(const Geom& g);
int launch_advance_ctu(cst_ctx*, const double* U, double dt, double* A, double* ws, cudaStream_t);   // ctu.cu
long long ctu_workspace_doubles(const Geom& g);
int launch_flatten(cst_ctx*, const double* U, cudaStream_t);   // flatten.cu: chi of every zone -1 .. n -> workspace
// diffuse.cu: A[rho E] += k_th lap T (and U_next[rho E] += ca * that when U_next != nullptr)
int launch_diffuse_add(cst_ctx*, const double* U, double* A, double* U_next, double ca, cudaStream_t);
// react.cu: R != 0
int launch_react_R(cst_ctx*, const double* U, double* R, cudaStream_t);
int launch_sdc_update_react(cst_ctx*, double* U_next, const double* U_m, double dt_m, const double* A_new_m,
                            const double* A_old_m, const double* R_old_next, int nquad, const double* const* A_quad,
                            const double* const* R_quad, const double* w_quad, double* R_new, cudaStream_t);
// exchange.cu: box lattice sharded over ranks
int xplan_create(cst_ctx*, const int global_nb[3], const int part[3], int rank);
void xplan_destroy(cst_ctx*);
int xplan_info(const cst_ctx*, int* npeers, int* peers, long long* send_off, long long* send_len,
               long long* recv_off, long long* recv_len, int cap);
int launch_exchange_pack(cst_ctx*, const double* U, double* sendbuf, cudaStream_t);
int launch_exchange_unpack(cst_ctx*, double* U, const double* recvbuf, cudaStream_t);
int launch_exchange_push(cst_ctx*, const double* U, double* const* peer_U, int npeers, cudaStream_t);
int launch_debug_rcp_sqrt(const double* x, double* r, double* s, long long n, cudaStream_t);
long long debug_tile_count(const Geom& g);
int launch_debug_tile_map(cst_ctx*, int* out, cudaStream_t);
