/*
 * cst.h -- C ABI of the B200-native hot path of Castro's SDC reactive-flow method
 *          (Zingale et al., arXiv:1910.12578; /root/reference/PAPER.md = "P").
 *
 * The library evaluates, on AMReX-style boxes of fp64 conserved state resident in GPU memory,
 *   S0  ghost-zone fill                        ("grids"/"boxes"; Q16)
 *   S1-S4  the advective term <A(U)> of Eq. (1) ("the divergence of the hydrodynamic
 *          fluxes along with hydrodynamic sources"; evaluated at a node time)
 *   S5  the SDC node update, Eq. (2), R = 0
 *   S6  the CFL time step                       (BASELINE.json north_star; Q20)
 * Beyond that path (each documented at its declaration below): the box lattice sharded over ranks
 * (cst_set_sublattice, cst_exchange_*), reactions R != 0 (cst_sdc_update_react), explicit diffusion (cst_set_diffusion),
 * shock flattening (cst_set_flattening), the fourth-order operator (cst_set_order), the unsplit CTU PPM operator
 * (cst_advance_ctu), kernel variants chosen by measurement (cst_tune_advance), S1-S6 in one call (cst_advance_A_update_cfl).
 * Every step runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * LAYOUT.  All arrays are fp64, C-contiguous, in DEVICE memory:
 *   U[b][c][k][j][i]  ghosted state, extents nbox x NVAR x (nz+2ng) x (ny+2ng) x (nx+2ng), i fastest
 *   A[b][c][k][j][i]  interior-only arrays, extents nbox x NVAR x nz x ny x nx
 *   c = 0 rho, 1 rho*u, 2 rho*v, 3 rho*w, 4 rho*E, 5+s rho*X_s;  NVAR = 5 + nspec
 *   b = bi + nbx*(bj + nby*bk); box (bi,bj,bk) covers global zones [bi*nx,(bi+1)*nx) x ...
 *
 * OWNERSHIP.  The caller owns every state/flux buffer, the workspace and the stream.  The context
 * owns only a few KB of device scratch (reduction cells).  No call allocates or frees device memory
 * after cst_create.
 * `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 * One context (and its workspace) serves ONE stream at a time: the reduction cells of cst_cfl_dt / cst_validate and
 * the workspace are shared by all calls on the context; use one context per concurrent stream.
 *
 * ERRORS.  Every call returns 0 (CST_OK) or a negative code; nothing throws, aborts or prints.
 * Launches are asynchronous: a device fault surfaces as CST_ECUDA from the next synchronising
 * call.  NaN / negative-pressure inputs are not detected on the hot path.
 */
#ifndef CST_H
#define CST_H

#ifdef __cplusplus
extern "C" {
#endif

enum { CST_OK = 0, CST_EINVAL = -1, CST_ECUDA = -2, CST_ENOMEM = -3, CST_ENOWORKSPACE = -4 };
enum { CST_BC_PERIODIC = 0, CST_BC_OUTFLOW = 1, CST_BC_REFLECT = 2 };
#define CST_MAX_QUAD 4      /* at most 4 quadrature nodes in one update (3 used by Simpson)     */
#define CST_MAX_NSPEC 59    /* NVAR <= 64                                                       */

typedef struct {
    int    nx, ny, nz;         /* interior zones per box (all boxes equal); each >= ng           */
    int    ng;                 /* ghost width; must be 4                                         */
    int    nbx, nby, nbz;      /* box lattice; nbox = nbx*nby*nbz                                */
    int    nspec;              /* passively advected species; NVAR = 5 + nspec                   */
    double dx, dy, dz;         /* zone widths (> 0)                                              */
    double gamma;              /* gamma-law EOS (> 1)                                            */
    double grav[3];            /* constant acceleration ("hydrodynamic source"); 0 = none */
    int    bc_lo[3], bc_hi[3]; /* CST_BC_*; periodic must be set on both sides of a direction    */
    double small_dens, small_pres; /* floors on interface rho, p and zone-centre p (Q11)         */
} cst_params;

typedef struct cst_ctx cst_ctx;    /* opaque */

/* Validates params (CST_EINVAL: NULL, ng != 4, n_d < ng, nspec out of range, more than 2^24 boxes, non-positive
 * widths, gamma <= 1, bad or one-sided-periodic BC) and allocates the context's scratch.
 * Range of the state: the kernels form products such as gamma*p*rho and use reciprocal / square-root sequences
 * without the special-case branches of the library routines, so rho and p (floors included) must stay within
 * about [1e-140, 1e140]; outside it results are unspecified (the default floors 1e-200 never bind inside it). */
int cst_create(const cst_params* params, cst_ctx** out);
int cst_destroy(cst_ctx* ctx);

/* Workspace of cst_advance_A / cst_advance_A_update / cst_step_host.  <A(U)> is evaluated by a hydro
 * kernel and a species kernel (F(rho X_s) = F(rho) * upwind X_s); the face mass fluxes F(rho) and
 * 1/rho travel between them through a caller-owned DEVICE buffer of cst_workspace_bytes() bytes
 * (about 34 bytes per ghosted zone; 16-byte aligned; contents are scratch, valid only within one
 * call).  cst_set_workspace stores the pointer (CST_EINVAL if NULL or too small); the advance calls
 * return CST_ENOWORKSPACE until it has been set.  One workspace serves one stream at a time. */
long long cst_workspace_bytes(const cst_ctx* ctx);
int cst_set_workspace(cst_ctx* ctx, void* workspace_dev, long long bytes);

/* S0.  Fills the whole 4-deep ghost shell of every box of U in place (faces,
 * edges, corners) from the interior of the box lattice: neighbour boxes inside the domain,
 * periodic wrap, outflow = copy of the nearest interior zone, reflecting = mirror image with the
 * wall-normal momentum negated.  Interior zones are not touched. */
int cst_fill_ghosts(cst_ctx* ctx, double* U, void* stream);

/* Box lattice sharded over ranks ("MPI distribute the AMR grids across nodes").
 * The global lattice of global_nb[0] x [1] x [2] boxes is cut into part[0] x part[1] x part[2] equal bricks, brick
 * (pi, pj, pk) owned by rank pi + part[0]*(pj + part[1]*pk); global_nb[d] must be a multiple of part[d].
 * cst_set_sublattice declares that the context (created with nbx, nby, nbz = the BRICK's lattice; bc_lo / bc_hi = the
 * boundaries of the GLOBAL domain) holds the brick of `rank`.  From then on cst_fill_ghosts uses the global zone map
 * and fills every ghost zone whose source box is local; the others arrive from the neighbouring ranks:
 *   cst_exchange_pack   writes, for every peer, one message (the source zones of all the peer's ghost regions that
 *                       read this brick, in the peer's zone order, reflecting-wall signs applied) into sendbuf;
 *   [the caller moves sendbuf[send_off[p] .. +send_len[p]) to peer p's recvbuf[recv_off .. +recv_len): NCCL / MPI]
 *   cst_exchange_unpack copies the received messages into the ghost regions of U.
 * cst_exchange_info: number of peers (<= 26) and, per peer (ascending rank), offsets and lengths in DOUBLES of its
 * message inside the send / receive buffers (DEVICE buffers owned by the caller, at least sum(len) doubles).
 * Every other call works on the local boxes unchanged; the time step needs a MIN over ranks of cst_cfl_dt.
 * CST_EINVAL: lattice not divisible, brick != the context's lattice, rank out of range, no plan set.
 *
 * cst_exchange_plan is the plan itself as a pure HOST function (no GPU, no context): the segments of `rank`
 * (recv = 1: its ghost regions with a remote source; recv = 0: what it sends), grouped by peer in ascending order.
 * `global` describes the GLOBAL lattice.  Returns the number of segments (call with segs = NULL to size the array). */
typedef struct {
    int peer;              /* rank on the other side                                                        */
    int box;               /* LOCAL box index on this side: source box (send) or destination box (recv)      */
    int lo[3];             /* ghosted (i, j, k) index of the first zone on this side                         */
    int step[3];           /* send: +1 neighbour / periodic, 0 outflow, -1 reflecting mirror; recv: +1        */
    int ext[3];            /* zones per direction (extents of the destination region)                        */
    int flip[3];           /* send: 1 = the momentum component along d changes sign (reflecting wall)        */
    long long offset;      /* doubles from the start of this peer's message; segment data is [c][k][j][i]    */
    int rbox;              /* the OTHER side's local box index (recv: the source box there; send: the box whose */
    int rlo[3];            /* ghost region is filled) and the first zone of the segment there                  */
} cst_xseg;
#define CST_MAX_PEERS 26
long long cst_exchange_plan(const cst_params* global, const int part[3], int rank, int recv,
                            cst_xseg* segs, long long cap);
int cst_set_sublattice(cst_ctx* ctx, const int global_nb[3], const int part[3], int rank);
int cst_exchange_info(const cst_ctx* ctx, int* npeers, int* peers, long long* send_off, long long* send_len,
                      long long* recv_off, long long* recv_len, int cap);
int cst_exchange_pack(cst_ctx* ctx, const double* U, double* sendbuf, void* stream);
int cst_exchange_unpack(cst_ctx* ctx, double* U, const double* recvbuf, void* stream);

/* The same exchange without staging buffers or a communication library: cst_exchange_push writes every zone that a
 * peer's ghost shell reads from this brick STRAIGHT into the peer's state array through a peer-mapped device pointer
 * (stores over NVLink / NVSwitch from one kernel; same zone map and signs as pack + unpack).  peer_U: HOST array of
 * npeers DEVICE pointers, in the order of cst_exchange_info, each the base of that peer's U (its whole brick).  The
 * caller separates pushes from the peers' reads of their shells (a barrier across the ranks before the push and one
 * after it, e.g. torch.distributed.barrier).
 * Pointers to another process's memory come from CUDA IPC: cst_ipc_export gives a 64-byte handle of the allocation
 * that contains dev_ptr plus the offset of dev_ptr inside it; cst_ipc_import opens such a handle in another process
 * and returns the mapped pointer (+ offset); cst_ipc_close unmaps it (pass the pointer minus the offset).
 * CST_ECUDA if the allocation cannot be shared (peer access unavailable, or an allocator that does not use cudaMalloc). */
int cst_exchange_push(cst_ctx* ctx, const double* U, double* const* peer_U, int npeers, void* stream);
int cst_ipc_export(const void* dev_ptr, unsigned char handle[64], long long* offset_bytes);
int cst_ipc_import(const unsigned char handle[64], long long offset_bytes, void** dev_ptr);
int cst_ipc_close(void* mapped_base);

/* S1-S4.  A <- <A(U)>: conserved->primitive with the gamma-law EOS, PPM
 * reconstruction (Colella & Woodward 1984 limiter, P:L52 ref [15]) of the primitives in x, y, z,
 * an HLLC Riemann solve at every face, flux divergence plus the constant-gravity source.
 * Reads U on the interior and the 3-deep face ghosts (which must be filled); writes all of A. */
int cst_advance_A(cst_ctx* ctx, const double* U, double* A, void* stream);

/* S5 (Eq. (2) with R = 0).  On interior zones of every box
 *   U_next = U_m + dt_m*(A_new_m - A_old_m) + sum_{q<nquad} w_quad[q]*A_quad[q]
 * w_quad (HOST array, weights already multiplied by dt) and A_quad (HOST array of nquad DEVICE
 * pointers, 0 <= nquad <= CST_MAX_QUAD) are copied by value at the call.  Ghosts of U_next are
 * left untouched (stale until cst_fill_ghosts).  U_next may alias U_m. */
int cst_sdc_update(cst_ctx* ctx, double* U_next, const double* U_m, double dt_m,
                   const double* A_new_m, const double* A_old_m,
                   int nquad, const double* const* A_quad, const double* w_quad, void* stream);

/* Kernel variants of the species half of <A(U)> on boxes made of full 16^3 tiles (csrc/species_tma.cuh); every variant
 * performs the same operations in the same order, so results are bit-identical.
 *   0  (default) conversion phase + three sweeps + write-out phase per species: the kernel that has been profiled;
 *   1  X = rho X / rho formed inside the x sweep (no conversion phase);
 *   2  as 1, and each component is written out from its own z sweep (no write-out phase);
 *   3  as 2, with the L2 prefetches (next species' tile, operands of the update) issued one sweep instead of one to
 *      two sweeps ahead of their use (less of the prefetched data is evicted again before it is read).
 * cst_set_variant selects one (CST_EINVAL outside 0..3); cst_get_variant returns the current one.
 * cst_set_species_split: how many consecutive CTAs share one tile, each taking a contiguous share of the species
 * (0 = the default, 3; at most 8; never more than nspec).  Does not change results either.
 * cst_tune_advance runs cst_advance_A_update (same arguments, same rules) `repeats` + 1 times with every variant on
 * the caller's buffers, times each with CUDA events on `stream` (minimum over the repeats; the first run of a
 * configuration is a warm-up), then tries 2 and 4 CTAs per tile with the winner, keeps the fastest configuration for all
 * later calls and leaves A_new_m / U_next valid; ms_out (HOST, 6 floats, may be NULL) receives the times in
 * milliseconds: variants 0, 1, 2, 3 at the default split, then the winner at split 2 and 4.  Synchronises the stream.
 * Measurement, not arithmetic: which configuration wins depends on the device and the box shape. */
int cst_set_variant(cst_ctx* ctx, int species_variant);
int cst_get_variant(const cst_ctx* ctx);
int cst_set_species_split(cst_ctx* ctx, int split);
int cst_get_species_split(const cst_ctx* ctx);
int cst_tune_advance(cst_ctx* ctx, const double* U_m, double* A_new_m, double* U_next, double dt_m,
                     const double* A_old_m, int nquad, const double* const* A_quad, const double* w_quad,
                     int repeats, float* ms_out, void* stream);

/* The unsplit CTU PPM operator ("the main unsplit PPM hydrodynamics scheme [15, 16]", the hydro solver of the
 * paper's Strang path; readings C1-C9): PPM parabolas with characteristic tracing over
 * dt / 2 (Colella & Woodward 1984), corner-transport-upwind transverse flux corrections (Miller & Colella 2002: one third
 * of dt for the first, one half for the final states; 12 HLLC solves per zone), divergence + gravity source:
 *   A <- A_ctu(U, dt) = -div F^{n+1/2} + S,      U^{n+1} = U^n + dt A   (e.g. cst_sdc_update with A_new = A_old, w = dt).
 * Unlike <A(U)> of the SDC path it depends on dt and is stable for dt <= min_d Delta_d / max(|u_d| + c).  Reads the
 * WHOLE 4-deep ghost shell.  workspace_dev: DEVICE scratch of cst_ctu_workspace_bytes() bytes (18 arrays of the size of
 * U), 16-byte aligned, owned by the caller (CST_ENOWORKSPACE if too small).  CST_EINVAL: NULL, dt < 0. */
long long cst_ctu_workspace_bytes(const cst_ctx* ctx);
int cst_advance_ctu(cst_ctx* ctx, const double* U, double dt, double* A, void* workspace_dev, long long bytes, void* stream);

/* Spatial order of <A(U)> ("a fourth-order method in space and time (using a Simpsons rule for the integral and
 * the spatial reconstruction of [12])"; readings G1-G9).  order = 2 (default, the graded
 * path): PPM + CW84 limiter as described at cst_advance_A.  order = 4: U and A are CELL AVERAGES and every later
 * cst_advance_A / cst_advance_A_update / cst_step_host evaluates the fourth-order finite-volume operator -- cell-centre
 * and cell-average primitives through undivided Laplacians / 24, (7/12, -1/12) face averages with the
 * extremum-preserving limiter of [12] (McCorquodale & Colella 2011; without its third-difference test, whose stencil
 * needs a fifth ghost zone), face-centred states, two HLLC solves per face and transverse Laplacians of the fluxes.
 * It reads the WHOLE 4-deep ghost shell; together with the 3-node Simpson weights of cst_sdc_update it is the paper's
 * fourth-order scheme.  The workspace is larger (cst_workspace_bytes(): about 5 NVAR doubles per zone): set the order
 * BEFORE sizing / setting the workspace.  Flattening does not apply to order 4.  CST_EINVAL: order not 2 or 4. */
int cst_set_order(cst_ctx* ctx, int order);

/* Shock flattening (Colella & Woodward 1984, appendix; P:L52 ref [15]; DESIGN.md readings
 * F1-F4), an option that is OFF by default (the graded path, Q4).  With on != 0 every later
 * cst_advance_A / cst_advance_A_update / cst_step_host first computes the flattening coefficient chi of every zone
 * (min over the three directions of CW84's pressure-jump / compression test) and blends every PPM parabola with its
 * zone average, q+- <- chi q+- + (1 - chi) q.  It reads the WHOLE 4-deep ghost shell (edges and corners included) and
 * runs on the general (any box shape) kernels.  Switching it on enlarges cst_workspace_bytes() by one double per
 * ghosted zone: call it BEFORE sizing / setting the workspace (else the advance calls return CST_ENOWORKSPACE). */
int cst_set_flattening(cst_ctx* ctx, int on);

/* Explicit thermal diffusion as an extra term of A ("thermal diffusion", "explicit diffusion"; SURVEY 8(f)
 * NEXT-4; readings D1-D3).  With kth > 0 every later cst_advance_A / cst_advance_A_update / cst_step_host adds
 *   k_th lap T,  T = p / ((gamma - 1) rho cv),  p the floored gamma-law pressure of S1,
 * (second-order centred differences on the +-1 star, summed ((x + y) + z)) to the rho E component of A, the fused
 * node update included.  Constant conductivity and c_v: the paper's conductivity tables are not available.
 * kth = 0 switches the term off (default).  CST_EINVAL: kth < 0 or cv <= 0. */
int cst_set_diffusion(cst_ctx* ctx, double kth, double cv);

/* Reactions: Eq. (1)-(2) with R != 0 ("implicit reaction updates").
 * The paper's 13-isotope network needs rate tables that are not available; R is a synthetic stiff chain with the same
 * structure (readings R1-R4): species k -> k+1 at the rate lambda_k(T) = rate[k] (T/T0)^nu (the last species
 * is stable), T = e / cv with e = E/rho - |v|^2/2, R(rho X_k) = rho (lambda_{k-1} X_{k-1} - lambda_k X_k),
 * R(rho E) = rho sum_k q[k] lambda_k X_k, R(rho) = R(rho v) = 0.  All nspec species of the context take part
 * (1 <= nspec <= CST_MAX_REACT, else CST_EINVAL).
 *   cst_react_R           R <- R(U) on interior zones; R has the layout of A (components 0..3 are written as zero).
 *   cst_sdc_update_react  the node update of Eq. (2), implicit in R: on every interior zone
 *                           c = U_m + dt_m (A_new_m - A_old_m) - dt_m R_old_next + sum_q w_quad[q] (A_quad[q] + R_quad[q])
 *                           U_next = c + dt_m R(U_next)
 *                         by Newton's method per zone (first iterate c; stops when the last correction is <= tol
 *                         relative to rho (species) / |rho E| (energy), at most max_iter iterations), and
 *                         R_new_out <- R(U_next).  R_old_next = R^{m+1,(k)}.  A_quad, R_quad: HOST arrays of nquad
 *                         DEVICE pointers (0 <= nquad <= CST_MAX_QUAD).  U_next may alias U_m; R_new_out may alias
 *                         R_old_next.  Ghosts of U_next are left untouched.
 *   cst_react_failures    *n_host (HOST) <- zones that did not converge since the last call; synchronises the stream. */
#define CST_MAX_REACT 15
typedef struct {
    double cv, T0, nu;             /* T = e / cv; rates scale as (T / T0)^nu                                   */
    double rate[CST_MAX_REACT];    /* rate[k] of species k -> k+1 at T = T0 (entry nspec-1 is ignored)         */
    double q[CST_MAX_REACT];       /* specific energy released by the reaction of species k                    */
    int    max_iter;               /* Newton iterations per zone (>= 1)                                        */
    double tol;                    /* relative size of the last correction at which the iteration stops (> 0)  */
} cst_react_params;
int cst_set_reactions(cst_ctx* ctx, const cst_react_params* react);
int cst_react_R(cst_ctx* ctx, const double* U, double* R, void* stream);
int cst_sdc_update_react(cst_ctx* ctx, double* U_next, const double* U_m, double dt_m,
                         const double* A_new_m, const double* A_old_m, const double* R_old_next,
                         int nquad, const double* const* A_quad, const double* const* R_quad, const double* w_quad,
                         double* R_new_out, void* stream);
int cst_react_failures(cst_ctx* ctx, long long* n_host, void* stream);

/* Fused S1-S5: A_new_m <- <A(U_m)> and the node update above with that A_new_m, in one pass over
 * U_m.  A_old_m or any A_quad[q] may be the A_new_m buffer itself (then they mean the value just
 * computed, as in the first SDC iteration where every node carries A(U^n)).  Neither output may be an
 * input: U_next == U_m, U_next == A_old_m / A_quad[q], U_next == A_new_m or U_m == A_new_m give CST_EINVAL
 * (partially overlapping buffers are not detected). */
int cst_advance_A_update(cst_ctx* ctx, const double* U_m, double* A_new_m, double* U_next,
                         double dt_m, const double* A_old_m,
                         int nquad, const double* const* A_quad, const double* w_quad, void* stream);

/* Fused S1-S6: cst_advance_A_update (same arguments, same rules) plus the CFL step of the SAME state U_m, left in
 * *dt_out_dev (DEVICE pointer) as by cst_cfl_dt_device(ctx, U_m, cfl, ...).  On lattices made of full 16^3 tiles the max
 * signal rate is gathered inside the z sweep of the hydro kernel, which has every zone's primitives at hand, and the
 * separate pass over the state is saved; otherwise the two calls simply run back to back.  Does not synchronise. */
int cst_advance_A_update_cfl(cst_ctx* ctx, const double* U_m, double* A_new_m, double* U_next,
                             double dt_m, const double* A_old_m,
                             int nquad, const double* const* A_quad, const double* w_quad,
                             double cfl, double* dt_out_dev, void* stream);

/* S6 (BASELINE.json north_star; sum form, Q20).
 *   dt = cfl / max over interior zones of [(|u|+c)/dx + (|v|+c)/dy + (|w|+c)/dz], c = sqrt(gamma p/rho)
 * cst_cfl_dt_device leaves dt in *dt_out_dev (DEVICE pointer) without synchronising;
 * cst_cfl_dt writes *dt_out_host (HOST pointer) and synchronises the stream. */
int cst_cfl_dt_device(cst_ctx* ctx, const double* U, double cfl, double* dt_out_dev, void* stream);
int cst_cfl_dt(cst_ctx* ctx, const double* U, double cfl, double* dt_out_host, void* stream);

/* Optional input check (not on the hot path, which does not detect bad states): *n_bad_host (HOST pointer)
 * receives the number of interior zones with a non-finite component, rho <= 0 or gamma-law pressure <= 0.
 * Synchronises the stream. */
int cst_validate(cst_ctx* ctx, const double* U, long long* n_bad_host, void* stream);

/* Host-buffer convenience used for the end-to-end measurement: copies the interior+ghost array
 * U_host (HOST, layout of U) to the device buffers owned by the caller (U_dev, U_next_dev,
 * A_dev), runs fill_ghosts + advance_A_update (forward-Euler node update: A_old = A_quad = A_new)
 * and copies A and U_next back to A_host / U_next_host.  As with every node update only interior zones of U_next are
 * written: the ghost zones of U_next_host are whatever U_next_dev held before the call.  Synchronises the stream. */
int cst_step_host(cst_ctx* ctx, const double* U_host, double* A_host, double* U_next_host,
                  double* U_dev, double* U_next_dev, double* A_dev,
                  double dt_m, void* stream);   /* needs the workspace, see cst_set_workspace */

/* Measurement aid (bench.py roofline): with timing on, cst_advance_A / cst_advance_A_update record CUDA
 * events on the caller's stream around their two kernels (hydro components, species components);
 * cst_last_advance_ms waits for the last recorded call and returns the two durations in
 * milliseconds (CST_EINVAL if timing was never switched on).  Off by default. */
int cst_set_timing(cst_ctx* ctx, int on);
int cst_last_advance_ms(cst_ctx* ctx, double* ms_hydro, double* ms_species);

/* Test aids (tests/ only; not on the hot path).
 * cst_debug_rcp_sqrt: rcp_dev[i], sqrt_dev[i] <- the kernels' own reciprocal / square-root sequences (MUFU seed +
 *   Newton steps, csrc/hydro.cuh) of x_dev[i], i < n (DEVICE arrays), for an accuracy test in ulps.
 * cst_debug_tile_map: map_dev (DEVICE, 8 ints per tile, cst_debug_tile_count() tiles) receives, for every CTA
 *   index of the advance kernels' grid, (box, i0, j0, k0, tx, ty, tz, tile id) of the 16^3-zone tile it works on:
 *   the map must be a bijection onto the tiles of all boxes. */
int cst_debug_rcp_sqrt(const double* x_dev, double* rcp_dev, double* sqrt_dev, long long n, void* stream);
long long cst_debug_tile_count(const cst_ctx* ctx);
int cst_debug_tile_map(cst_ctx* ctx, int* map_dev, void* stream);

/* Number of kernel launches issued through this context since creation (for bench accounting). */
long long cst_launch_count(const cst_ctx* ctx);

const char* cst_strerror(int code);   /* static string; for CST_ECUDA the last CUDA error text  */
const char* cst_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CST_H */
