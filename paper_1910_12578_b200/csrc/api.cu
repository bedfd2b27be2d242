// api.cu -- the C ABI of libcst (include/cst.h): validation, context, argument marshalling.
// No arithmetic of the method lives here; every step runs in the kernels of this directory.
#include <new>
#include <string.h>
#include "common.cuh"

static thread_local char g_cuda_msg[256] = "no CUDA error recorded";

static int cuda_fail(cudaError_t e)
{
    strncpy(g_cuda_msg, cudaGetErrorString(e), sizeof(g_cuda_msg) - 1);
    g_cuda_msg[sizeof(g_cuda_msg) - 1] = 0;
    return CST_ECUDA;
}
static int check_launch(int rc)
{
    if (rc == CST_ECUDA) return cuda_fail(cudaGetLastError());
    return rc;
}

static int validate(const cst_params* p)
{
    if (!p) return CST_EINVAL;
    if (p->ng != CST_NG) return CST_EINVAL;
    if (p->nx < p->ng || p->ny < p->ng || p->nz < p->ng) return CST_EINVAL;
    if (p->nbx < 1 || p->nby < 1 || p->nbz < 1) return CST_EINVAL;
    if ((long long)p->nbx * p->nby * p->nbz > (1 << 24)) return CST_EINVAL;
    if (p->nspec < 0 || p->nspec > CST_MAX_NSPEC) return CST_EINVAL;
    if (!(p->dx > 0) || !(p->dy > 0) || !(p->dz > 0) || !(p->gamma > 1)) return CST_EINVAL;
    for (int d = 0; d < 3; ++d) {
        if (p->bc_lo[d] < 0 || p->bc_lo[d] > 2 || p->bc_hi[d] < 0 || p->bc_hi[d] > 2) return CST_EINVAL;
        if ((p->bc_lo[d] == CST_BC_PERIODIC) != (p->bc_hi[d] == CST_BC_PERIODIC)) return CST_EINVAL;
    }
    return CST_OK;
}

extern "C" int cst_create(const cst_params* p, cst_ctx** out)
{
    if (!out) return CST_EINVAL;
    *out = nullptr;
    int rc = validate(p);
    if (rc) return rc;
    cst_ctx* c = new (std::nothrow) cst_ctx();
    if (!c) return CST_ENOMEM;
    c->p = *p;
    Geom& g = c->g;
    g.nx = p->nx; g.ny = p->ny; g.nz = p->nz;
    g.ex = p->nx + 2 * CST_NG; g.ey = p->ny + 2 * CST_NG; g.ez = p->nz + 2 * CST_NG;
    g.nbx = p->nbx; g.nby = p->nby; g.nbz = p->nbz; g.nbox = p->nbx * p->nby * p->nbz;
    g.gnbx = p->nbx; g.gnby = p->nby; g.gnbz = p->nbz; g.obx = g.oby = g.obz = 0;   // the whole lattice is local
    g.nspec = p->nspec; g.nvar = 5 + p->nspec;
    for (int d = 0; d < 3; ++d) { g.bc_lo[d] = p->bc_lo[d]; g.bc_hi[d] = p->bc_hi[d]; g.grav[d] = p->grav[d]; }
    g.dx = p->dx; g.dy = p->dy; g.dz = p->dz;
    g.rdx = 1.0 / p->dx; g.rdy = 1.0 / p->dy; g.rdz = 1.0 / p->dz;
    g.gamma = p->gamma; g.gm1 = p->gamma - 1.0; g.rgm1 = 1.0 / (p->gamma - 1.0);
    g.gfac = (p->gamma + 1.0) / (2.0 * p->gamma);
    g.small_dens = p->small_dens; g.small_pres = p->small_pres;
    g.plane_g = (long long)g.ex * g.ey;
    g.comp_g = g.plane_g * g.ez;
    g.box_g = g.comp_g * g.nvar;
    g.comp_a = (long long)g.nx * g.ny * g.nz;
    g.box_a = g.comp_a * g.nvar;
    c->launches = 0;
    c->ws = nullptr; c->ws_bytes = 0;
    c->timing = 0;
    c->xplan = nullptr;
    c->has_react = 0;
    c->diff_kth = 0.0; c->diff_cv = 1.0;
    c->flatten = 0;
    c->order = 2;
    c->species_variant = 0;
    c->species_split = 0;
    for (int n = 0; n < 3; ++n) c->ev[n] = nullptr;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaMalloc(&c->d_scratch, 64 * sizeof(double));
    if (e != cudaSuccess) { delete c; return cuda_fail(e); }
    *out = c;
    return CST_OK;
}

extern "C" int cst_destroy(cst_ctx* c)
{
    if (!c) return CST_EINVAL;
    xplan_destroy(c);
    cudaFree(c->d_scratch);
    for (int n = 0; n < 3; ++n) if (c->ev[n]) cudaEventDestroy(c->ev[n]);
    delete c;
    return CST_OK;
}

extern "C" long long cst_workspace_bytes(const cst_ctx* c)
{
    return c ? workspace_bytes(c) : -1;
}

extern "C" int cst_set_workspace(cst_ctx* c, void* ws, long long bytes)
{
    if (!c || !ws || bytes < workspace_bytes(c) || ((uintptr_t)ws & 15)) return CST_EINVAL;
    c->ws = (double*)ws; c->ws_bytes = bytes;
    return CST_OK;
}

static int make_quad(int nquad, const double* const* A_quad, const double* w_quad, QuadArgs& q)
{
    if (nquad < 0 || nquad > CST_MAX_QUAD) return CST_EINVAL;
    if (nquad > 0 && (!A_quad || !w_quad)) return CST_EINVAL;
    q.nquad = nquad;
    for (int n = 0; n < CST_MAX_QUAD; ++n) { q.A[n] = nullptr; q.w[n] = 0.0; }
    for (int n = 0; n < nquad; ++n) {
        if (!A_quad[n]) return CST_EINVAL;
        q.A[n] = A_quad[n]; q.w[n] = w_quad[n];
    }
    return CST_OK;
}

extern "C" int cst_fill_ghosts(cst_ctx* c, double* U, void* stream)
{
    if (!c || !U) return CST_EINVAL;
    return check_launch(launch_fill_ghosts(c, U, (cudaStream_t)stream));
}

extern "C" int cst_advance_A(cst_ctx* c, const double* U, double* A, void* stream)
{
    if (!c || !U || !A) return CST_EINVAL;
    QuadArgs q{};
    return check_launch(launch_advance_A(c, U, A, nullptr, 0.0, nullptr, q, false, (cudaStream_t)stream));
}

extern "C" int cst_sdc_update(cst_ctx* c, double* U_next, const double* U_m, double dt_m,
                              const double* A_new_m, const double* A_old_m,
                              int nquad, const double* const* A_quad, const double* w_quad, void* stream)
{
    if (!c || !U_next || !U_m || !A_new_m || !A_old_m) return CST_EINVAL;
    QuadArgs q;
    int rc = make_quad(nquad, A_quad, w_quad, q);
    if (rc) return rc;
    return check_launch(launch_sdc_update(c, U_next, U_m, dt_m, A_new_m, A_old_m, q, (cudaStream_t)stream));
}

extern "C" int cst_advance_A_update(cst_ctx* c, const double* U_m, double* A_new_m, double* U_next,
                                    double dt_m, const double* A_old_m,
                                    int nquad, const double* const* A_quad, const double* w_quad, void* stream)
{
    if (!c || !U_m || !A_new_m || !U_next || !A_old_m) return CST_EINVAL;
    if (U_next == U_m) return CST_EINVAL;
    QuadArgs q;
    int rc = make_quad(nquad, A_quad, w_quad, q);
    if (rc) return rc;
    // the outputs are written while the inputs are still being read through read-only loads: no output may be
    // an input (A_old_m / A_quad[q] == A_new_m is the documented exception: it means "the value just computed")
    const void* in[2 + CST_MAX_QUAD] = { U_m, A_old_m };
    for (int n = 0; n < nquad; ++n) in[2 + n] = q.A[n];
    for (int n = 0; n < 2 + nquad; ++n) {
        if (in[n] == (const void*)U_next) return CST_EINVAL;
        if (n != 0 && in[n] == (const void*)A_new_m) continue;
        if (in[n] == (const void*)A_new_m) return CST_EINVAL;
    }
    if ((const void*)U_next == (const void*)A_new_m) return CST_EINVAL;
    return check_launch(launch_advance_A(c, U_m, A_new_m, U_next, dt_m, A_old_m, q, true, (cudaStream_t)stream));
}

extern "C" int cst_advance_A_update_cfl(cst_ctx* c, const double* U_m, double* A_new_m, double* U_next,
                                        double dt_m, const double* A_old_m,
                                        int nquad, const double* const* A_quad, const double* w_quad,
                                        double cfl, double* dt_out_dev, void* stream)
{
    if (!c || !U_m || !A_new_m || !U_next || !A_old_m || !dt_out_dev || !(cfl > 0)) return CST_EINVAL;
    if (U_next == U_m) return CST_EINVAL;
    QuadArgs q;
    int rc = make_quad(nquad, A_quad, w_quad, q);
    if (rc) return rc;
    const void* in[2 + CST_MAX_QUAD] = { U_m, A_old_m };
    for (int n = 0; n < nquad; ++n) in[2 + n] = q.A[n];
    for (int n = 0; n < 2 + nquad; ++n) {
        if (in[n] == (const void*)U_next) return CST_EINVAL;
        if (n != 0 && in[n] == (const void*)A_new_m) continue;
        if (in[n] == (const void*)A_new_m) return CST_EINVAL;
    }
    if ((const void*)U_next == (const void*)A_new_m) return CST_EINVAL;
    return check_launch(launch_advance_A_cfl(c, U_m, A_new_m, U_next, dt_m, A_old_m, q, true, cfl, dt_out_dev,
                                             (cudaStream_t)stream));
}

extern "C" int cst_cfl_dt_device(cst_ctx* c, const double* U, double cfl, double* dt_out_dev, void* stream)
{
    if (!c || !U || !dt_out_dev || !(cfl > 0)) return CST_EINVAL;
    return check_launch(launch_cfl(c, U, cfl, dt_out_dev, (cudaStream_t)stream));
}

extern "C" int cst_cfl_dt(cst_ctx* c, const double* U, double cfl, double* dt_out_host, void* stream)
{
    if (!c || !U || !dt_out_host || !(cfl > 0)) return CST_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = check_launch(launch_cfl(c, U, cfl, c->d_scratch + 1, st));
    if (rc) return rc;
    cudaError_t e = cudaMemcpyAsync(dt_out_host, c->d_scratch + 1, sizeof(double), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? CST_OK : cuda_fail(e);
}

extern "C" int cst_validate(cst_ctx* c, const double* U, long long* n_bad_host, void* stream)
{
    if (!c || !U || !n_bad_host) return CST_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = check_launch(launch_validate(c, U, st));
    if (rc) return rc;
    unsigned long long n = 0;
    cudaError_t e = cudaMemcpyAsync(&n, c->d_scratch + 2, sizeof(n), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e);
    *n_bad_host = (long long)n;
    return CST_OK;
}

extern "C" int cst_step_host(cst_ctx* c, const double* U_host, double* A_host, double* U_next_host,
                             double* U_dev, double* U_next_dev, double* A_dev, double dt_m, void* stream)
{
    if (!c || !U_host || !A_host || !U_next_host || !U_dev || !U_next_dev || !A_dev) return CST_EINVAL;
    if (U_dev == U_next_dev) return CST_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Geom& g = c->g;
    const size_t ub = (size_t)g.box_g * g.nbox * sizeof(double), ab = (size_t)g.box_a * g.nbox * sizeof(double);
    cudaError_t e = cudaMemcpyAsync(U_dev, U_host, ub, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e);
    // only interior zones of U_next are written: its ghost shell keeps whatever U_next_dev held (cst.h)
    int rc = check_launch(launch_fill_ghosts(c, U_dev, st));
    if (rc) return rc;
    QuadArgs q{};
    q.nquad = 2; q.A[0] = A_dev; q.A[1] = A_dev; q.w[0] = 0.5 * dt_m; q.w[1] = 0.5 * dt_m;
    rc = check_launch(launch_advance_A(c, U_dev, A_dev, U_next_dev, dt_m, A_dev, q, true, st));
    if (rc) return rc;
    e = cudaMemcpyAsync(A_host, A_dev, ab, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(U_next_host, U_next_dev, ub, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return e == cudaSuccess ? CST_OK : cuda_fail(e);
}

extern "C" int cst_set_variant(cst_ctx* c, int species_variant)
{
    if (!c || species_variant < 0 || species_variant > 3) return CST_EINVAL;
    c->species_variant = species_variant;
    return CST_OK;
}

extern "C" int cst_set_species_split(cst_ctx* c, int split)
{
    if (!c || split < 0 || split > 8) return CST_EINVAL;
    c->species_split = split;
    return CST_OK;
}

extern "C" int cst_get_variant(const cst_ctx* c) { return c ? c->species_variant : CST_EINVAL; }
extern "C" int cst_get_species_split(const cst_ctx* c) { return c ? c->species_split : CST_EINVAL; }

// Times the fused advance with every species-kernel variant on the caller's own buffers and keeps the fastest.
extern "C" int cst_tune_advance(cst_ctx* c, const double* U_m, double* A_new_m, double* U_next, double dt_m,
                                const double* A_old_m, int nquad, const double* const* A_quad, const double* w_quad,
                                int repeats, float* ms_out, void* stream)
{
    if (!c || repeats < 1) return CST_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        if (e0) cudaEventDestroy(e0);
        return cuda_fail(cudaGetLastError());
    }
    const int keep_timing = c->timing;
    c->timing = 0;
    int best = 0, rc = CST_OK;
    float best_ms = 0.f;
    for (int v = 0; v <= 3 && rc == CST_OK; ++v) {
        c->species_variant = v;
        float ms_v = 0.f;
        for (int n = 0; n <= repeats && rc == CST_OK; ++n) {          // the first run of a variant is a warm-up
            cudaEventRecord(e0, st);
            rc = cst_advance_A_update(c, U_m, A_new_m, U_next, dt_m, A_old_m, nquad, A_quad, w_quad, stream);
            cudaEventRecord(e1, st);
            if (rc != CST_OK) break;
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = cuda_fail(cudaGetLastError()); break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (n == 1 || (n > 1 && ms < ms_v)) ms_v = ms;
        }
        if (ms_out) ms_out[v] = ms_v;
        if (v == 0 || ms_v < best_ms) { best = v; best_ms = ms_v; }
    }
    c->species_variant = (rc == CST_OK) ? best : 0;
    // second knob, for the winner only: how many CTAs share one tile (default 3); keep another value only if it is faster
    int best_split = 0;
    for (int sp = 2; sp <= 4 && rc == CST_OK; sp += 2) {
        c->species_split = sp;
        float ms_s = 0.f;
        for (int n = 0; n <= repeats && rc == CST_OK; ++n) {
            cudaEventRecord(e0, st);
            rc = cst_advance_A_update(c, U_m, A_new_m, U_next, dt_m, A_old_m, nquad, A_quad, w_quad, stream);
            cudaEventRecord(e1, st);
            if (rc != CST_OK) break;
            if (cudaEventSynchronize(e1) != cudaSuccess) { rc = cuda_fail(cudaGetLastError()); break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (n == 1 || (n > 1 && ms < ms_s)) ms_s = ms;
        }
        if (ms_out) ms_out[4 + (sp == 4)] = ms_s;
        if (rc == CST_OK && ms_s < best_ms) { best_split = sp; best_ms = ms_s; }
    }
    c->species_split = (rc == CST_OK) ? best_split : 0;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    c->timing = keep_timing;
    if (rc == CST_OK)                   // leave the outputs as the chosen configuration writes them (all agree bit for bit)
        rc = cst_advance_A_update(c, U_m, A_new_m, U_next, dt_m, A_old_m, nquad, A_quad, w_quad, stream);
    return rc;
}

extern "C" long long cst_ctu_workspace_bytes(const cst_ctx* c)
{
    return c ? ctu_workspace_doubles(c->g) * (long long)sizeof(double) : -1;
}

extern "C" int cst_advance_ctu(cst_ctx* c, const double* U, double dt, double* A, void* workspace_dev, long long bytes,
                               void* stream)
{
    if (!c || !U || !A || !workspace_dev || !(dt >= 0.0)) return CST_EINVAL;
    if (bytes < cst_ctu_workspace_bytes(c) || ((uintptr_t)workspace_dev & 15)) return CST_ENOWORKSPACE;
    return check_launch(launch_advance_ctu(c, U, dt, A, (double*)workspace_dev, (cudaStream_t)stream));
}

extern "C" int cst_set_order(cst_ctx* c, int order)
{
    if (!c || (order != 2 && order != 4)) return CST_EINVAL;
    c->order = order;
    return CST_OK;
}

extern "C" int cst_set_flattening(cst_ctx* c, int on)
{
    if (!c) return CST_EINVAL;
    c->flatten = on ? 1 : 0;
    return CST_OK;
}

extern "C" int cst_set_diffusion(cst_ctx* c, double kth, double cv)
{
    if (!c || !(kth >= 0.0) || !(cv > 0.0)) return CST_EINVAL;
    c->diff_kth = kth; c->diff_cv = cv;
    return CST_OK;
}

extern "C" int cst_set_reactions(cst_ctx* c, const cst_react_params* r)
{
    if (!c || !r) return CST_EINVAL;
    if (c->g.nspec < 1 || c->g.nspec > CST_MAX_REACT) return CST_EINVAL;
    if (!(r->cv > 0) || !(r->T0 > 0) || r->max_iter < 1 || !(r->tol > 0)) return CST_EINVAL;
    const unsigned long long zero = 0;
    cudaError_t e = cudaMemcpyAsync(c->d_scratch + 3, &zero, sizeof(zero), cudaMemcpyHostToDevice, 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) return cuda_fail(e);
    c->react = *r;
    c->has_react = 1;
    return CST_OK;
}

extern "C" int cst_react_R(cst_ctx* c, const double* U, double* R, void* stream)
{
    if (!c || !U || !R) return CST_EINVAL;
    return check_launch(launch_react_R(c, U, R, (cudaStream_t)stream));
}

extern "C" int cst_sdc_update_react(cst_ctx* c, double* U_next, const double* U_m, double dt_m,
                                    const double* A_new_m, const double* A_old_m, const double* R_old_next,
                                    int nquad, const double* const* A_quad, const double* const* R_quad,
                                    const double* w_quad, double* R_new_out, void* stream)
{
    if (!c || !U_next || !U_m || !A_new_m || !A_old_m || !R_old_next || !R_new_out) return CST_EINVAL;
    if (nquad < 0 || nquad > CST_MAX_QUAD || (nquad > 0 && (!A_quad || !R_quad || !w_quad))) return CST_EINVAL;
    for (int n = 0; n < nquad; ++n) if (!A_quad[n] || !R_quad[n]) return CST_EINVAL;
    return check_launch(launch_sdc_update_react(c, U_next, U_m, dt_m, A_new_m, A_old_m, R_old_next, nquad, A_quad,
                                                R_quad, w_quad, R_new_out, (cudaStream_t)stream));
}

extern "C" int cst_react_failures(cst_ctx* c, long long* n_host, void* stream)
{
    if (!c || !n_host || !c->has_react) return CST_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long n = 0;
    const unsigned long long zero = 0;
    cudaError_t e = cudaMemcpyAsync(&n, c->d_scratch + 3, sizeof(n), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_scratch + 3, &zero, sizeof(zero), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e);
    *n_host = (long long)n;
    return CST_OK;
}

extern "C" int cst_set_sublattice(cst_ctx* c, const int global_nb[3], const int part[3], int rank)
{
    if (!c || !global_nb || !part) return CST_EINVAL;
    const int rc = xplan_create(c, global_nb, part, rank);
    return rc == CST_ECUDA ? cuda_fail(cudaGetLastError()) : rc;
}

extern "C" int cst_exchange_info(const cst_ctx* c, int* npeers, int* peers, long long* send_off, long long* send_len,
                                 long long* recv_off, long long* recv_len, int cap)
{
    if (!c) return CST_EINVAL;
    return xplan_info(c, npeers, peers, send_off, send_len, recv_off, recv_len, cap);
}

extern "C" int cst_exchange_pack(cst_ctx* c, const double* U, double* sendbuf, void* stream)
{
    if (!c || !U || !sendbuf) return CST_EINVAL;
    return check_launch(launch_exchange_pack(c, U, sendbuf, (cudaStream_t)stream));
}

extern "C" int cst_exchange_unpack(cst_ctx* c, double* U, const double* recvbuf, void* stream)
{
    if (!c || !U || !recvbuf) return CST_EINVAL;
    return check_launch(launch_exchange_unpack(c, U, recvbuf, (cudaStream_t)stream));
}

extern "C" int cst_exchange_push(cst_ctx* c, const double* U, double* const* peer_U, int npeers, void* stream)
{
    if (!c || !U || (npeers > 0 && !peer_U) || npeers < 0) return CST_EINVAL;
    return check_launch(launch_exchange_push(c, U, peer_U, npeers, (cudaStream_t)stream));
}

// CUDA IPC: share the allocation that contains dev_ptr with another process (the ghost exchange over peer memory)
extern "C" int cst_ipc_export(const void* dev_ptr, unsigned char handle[64], long long* offset_bytes)
{
    if (!dev_ptr || !handle || !offset_bytes) return CST_EINVAL;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
    // base of the allocation: the driver's cuMemGetAddressRange (libcst does not link libcuda)
    typedef int (*range_fn)(unsigned long long*, size_t*, unsigned long long);
    void* fp = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fp, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess || !fp)
        return cuda_fail(cudaGetLastError());
    unsigned long long base = 0;
    size_t size = 0;
    if (((range_fn)fp)(&base, &size, (unsigned long long)(uintptr_t)dev_ptr) != 0) return CST_EINVAL;
    cudaIpcMemHandle_t h;
    const cudaError_t e = cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base);
    if (e != cudaSuccess) return cuda_fail(e);
    memcpy(handle, &h, 64);
    *offset_bytes = (long long)((unsigned long long)(uintptr_t)dev_ptr - base);
    return CST_OK;
}

extern "C" int cst_ipc_import(const unsigned char handle[64], long long offset_bytes, void** dev_ptr)
{
    if (!handle || !dev_ptr || offset_bytes < 0) return CST_EINVAL;
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    void* base = nullptr;
    const cudaError_t e = cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess);
    if (e != cudaSuccess) return cuda_fail(e);
    *dev_ptr = (char*)base + offset_bytes;
    return CST_OK;
}

extern "C" int cst_ipc_close(void* mapped_base)
{
    if (!mapped_base) return CST_EINVAL;
    const cudaError_t e = cudaIpcCloseMemHandle(mapped_base);
    return e == cudaSuccess ? CST_OK : cuda_fail(e);
}

extern "C" int cst_set_timing(cst_ctx* c, int on)
{
    if (!c) return CST_EINVAL;
    if (on && !c->ev[0]) {
        for (int n = 0; n < 3; ++n)
            if (cudaEventCreate(&c->ev[n]) != cudaSuccess) {
                const int rc = cuda_fail(cudaGetLastError());
                for (int m = 0; m < 3; ++m) { if (c->ev[m]) cudaEventDestroy(c->ev[m]); c->ev[m] = nullptr; }
                return rc;
            }
    }
    c->timing = on ? 1 : 0;
    return CST_OK;
}

extern "C" int cst_last_advance_ms(cst_ctx* c, double* ms_hydro, double* ms_species)
{
    if (!c || !ms_hydro || !ms_species || !c->ev[0]) return CST_EINVAL;
    cudaError_t e = cudaEventSynchronize(c->ev[2]);
    float a = 0.f, b = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&a, c->ev[0], c->ev[1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&b, c->ev[1], c->ev[2]);
    if (e != cudaSuccess) return cuda_fail(e);
    *ms_hydro = a; *ms_species = b;
    return CST_OK;
}

extern "C" int cst_debug_rcp_sqrt(const double* x_dev, double* rcp_dev, double* sqrt_dev, long long n, void* stream)
{
    if (!x_dev || !rcp_dev || !sqrt_dev || n < 0) return CST_EINVAL;
    return check_launch(launch_debug_rcp_sqrt(x_dev, rcp_dev, sqrt_dev, n, (cudaStream_t)stream));
}

extern "C" long long cst_debug_tile_count(const cst_ctx* c) { return c ? debug_tile_count(c->g) : -1; }

extern "C" int cst_debug_tile_map(cst_ctx* c, int* map_dev, void* stream)
{
    if (!c || !map_dev) return CST_EINVAL;
    return check_launch(launch_debug_tile_map(c, map_dev, (cudaStream_t)stream));
}

extern "C" long long cst_launch_count(const cst_ctx* c) { return c ? c->launches : -1; }

extern "C" const char* cst_strerror(int code)
{
    switch (code) {
    case CST_OK: return "ok";
    case CST_EINVAL: return "invalid argument";
    case CST_ECUDA: return g_cuda_msg;
    case CST_ENOMEM: return "out of host memory";
    case CST_ENOWORKSPACE: return "workspace not set (cst_set_workspace)";
    default: return "unknown error code";
    }
}

extern "C" const char* cst_version(void) { return "libcst 0.3 (sm_100a)"; }
