"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle's tests and the CUDA path, so it holds none of the
method's arithmetic: it only draws random numbers, evaluates the initial-condition formulas
of the configs and packs primitive values into the conserved layout U[b][c][k][j][i].
It never imports the oracle or the CUDA binding.

Every config is generated one GLOBAL k-plane at a time from
numpy.random.default_rng([SEED, config_index, k_global]) (PCG64), so the state does not depend
on how the domain is cut into boxes and big configs can be produced and checked in slabs.
"""
import numpy as np

SEED = 191012578
NG = 4
BC_PERIODIC, BC_OUTFLOW, BC_REFLECT = 0, 1, 2


def _base(name, index, n, nb, nspec, gamma, bc_lo, bc_hi, L, grav=(0.0, 0.0, 0.0), steps=1, cfl=0.5):
    nx, ny, nz = n
    nbx, nby, nbz = nb
    return dict(name=name, index=index, nx=nx, ny=ny, nz=nz, ng=NG, nbx=nbx, nby=nby, nbz=nbz,
                nspec=nspec, dx=L[0] / (nx * nbx), dy=L[1] / (ny * nby), dz=L[2] / (nz * nbz),
                gamma=gamma, grav=tuple(grav), bc_lo=tuple(bc_lo), bc_hi=tuple(bc_hi),
                small_dens=1e-200, small_pres=1e-200, steps=steps, cfl=cfl, L=tuple(L))


def make_config(index, n=None, nb=None, nspec=None):
    """BASELINE.json configs[index]; n = interior zones per box (int or 3-tuple) and nb = box
    lattice (3-tuple) may be overridden to make the small parity-test versions."""
    def tri(v, default):
        if v is None:
            v = default
        return (v, v, v) if isinstance(v, int) else tuple(v)
    P, O, R = BC_PERIODIC, BC_OUTFLOW, BC_REFLECT
    if index == 0:      # Sod split along x + 1e-3 density perturbation, periodic, 1 A + 1 update
        return _base("sod32_periodic", 0, tri(n, 32), tri(nb, 1), 0 if nspec is None else nspec, 1.4,
                     (P, P, P), (P, P, P), (1.0, 1.0, 1.0), steps=1)
    if index == 1:      # oblique Sod, outflow, 50 SDC steps
        return _base("sod3d_oblique", 1, tri(n, 128), tri(nb, 1), 0 if nspec is None else nspec, 1.4,
                     (O, O, O), (O, O, O), (1.0, 1.0, 1.0), steps=50)
    if index == 2:      # Gaussian density pulse, periodic, 20 steps
        return _base("gauss_pulse", 2, tri(n, 256), tri(nb, 1), 0 if nspec is None else nspec, 5.0 / 3.0,
                     (P, P, P), (P, P, P), (1.0, 1.0, 1.0), steps=20)
    if index == 3:      # white-noise box with 13 species
        return _base("noise512_13spec", 3, tri(n, 512), tri(nb, 1), 13 if nspec is None else nspec,
                     5.0 / 3.0, (P, P, P), (P, P, P), (1.0, 1.0, 1.0), steps=1)
    if index == 4:      # XRB-shaped batch of boxes: isothermal atmosphere, reflecting z, gravity
        n3, nb3 = tri(n, 64), tri(nb, (16, 8, 4))
        Dz = n3[2] * nb3[2]
        dz = 1.0 / Dz                       # L_z = 1, dx = dy = dz (SURVEY 8(d) cfg 4)
        L = (n3[0] * nb3[0] * dz, n3[1] * nb3[1] * dz, 1.0)
        return _base("xrb_boxes", 4, n3, nb3, 13 if nspec is None else nspec, 5.0 / 3.0,
                     (P, P, R), (P, P, R), L, grav=(0.0, 0.0, -8.0), steps=10)
    raise ValueError("config index must be 0..4")


def nvar(cfg):
    return 5 + cfg["nspec"]


def domain(cfg):
    return cfg["nx"] * cfg["nbx"], cfg["ny"] * cfg["nby"], cfg["nz"] * cfg["nbz"]


def nzones(cfg):
    Dx, Dy, Dz = domain(cfg)
    return Dx * Dy * Dz


def u_shape(cfg):
    ng = cfg["ng"]
    return (cfg["nbx"] * cfg["nby"] * cfg["nbz"], nvar(cfg),
            cfg["nz"] + 2 * ng, cfg["ny"] + 2 * ng, cfg["nx"] + 2 * ng)


def a_shape(cfg):
    return (cfg["nbx"] * cfg["nby"] * cfg["nbz"], nvar(cfg), cfg["nz"], cfg["ny"], cfg["nx"])


def _dirichlet(rng, nspec, shape):
    E = rng.standard_exponential(size=(nspec,) + shape)
    return E / E.sum(axis=0, keepdims=True)


def prim_plane(cfg, kg):
    """Primitive values W[c][j][i] = (rho, u, v, w, p, X_s) on global plane kg (shape [N, Dy, Dx])."""
    Dx, Dy, Dz = domain(cfg)
    N, ns, idx = nvar(cfg), cfg["nspec"], cfg["index"]
    rng = np.random.default_rng([SEED, idx, int(kg)])
    x = ((np.arange(Dx) + 0.5) * cfg["dx"])[None, :]
    y = ((np.arange(Dy) + 0.5) * cfg["dy"])[:, None]
    z = (kg + 0.5) * cfg["dz"]
    W = np.zeros((N, Dy, Dx))
    shape = (Dy, Dx)
    if idx == 0:
        left = np.broadcast_to(x < 0.5, shape)
        xi = rng.random(shape)
        W[0] = np.where(left, 1.0, 0.125) * (1.0 + 1e-3 * (2.0 * xi - 1.0))
        W[4] = np.where(left, 1.0, 0.1)
    elif idx == 1:
        left = (x + y + z) < 1.5
        W[0] = np.where(left, 1.0, 0.125)
        W[4] = np.where(left, 1.0, 0.1)
    elif idx == 2:
        r2 = (x - 0.5) ** 2 + (y - 0.5) ** 2 + (z - 0.5) ** 2
        W[0] = 1.0 + 0.5 * np.exp(-r2 / 0.01)
        W[1:4] = 1.0
        W[4] = 1.0
    elif idx == 3:
        W[0] = np.exp(0.3 * rng.standard_normal(shape))
        W[1:4] = (0.3 * np.sqrt(cfg["gamma"]) / np.sqrt(3.0)) * rng.standard_normal((3,) + shape)
        W[4] = 1.0
    elif idx == 4:
        H = 1.0 / 8.0
        W[0] = np.exp(-z / H)
        W[1:4] = 1e-4 * np.sqrt(cfg["gamma"]) * rng.standard_normal((3,) + shape)
        W[4] = W[0]
    if ns > 0:
        if idx == 3:
            W[5:] = _dirichlet(rng, ns, shape)
        elif idx == 4:
            # two fixed compositions blended by tanh across mid-height (width 4 dz)
            fix = np.random.default_rng([SEED, idx, 10 ** 6])
            Xa = _dirichlet(fix, ns, (1, 1))
            Xb = _dirichlet(fix, ns, (1, 1))
            s = 0.5 * (1.0 + np.tanh((z - 0.5) / (4.0 * cfg["dz"])))
            W[5:] = (1.0 - s) * Xa + s * Xb
        else:
            # NVAR=5 configs run with species only in extra tests: smooth, space-dependent X
            Xs = 1.0 + 0.5 * np.sin(2 * np.pi * (x + 2 * y + 3 * z) + np.arange(ns)[:, None, None])
            W[5:] = Xs / Xs.sum(axis=0, keepdims=True)
    return W


def cons_from_prim(cfg, W):
    """Pack primitives into the conserved layout (input preparation, not the method's S1)."""
    U = np.empty_like(W)
    rho = W[0]
    U[0] = rho
    U[1:4] = rho * W[1:4]
    U[4] = W[4] / (cfg["gamma"] - 1.0) + 0.5 * rho * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)
    U[5:] = rho * W[5:]
    return U


def cons_plane(cfg, kg):
    return cons_from_prim(cfg, prim_plane(cfg, kg))


def scatter_plane(cfg, Ubox, kg, plane, brick=None):
    """Write global plane kg (array [N, Dy, Dx], numpy or torch) into the box-layout array
    Ubox[b][c][k][j][i] (numpy or torch; ghosts untouched).  brick = (origin, lattice) of a rank's brick of the box
    lattice (box coordinates; paper_1910_12578_b200/shard.py): Ubox then holds only that brick's boxes, in the
    brick's local order, and planes outside it are ignored."""
    ng, nx, ny, nz = cfg["ng"], cfg["nx"], cfg["ny"], cfg["nz"]
    (ox, oy, oz), (lx, ly, lz) = brick if brick is not None else ((0, 0, 0), (cfg["nbx"], cfg["nby"], cfg["nbz"]))
    bk, lk = divmod(int(kg), nz)
    if not (oz <= bk < oz + lz):
        return
    for bj in range(oy, oy + ly):
        for bi in range(ox, ox + lx):
            b = (bi - ox) + lx * ((bj - oy) + ly * (bk - oz))
            Ubox[b, :, lk + ng, ng:ng + ny, ng:ng + nx] = \
                plane[:, bj * ny:(bj + 1) * ny, bi * nx:(bi + 1) * nx]


def initial_state(cfg, ghost_value=np.nan):
    """Whole ghosted state on the host; ghosts hold ghost_value until a ghost fill."""
    U = np.full(u_shape(cfg), ghost_value, dtype=np.float64)
    for kg in range(domain(cfg)[2]):
        scatter_plane(cfg, U, kg, cons_plane(cfg, kg))
    return U


def to_global(cfg, Abox, ghosted=False):
    """Box-layout interior array -> global array [N, Dz, Dy, Dx] (for checks and plots)."""
    ng = cfg["ng"] if ghosted else 0
    nx, ny, nz = cfg["nx"], cfg["ny"], cfg["nz"]
    Dx, Dy, Dz = domain(cfg)
    G = np.empty((nvar(cfg), Dz, Dy, Dx))
    for bk in range(cfg["nbz"]):
        for bj in range(cfg["nby"]):
            for bi in range(cfg["nbx"]):
                b = bi + cfg["nbx"] * (bj + cfg["nby"] * bk)
                G[:, bk * nz:(bk + 1) * nz, bj * ny:(bj + 1) * ny, bi * nx:(bi + 1) * nx] = \
                    Abox[b][:, ng:ng + nz, ng:ng + ny, ng:ng + nx]
    return G


def from_global(cfg, G):
    """Global interior array [N, Dz, Dy, Dx] -> ghosted box layout (ghosts NaN)."""
    U = np.full(u_shape(cfg), np.nan)
    for kg in range(G.shape[1]):
        scatter_plane(cfg, U, kg, G[:, kg])
    return U


def random_state(cfg, seed, amp=0.3):
    """Generic seeded white-noise state for invariance tests: log-normal rho, Gaussian v,
    log-normal p, Dirichlet X.  Returns ghosted box layout with NaN ghosts."""
    Dx, Dy, Dz = domain(cfg)
    rng = np.random.default_rng([SEED, 99, int(seed)])
    W = np.zeros((nvar(cfg), Dz, Dy, Dx))
    W[0] = np.exp(amp * rng.standard_normal((Dz, Dy, Dx)))
    W[1:4] = amp * rng.standard_normal((3, Dz, Dy, Dx))
    W[4] = np.exp(amp * rng.standard_normal((Dz, Dy, Dx)))
    if cfg["nspec"]:
        E = rng.standard_exponential((cfg["nspec"], Dz, Dy, Dx))
        W[5:] = E / E.sum(axis=0, keepdims=True)
    return from_global(cfg, cons_from_prim(cfg, W))


def react_params(nspec, stiff=1.0, nu=4.0, seed=0):
    """Parameters of the synthetic stiff reaction chain X_0 -> X_1 -> ... (readings R1-R4; stands in for
    the paper's 13-isotope network, whose rate tables are not available).  Input data only: rate[k] of species k ->
    k+1 at T = T0 (spread over two decades, seeded), the specific energy release q[k], the constant c_v of the
    temperature T = e / c_v, the exponent nu of the rates' power law, and the Newton controls."""
    rng = np.random.default_rng([SEED, 77, int(seed), int(nspec)])
    rate = stiff * 10.0 ** rng.uniform(0.0, 2.0, size=nspec)
    q = 0.02 * rng.uniform(0.5, 1.5, size=nspec)
    return dict(cv=1.5, T0=1.0, nu=float(nu), rate=[float(x) for x in rate], q=[float(x) for x in q],
                max_iter=50, tol=1e-13)
