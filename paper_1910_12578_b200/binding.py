"""Thin Python binding of the C-ABI library libcst.so (include/cst.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  torch is used for device
memory and streams.  There is no CPU fallback: if libcst.so is missing or cannot be loaded the
first call raises.  Function names mirror the C entry points without the cst_ prefix.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcst.so")
MAX_QUAD = 4

EXPORTS = ["cst_create", "cst_destroy", "cst_workspace_bytes", "cst_set_workspace", "cst_fill_ghosts", "cst_advance_A", "cst_sdc_update",
           "cst_advance_A_update", "cst_cfl_dt_device", "cst_cfl_dt", "cst_validate", "cst_step_host",
           "cst_set_timing", "cst_last_advance_ms", "cst_launch_count", "cst_strerror", "cst_version"]


class CstParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
                ("nbx", C.c_int), ("nby", C.c_int), ("nbz", C.c_int), ("nspec", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("gamma", C.c_double), ("grav", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("small_dens", C.c_double), ("small_pres", C.c_double)]


class CstError(RuntimeError):
    def __init__(self, code, what, msg):
        super().__init__(f"{what}: error {code} ({msg})")
        self.code = code


_lib = None
_vp, _dp = C.c_void_p, C.POINTER(C.c_double)


def load():
    """Load libcst.so; raises (loudly) if the CUDA extension has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1910_12578_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    P = C.POINTER(CstParams)
    lib.cst_create.argtypes = [P, C.POINTER(_vp)]
    lib.cst_destroy.argtypes = [_vp]
    lib.cst_workspace_bytes.argtypes = [_vp]
    lib.cst_workspace_bytes.restype = C.c_longlong
    lib.cst_set_workspace.argtypes = [_vp, _vp, C.c_longlong]
    lib.cst_fill_ghosts.argtypes = [_vp, _vp, _vp]
    lib.cst_advance_A.argtypes = [_vp, _vp, _vp, _vp]
    lib.cst_sdc_update.argtypes = [_vp, _vp, _vp, C.c_double, _vp, _vp, C.c_int, C.POINTER(_vp), _dp, _vp]
    lib.cst_advance_A_update.argtypes = [_vp, _vp, _vp, _vp, C.c_double, _vp, C.c_int, C.POINTER(_vp), _dp, _vp]
    lib.cst_cfl_dt_device.argtypes = [_vp, _vp, C.c_double, _vp, _vp]
    lib.cst_cfl_dt.argtypes = [_vp, _vp, C.c_double, _dp, _vp]
    lib.cst_validate.argtypes = [_vp, _vp, C.POINTER(C.c_longlong), _vp]
    lib.cst_step_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_double, _vp]
    lib.cst_set_timing.argtypes = [_vp, C.c_int]
    lib.cst_last_advance_ms.argtypes = [_vp, _dp, _dp]
    lib.cst_launch_count.argtypes = [_vp]
    lib.cst_launch_count.restype = C.c_longlong
    lib.cst_strerror.argtypes = [C.c_int]
    lib.cst_strerror.restype = C.c_char_p
    lib.cst_version.restype = C.c_char_p
    _lib = lib
    return lib


def make_params(cfg) -> CstParams:
    p = CstParams()
    for k in ("nx", "ny", "nz", "ng", "nbx", "nby", "nbz", "nspec"):
        setattr(p, k, int(cfg[k]))
    for k in ("dx", "dy", "dz", "gamma", "small_dens", "small_pres"):
        setattr(p, k, float(cfg[k]))
    for d in range(3):
        p.grav[d] = float(cfg["grav"][d])
        p.bc_lo[d] = int(cfg["bc_lo"][d])
        p.bc_hi[d] = int(cfg["bc_hi"][d])
    return p


def _ptr(t):
    """Device (or host) address of a contiguous float64 torch tensor / numpy array / int."""
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous() and t.element_size() == 8
        return t.data_ptr()
    assert t.flags["C_CONTIGUOUS"] and t.itemsize == 8
    return t.ctypes.data


def _stream(stream):
    if stream is not None:
        return int(stream)
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


class Context:
    """Owns one cst_ctx.  Methods mirror the C entry points (same names, same argument order)."""

    def __init__(self, cfg, workspace="auto"):
        """workspace="auto": a torch uint8 tensor of workspace_bytes() is allocated on the current CUDA
        device and handed to cst_set_workspace (the library itself never allocates it);
        workspace=None: the caller calls set_workspace() later."""
        self.lib = load()
        self.cfg = dict(cfg)
        self._h = _vp()
        self._ws = None
        self._check(self.lib.cst_create(C.byref(make_params(cfg)), C.byref(self._h)), "cst_create")
        if workspace == "auto":
            import torch
            self.set_workspace(torch.empty(self.workspace_bytes(), dtype=torch.uint8, device="cuda"))
        elif workspace is not None:
            self.set_workspace(workspace)

    def workspace_bytes(self):
        return int(self.lib.cst_workspace_bytes(self._h))

    def set_workspace(self, buf):
        """buf: contiguous torch CUDA tensor (any dtype) of at least workspace_bytes() bytes; kept alive here."""
        nbytes = buf.numel() * buf.element_size()
        self._check(self.lib.cst_set_workspace(self._h, buf.data_ptr(), nbytes), "cst_set_workspace")
        self._ws = buf

    def _check(self, rc, what):
        if rc != 0:
            raise CstError(rc, what, self.lib.cst_strerror(rc).decode())

    def destroy(self):
        if self._h:
            self.lib.cst_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _quad(self, A_quad, w_quad):
        n = len(A_quad)
        assert n == len(w_quad)
        arr = (_vp * max(n, 1))(*[_ptr(a) for a in A_quad])
        w = (C.c_double * max(n, 1))(*[float(x) for x in w_quad])
        return n, arr, w

    def fill_ghosts(self, U, stream=None):
        self._check(self.lib.cst_fill_ghosts(self._h, _ptr(U), _stream(stream)), "cst_fill_ghosts")

    def advance_A(self, U, A, stream=None):
        self._check(self.lib.cst_advance_A(self._h, _ptr(U), _ptr(A), _stream(stream)), "cst_advance_A")

    def sdc_update(self, U_next, U_m, dt_m, A_new_m, A_old_m, A_quad, w_quad, stream=None):
        n, arr, w = self._quad(A_quad, w_quad)
        self._check(self.lib.cst_sdc_update(self._h, _ptr(U_next), _ptr(U_m), float(dt_m), _ptr(A_new_m),
                                            _ptr(A_old_m), n, arr, w, _stream(stream)), "cst_sdc_update")

    def advance_A_update(self, U_m, A_new_m, U_next, dt_m, A_old_m, A_quad, w_quad, stream=None):
        n, arr, w = self._quad(A_quad, w_quad)
        self._check(self.lib.cst_advance_A_update(self._h, _ptr(U_m), _ptr(A_new_m), _ptr(U_next), float(dt_m),
                                                  _ptr(A_old_m), n, arr, w, _stream(stream)),
                    "cst_advance_A_update")

    def cfl_dt_device(self, U, cfl, dt_out_dev, stream=None):
        self._check(self.lib.cst_cfl_dt_device(self._h, _ptr(U), float(cfl), _ptr(dt_out_dev), _stream(stream)),
                    "cst_cfl_dt_device")

    def cfl_dt(self, U, cfl, stream=None):
        out = C.c_double(0.0)
        self._check(self.lib.cst_cfl_dt(self._h, _ptr(U), float(cfl), C.byref(out), _stream(stream)), "cst_cfl_dt")
        return out.value

    def validate(self, U, stream=None):
        n = C.c_longlong(0)
        self._check(self.lib.cst_validate(self._h, _ptr(U), C.byref(n), _stream(stream)), "cst_validate")
        return n.value

    def step_host(self, U_host, A_host, U_next_host, U_dev, U_next_dev, A_dev, dt_m, stream=None):
        self._check(self.lib.cst_step_host(self._h, _ptr(U_host), _ptr(A_host), _ptr(U_next_host), _ptr(U_dev),
                                           _ptr(U_next_dev), _ptr(A_dev), float(dt_m), _stream(stream)),
                    "cst_step_host")

    def set_timing(self, on):
        self._check(self.lib.cst_set_timing(self._h, int(bool(on))), "cst_set_timing")

    def last_advance_ms(self):
        a, b = C.c_double(0.0), C.c_double(0.0)
        self._check(self.lib.cst_last_advance_ms(self._h, C.byref(a), C.byref(b)), "cst_last_advance_ms")
        return a.value, b.value

    def launch_count(self):
        return int(self.lib.cst_launch_count(self._h))


def sdc_step_2nd(ctx, U, U1, A0, A1, dt, stream=None):
    """One 2-node, 2-iteration SDC step (trapezoid, R = 0) from library calls only.
    U: state with interior valid (ghosts are filled here); result left in U (interior).
    U1, A0, A1: caller-owned work buffers (U1 like U, A0/A1 interior-sized)."""
    w = [0.5 * dt, 0.5 * dt]
    ctx.fill_ghosts(U, stream)
    # iteration 1: every node carries A(U^n): A0 = A(U), U1 = U + dt*A0 (fused)
    ctx.advance_A_update(U, A0, U1, dt, A0, [A0, A0], w, stream)
    ctx.fill_ghosts(U1, stream)
    ctx.advance_A(U1, A1, stream)
    # iteration 2: node 0 unchanged, integral from iteration-1 values (trapezoid)
    ctx.sdc_update(U, U, dt, A0, A0, [A0, A1], w, stream)


# Gauss-Lobatto node-to-node quadrature weights (fractions of dt) for M = 2 (trapezoid) and M = 3 (Simpson),
# PAPER.md L44; rows m = 0..M-2, columns j = 0..M-1 (Q17).
_SDC_WEIGHTS = {2: [[1.0 / 2.0, 1.0 / 2.0]],
                3: [[5.0 / 24.0, 8.0 / 24.0, -1.0 / 24.0], [-1.0 / 24.0, 8.0 / 24.0, 5.0 / 24.0]]}


def sdc_step_nodes(ctx, U, dt, M=3, K=4, stream=None):
    """One SDC step with M Gauss-Lobatto nodes and K iterations (Eq. (2) of the paper, R = 0) from library
    calls only: cst_fill_ghosts, cst_advance_A, cst_sdc_update.  U: state with interior valid; result left
    in U (interior).  Work buffers (M - 1 states, 2 M - 1 A arrays) are torch allocations made here."""
    import torch
    wt = _SDC_WEIGHTS[M]
    dtm = dt / (M - 1)
    ashape = (U.shape[0], U.shape[1], U.shape[2] - 8, U.shape[3] - 8, U.shape[4] - 8)
    new_A = lambda: torch.empty(ashape, dtype=U.dtype, device=U.device)
    ctx.fill_ghosts(U, stream)
    A0 = new_A()
    ctx.advance_A(U, A0, stream)
    A_old = [A0] * M
    A_buf = [[new_A() for _ in range(M - 1)] for _ in range(2)]
    U_nodes = [U] + [torch.empty_like(U) for _ in range(M - 1)]
    for k in range(K):
        A_new = [A0]
        for m in range(M - 1):
            ctx.sdc_update(U_nodes[m + 1], U_nodes[m], dtm, A_new[m], A_old[m], A_old,
                           [w * dt for w in wt[m]], stream)
            if k == K - 1 and m == M - 2:
                break
            ctx.fill_ghosts(U_nodes[m + 1], stream)
            ctx.advance_A(U_nodes[m + 1], A_buf[k % 2][m], stream)
            A_new.append(A_buf[k % 2][m])
        A_old = A_new
    if M > 1:
        U.copy_(U_nodes[M - 1])
