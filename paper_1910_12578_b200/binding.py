"""Thin Python binding of the C-ABI library libcst.so (include/cst.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI.  torch is used for device
memory and streams.  There is no CPU fallback: if libcst.so is missing or cannot be loaded the
first call raises.  Function names mirror the C entry points without the cst_ prefix.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("CST_LIB_PATH") or os.path.join(_HERE, "libcst.so")   # override: A/B builds while tuning
MAX_QUAD = 4

EXPORTS = ["cst_create", "cst_destroy", "cst_workspace_bytes", "cst_set_workspace", "cst_fill_ghosts", "cst_advance_A", "cst_sdc_update",
           "cst_advance_A_update", "cst_advance_A_update_cfl", "cst_cfl_dt_device", "cst_cfl_dt", "cst_validate", "cst_step_host",
           "cst_set_timing", "cst_last_advance_ms", "cst_launch_count", "cst_strerror", "cst_version",
           "cst_debug_rcp_sqrt", "cst_debug_tile_count", "cst_debug_tile_map",
           "cst_set_variant", "cst_get_variant", "cst_set_species_split", "cst_get_species_split",
           "cst_tune_advance", "cst_ctu_workspace_bytes", "cst_advance_ctu", "cst_set_order", "cst_set_flattening", "cst_set_diffusion", "cst_set_reactions", "cst_react_R", "cst_sdc_update_react", "cst_react_failures",
           "cst_exchange_plan", "cst_set_sublattice", "cst_exchange_info", "cst_exchange_pack", "cst_exchange_unpack",
           "cst_exchange_push", "cst_ipc_export", "cst_ipc_import", "cst_ipc_close"]


class CstParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
                ("nbx", C.c_int), ("nby", C.c_int), ("nbz", C.c_int), ("nspec", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("gamma", C.c_double), ("grav", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("small_dens", C.c_double), ("small_pres", C.c_double)]


MAX_REACT = 15


class CstReactParams(C.Structure):
    """cst_react_params of include/cst.h: the synthetic stiff reaction chain."""
    _fields_ = [("cv", C.c_double), ("T0", C.c_double), ("nu", C.c_double),
                ("rate", C.c_double * MAX_REACT), ("q", C.c_double * MAX_REACT),
                ("max_iter", C.c_int), ("tol", C.c_double)]


class CstXseg(C.Structure):
    """cst_xseg of include/cst.h: one ghost region that crosses ranks."""
    _fields_ = [("peer", C.c_int), ("box", C.c_int), ("lo", C.c_int * 3), ("step", C.c_int * 3),
                ("ext", C.c_int * 3), ("flip", C.c_int * 3), ("offset", C.c_longlong),
                ("rbox", C.c_int), ("rlo", C.c_int * 3)]


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
    lib.cst_advance_A_update_cfl.argtypes = [_vp, _vp, _vp, _vp, C.c_double, _vp, C.c_int, C.POINTER(_vp), _dp,
                                             C.c_double, _vp, _vp]
    lib.cst_cfl_dt_device.argtypes = [_vp, _vp, C.c_double, _vp, _vp]
    lib.cst_cfl_dt.argtypes = [_vp, _vp, C.c_double, _dp, _vp]
    lib.cst_validate.argtypes = [_vp, _vp, C.POINTER(C.c_longlong), _vp]
    lib.cst_step_host.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, C.c_double, _vp]
    lib.cst_set_timing.argtypes = [_vp, C.c_int]
    lib.cst_last_advance_ms.argtypes = [_vp, _dp, _dp]
    lib.cst_debug_rcp_sqrt.argtypes = [_vp, _vp, _vp, C.c_longlong, _vp]
    lib.cst_debug_tile_count.argtypes = [_vp]
    lib.cst_debug_tile_count.restype = C.c_longlong
    lib.cst_debug_tile_map.argtypes = [_vp, _vp, _vp]
    lib.cst_launch_count.argtypes = [_vp]
    lib.cst_launch_count.restype = C.c_longlong
    lib.cst_set_variant.argtypes = [_vp, C.c_int]
    lib.cst_get_variant.argtypes = [_vp]
    lib.cst_set_species_split.argtypes = [_vp, C.c_int]
    lib.cst_get_species_split.argtypes = [_vp]
    lib.cst_tune_advance.argtypes = [_vp, _vp, _vp, _vp, C.c_double, _vp, C.c_int, C.POINTER(_vp), _dp, C.c_int,
                                     C.POINTER(C.c_float), _vp]
    lib.cst_ctu_workspace_bytes.argtypes = [_vp]
    lib.cst_ctu_workspace_bytes.restype = C.c_longlong
    lib.cst_advance_ctu.argtypes = [_vp, _vp, C.c_double, _vp, _vp, C.c_longlong, _vp]
    lib.cst_set_order.argtypes = [_vp, C.c_int]
    lib.cst_set_flattening.argtypes = [_vp, C.c_int]
    lib.cst_set_diffusion.argtypes = [_vp, C.c_double, C.c_double]
    lib.cst_set_reactions.argtypes = [_vp, C.POINTER(CstReactParams)]
    lib.cst_react_R.argtypes = [_vp, _vp, _vp, _vp]
    lib.cst_sdc_update_react.argtypes = [_vp, _vp, _vp, C.c_double, _vp, _vp, _vp, C.c_int, C.POINTER(_vp),
                                         C.POINTER(_vp), _dp, _vp, _vp]
    lib.cst_react_failures.argtypes = [_vp, C.POINTER(C.c_longlong), _vp]
    I3, LLP = C.POINTER(C.c_int), C.POINTER(C.c_longlong)
    lib.cst_exchange_plan.argtypes = [P, I3, C.c_int, C.c_int, C.POINTER(CstXseg), C.c_longlong]
    lib.cst_exchange_plan.restype = C.c_longlong
    lib.cst_set_sublattice.argtypes = [_vp, I3, I3, C.c_int]
    lib.cst_exchange_info.argtypes = [_vp, I3, I3, LLP, LLP, LLP, LLP, C.c_int]
    lib.cst_exchange_pack.argtypes = [_vp, _vp, _vp, _vp]
    lib.cst_exchange_unpack.argtypes = [_vp, _vp, _vp, _vp]
    lib.cst_exchange_push.argtypes = [_vp, _vp, C.POINTER(_vp), C.c_int, _vp]
    lib.cst_ipc_export.argtypes = [_vp, C.c_char_p, LLP]
    lib.cst_ipc_import.argtypes = [C.c_char_p, C.c_longlong, C.POINTER(_vp)]
    lib.cst_ipc_close.argtypes = [_vp]
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


def exchange_plan(cfg_global, part, rank, recv):
    """cst_exchange_plan (pure host function, needs no GPU): the list of CstXseg of `rank` for the GLOBAL lattice
    described by cfg_global cut into part[0] x part[1] x part[2] bricks."""
    lib = load()
    p = make_params(cfg_global)
    pa = (C.c_int * 3)(*[int(x) for x in part])
    n = lib.cst_exchange_plan(C.byref(p), pa, int(rank), int(bool(recv)), None, 0)
    if n < 0:
        raise CstError(n, "cst_exchange_plan", lib.cst_strerror(int(n)).decode())
    segs = (CstXseg * max(int(n), 1))()
    lib.cst_exchange_plan(C.byref(p), pa, int(rank), int(bool(recv)), segs, n)
    return [segs[i] for i in range(int(n))]


def ipc_export(t):
    """(64-byte handle, offset) of the CUDA allocation that holds the tensor / address t, for cst_ipc_import elsewhere."""
    lib = load()
    h = C.create_string_buffer(64)
    off = C.c_longlong(0)
    rc = lib.cst_ipc_export(_ptr(t), h, C.byref(off))
    if rc:
        raise CstError(rc, "cst_ipc_export", lib.cst_strerror(rc).decode())
    return h.raw, off.value


def ipc_import(handle, offset):
    """device address (int) of another process's array; close with ipc_close(address - offset)."""
    lib = load()
    p = _vp()
    rc = lib.cst_ipc_import(handle, int(offset), C.byref(p))
    if rc:
        raise CstError(rc, "cst_ipc_import", lib.cst_strerror(rc).decode())
    return int(p.value)


def ipc_close(mapped_base):
    load().cst_ipc_close(int(mapped_base))


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

    def advance_A_update_cfl(self, U_m, A_new_m, U_next, dt_m, A_old_m, A_quad, w_quad, cfl, dt_out_dev, stream=None):
        n, arr, w = self._quad(A_quad, w_quad)
        self._check(self.lib.cst_advance_A_update_cfl(self._h, _ptr(U_m), _ptr(A_new_m), _ptr(U_next), float(dt_m),
                                                      _ptr(A_old_m), n, arr, w, float(cfl), _ptr(dt_out_dev),
                                                      _stream(stream)), "cst_advance_A_update_cfl")

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

    def set_variant(self, species_variant):
        self._check(self.lib.cst_set_variant(self._h, int(species_variant)), "cst_set_variant")

    def get_variant(self):
        return int(self.lib.cst_get_variant(self._h))

    def set_species_split(self, split):
        self._check(self.lib.cst_set_species_split(self._h, int(split)), "cst_set_species_split")

    def get_species_split(self):
        return int(self.lib.cst_get_species_split(self._h))

    def tune_advance(self, U_m, A_new_m, U_next, dt_m, A_old_m, A_quad, w_quad, repeats=2, stream=None):
        """cst_tune_advance: times the fused advance with every species-kernel variant, keeps the fastest.
        -> (chosen variant, [ms of variant 0, 1, 2, 3 at the default split, ms of the winner at split 2 and 4])."""
        n, arr, w = self._quad(A_quad, w_quad)
        ms = (C.c_float * 6)()
        self._check(self.lib.cst_tune_advance(self._h, _ptr(U_m), _ptr(A_new_m), _ptr(U_next), float(dt_m), _ptr(A_old_m),
                                              n, arr, w, int(repeats), ms, _stream(stream)), "cst_tune_advance")
        return self.get_variant(), [float(x) for x in ms]

    def ctu_workspace_bytes(self):
        return int(self.lib.cst_ctu_workspace_bytes(self._h))

    def advance_ctu(self, U, dt, A, workspace, stream=None):
        """A <- A_ctu(U, dt) (unsplit CTU PPM); workspace: contiguous device tensor of >= ctu_workspace_bytes() bytes."""
        nbytes = workspace.numel() * workspace.element_size()
        self._check(self.lib.cst_advance_ctu(self._h, _ptr(U), float(dt), _ptr(A), workspace.data_ptr(), nbytes,
                                             _stream(stream)), "cst_advance_ctu")

    def set_order(self, order):
        """Spatial order of <A(U)>: 2 (default) or 4; changes workspace_bytes(): set the workspace afterwards."""
        self._check(self.lib.cst_set_order(self._h, int(order)), "cst_set_order")

    def set_flattening(self, on):
        """Switch CW84 shock flattening on / off; enlarges workspace_bytes(): set the workspace afterwards."""
        self._check(self.lib.cst_set_flattening(self._h, int(bool(on))), "cst_set_flattening")

    def set_diffusion(self, kth, cv):
        self._check(self.lib.cst_set_diffusion(self._h, float(kth), float(cv)), "cst_set_diffusion")

    def set_reactions(self, react):
        """react: dict(cv, T0, nu, rate=[...], q=[...], max_iter, tol) (workloads.react_params)."""
        r = CstReactParams()
        r.cv, r.T0, r.nu = float(react["cv"]), float(react["T0"]), float(react["nu"])
        for k, v in enumerate(react["rate"]):
            r.rate[k] = float(v)
        for k, v in enumerate(react["q"]):
            r.q[k] = float(v)
        r.max_iter, r.tol = int(react["max_iter"]), float(react["tol"])
        self._check(self.lib.cst_set_reactions(self._h, C.byref(r)), "cst_set_reactions")

    def react_R(self, U, R, stream=None):
        self._check(self.lib.cst_react_R(self._h, _ptr(U), _ptr(R), _stream(stream)), "cst_react_R")

    def sdc_update_react(self, U_next, U_m, dt_m, A_new_m, A_old_m, R_old_next, A_quad, R_quad, w_quad, R_new_out,
                         stream=None):
        n, arr, w = self._quad(A_quad, w_quad)
        assert len(R_quad) == n
        rarr = (_vp * max(n, 1))(*[_ptr(a) for a in R_quad])
        self._check(self.lib.cst_sdc_update_react(self._h, _ptr(U_next), _ptr(U_m), float(dt_m), _ptr(A_new_m),
                                                  _ptr(A_old_m), _ptr(R_old_next), n, arr, rarr, w, _ptr(R_new_out),
                                                  _stream(stream)), "cst_sdc_update_react")

    def react_failures(self, stream=None):
        n = C.c_longlong(0)
        self._check(self.lib.cst_react_failures(self._h, C.byref(n), _stream(stream)), "cst_react_failures")
        return n.value

    def set_sublattice(self, global_nb, part, rank):
        g = (C.c_int * 3)(*[int(x) for x in global_nb])
        p = (C.c_int * 3)(*[int(x) for x in part])
        self._check(self.lib.cst_set_sublattice(self._h, g, p, int(rank)), "cst_set_sublattice")

    def exchange_info(self):
        """-> list of (peer, send_off, send_len, recv_off, recv_len), offsets / lengths in doubles."""
        cap = 32
        n = C.c_int(0)
        peers = (C.c_int * cap)()
        arr = [(C.c_longlong * cap)() for _ in range(4)]
        self._check(self.lib.cst_exchange_info(self._h, C.byref(n), peers, arr[0], arr[1], arr[2], arr[3], cap),
                    "cst_exchange_info")
        return [(peers[i], arr[0][i], arr[1][i], arr[2][i], arr[3][i]) for i in range(n.value)]

    def exchange_pack(self, U, sendbuf, stream=None):
        self._check(self.lib.cst_exchange_pack(self._h, _ptr(U), _ptr(sendbuf), _stream(stream)), "cst_exchange_pack")

    def exchange_unpack(self, U, recvbuf, stream=None):
        self._check(self.lib.cst_exchange_unpack(self._h, _ptr(U), _ptr(recvbuf), _stream(stream)), "cst_exchange_unpack")

    def exchange_push(self, U, peer_U, stream=None):
        """peer_U: one device array / address per peer (exchange_info order): the base of that peer's U."""
        n = len(peer_U)
        arr = (_vp * max(n, 1))(*[_ptr(p) for p in peer_U])
        self._check(self.lib.cst_exchange_push(self._h, _ptr(U), arr, n, _stream(stream)), "cst_exchange_push")

    def set_timing(self, on):
        self._check(self.lib.cst_set_timing(self._h, int(bool(on))), "cst_set_timing")

    def last_advance_ms(self):
        a, b = C.c_double(0.0), C.c_double(0.0)
        self._check(self.lib.cst_last_advance_ms(self._h, C.byref(a), C.byref(b)), "cst_last_advance_ms")
        return a.value, b.value

    def launch_count(self):
        return int(self.lib.cst_launch_count(self._h))

    def debug_rcp_sqrt(self, x, rcp, sqrt, stream=None):
        self._check(self.lib.cst_debug_rcp_sqrt(_ptr(x), _ptr(rcp), _ptr(sqrt), x.numel(), _stream(stream)),
                    "cst_debug_rcp_sqrt")

    def debug_tile_count(self):
        return int(self.lib.cst_debug_tile_count(self._h))

    def debug_tile_map(self, out_int32, stream=None):
        assert out_int32.is_contiguous() and out_int32.element_size() == 4
        self._check(self.lib.cst_debug_tile_map(self._h, out_int32.data_ptr(), _stream(stream)), "cst_debug_tile_map")
