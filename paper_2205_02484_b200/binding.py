"""ctypes binding of libcuharm.so: the functions of include/cuharm.h under the same names, plus `Solver`,
a convenience object that owns the torch tensors (prim, workspace) the library borrows.

Marshalling only.  Device pointers come from torch CUDA tensors; host scalars come back as Python floats.
"""
import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


class CuharmError(RuntimeError):
    pass


class CuharmParams(C.Structure):
    """Mirror of `cuharm_params` (include/cuharm.h)."""
    _fields_ = [
        ("struct_bytes", C.c_int32),
        ("n1", C.c_int32), ("n2", C.c_int32), ("n3", C.c_int32), ("ng", C.c_int32),
        ("coords", C.c_int32),
        ("a", C.c_double), ("gam", C.c_double),
        ("r_in", C.c_double), ("r_out", C.c_double), ("R0", C.c_double), ("hslope", C.c_double),
        ("xmin", C.c_double * 3), ("xmax", C.c_double * 3),
        ("recon", C.c_int32), ("riemann", C.c_int32),
        ("bc_x1", C.c_int32), ("bc_x2", C.c_int32), ("bc_x3", C.c_int32),
        ("rho_fl_coef", C.c_double), ("rho_fl_pow", C.c_double), ("rho_fl_abs", C.c_double),
        ("u_fl_coef", C.c_double), ("u_fl_pow", C.c_double), ("u_fl_abs", C.c_double),
        ("sigma_max", C.c_double), ("b2_over_u_max", C.c_double), ("gamma_max", C.c_double),
        ("newton_tol", C.c_double),
        ("newton_maxit", C.c_int32), ("newton_extra", C.c_int32),
        ("fixup_max_passes", C.c_int32), ("n_x", C.c_int32),
        ("r_break", C.c_double),
        ("inv_chain", C.c_int32), ("brent_maxit", C.c_int32),
        ("beta_min", C.c_double), ("brent_tol", C.c_double),
        ("polar_damp", C.c_int32),
        ("n1_global", C.c_int32), ("i_offset", C.c_int32), ("slab_lo", C.c_int32), ("slab_hi", C.c_int32),
        ("reserved", C.c_int32),
    ]


def make_params(d: dict) -> CuharmParams:
    p = CuharmParams()
    p.struct_bytes = C.sizeof(CuharmParams)
    for k, v in d.items():
        if k in ("xmin", "xmax"):
            setattr(p, k, (C.c_double * 3)(*v))
        else:
            setattr(p, k, v)
    return p


def lib_path() -> str:
    """The in-tree library (the only one this binding loads)."""
    return os.path.join(HERE, "libcuharm.so")


def lib():
    """Load libcuharm.so (built in-tree by `python -m paper_2205_02484_b200.build`).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise CuharmError(f"{path} is missing: build it with `python -m paper_2205_02484_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
        L.cuharm_grid_init.argtypes = [C.POINTER(vp), C.POINTER(CuharmParams), vp]
        L.cuharm_workspace_bytes.argtypes = [vp]
        L.cuharm_workspace_bytes.restype = C.c_size_t
        L.cuharm_bind.argtypes = [vp, dp, vp, C.c_size_t]
        L.cuharm_metric_precompute.argtypes = [vp]
        L.cuharm_step.argtypes = [vp, C.c_double]
        L.cuharm_step_cfl.argtypes = [vp, C.c_double, C.c_double]
        L.cuharm_set_dt.argtypes = [vp, C.c_double]
        L.cuharm_substep.argtypes = [vp, C.c_int32]
        L.cuharm_substep_update.argtypes = [vp, C.c_int32]
        L.cuharm_repair_pass.argtypes = [vp, C.c_int32, C.c_int32, C.POINTER(C.c_int64)]
        L.cuharm_substep_finish.argtypes = [vp, C.c_int32]
        L.cuharm_flag_offset.argtypes = [vp]
        L.cuharm_flag_offset.restype = C.c_size_t
        L.cuharm_half_offset.argtypes = [vp]
        L.cuharm_half_offset.restype = C.c_size_t
        L.cuharm_last_cw.argtypes = [vp, C.POINTER(C.c_double)]
        L.cuharm_cfl_cw.argtypes = [vp, C.POINTER(C.c_double)]
        L.cuharm_dt_of_cw.argtypes = [vp, C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.cuharm_get_time.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.cuharm_apply_floors.argtypes = [vp, dp, ip]
        L.cuharm_repair.argtypes = [vp, dp, ip]
        L.cuharm_cons_to_prim.argtypes = [vp, dp, dp, ip]
        L.cuharm_prim_to_cons.argtypes = [vp, dp, dp]
        L.cuharm_invert_fallback.argtypes = [vp, C.c_int32, dp, dp, dp, ip]
        L.cuharm_cfl_dt.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
        L.cuharm_last_cfl_dt.argtypes = [vp, C.c_double, C.POINTER(C.c_double)]
        L.cuharm_divb.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.cuharm_divb_noalloc.argtypes = [dp, dp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double),
                                          C.c_int32, vp, dp]
        L.cuharm_divb_noalloc_errtext.argtypes = []
        L.cuharm_divb_noalloc_errtext.restype = C.c_char_p
        L.cuharm_shell_fluxes.argtypes = [vp, C.c_int32, C.POINTER(C.c_double)]
        L.cuharm_get_geom.argtypes = [vp, C.c_int32, dp]
        L.cuharm_apply_bc.argtypes = [vp, dp]
        L.cuharm_flux_dir.argtypes = [vp, dp, C.c_int32, dp, dp]
        L.cuharm_get_stats.argtypes = [vp, C.POINTER(C.c_int64)]
        L.cuharm_get_chain_stats.argtypes = [vp, C.POINTER(C.c_int64)]
        L.cuharm_use_graph.argtypes = [vp, C.c_int32]
        L.cuharm_launch_count.argtypes = [vp]
        L.cuharm_launch_count.restype = C.c_int64
        L.cuharm_set_timing.argtypes = [vp, C.c_int32]
        L.cuharm_get_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.cuharm_destroy.argtypes = [vp]
        L.cuharm_strerror.argtypes = [C.c_int]
        L.cuharm_strerror.restype = C.c_char_p
        _lib = L
    return _lib


def cuharm_strerror(code: int) -> str:
    return lib().cuharm_strerror(int(code)).decode()


def _check(rc: int, what: str):
    if rc != 0:
        raise CuharmError(f"{what} failed ({rc}): {cuharm_strerror(rc)}")


def _dptr(t):
    """Device pointer of a contiguous torch CUDA tensor (None -> NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise CuharmError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


# ---- the calls of include/cuharm.h, same names, torch tensors for device memory ----
def cuharm_grid_init(params: dict, stream=None):
    h = C.c_void_p()
    p = make_params(params)
    s = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    _check(lib().cuharm_grid_init(C.byref(h), C.byref(p), s), "cuharm_grid_init")
    return h


def cuharm_workspace_bytes(h) -> int:
    return int(lib().cuharm_workspace_bytes(h))


def cuharm_bind(h, prim, workspace):
    _check(lib().cuharm_bind(h, _dptr(prim), _dptr(workspace), workspace.numel() * workspace.element_size()), "cuharm_bind")


def cuharm_metric_precompute(h):
    _check(lib().cuharm_metric_precompute(h), "cuharm_metric_precompute")


def cuharm_step(h, dt: float):
    _check(lib().cuharm_step(h, float(dt)), "cuharm_step")


def cuharm_step_cfl(h, xi: float, dt_max: float = 0.0):
    _check(lib().cuharm_step_cfl(h, float(xi), float(dt_max)), "cuharm_step_cfl")


def cuharm_get_time(h):
    """(integrated time since bind, size of the last step)."""
    t, dt = C.c_double(), C.c_double()
    _check(lib().cuharm_get_time(h, C.byref(t), C.byref(dt)), "cuharm_get_time")
    return t.value, dt.value


def cuharm_apply_floors(h, prim, mask=None):
    _check(lib().cuharm_apply_floors(h, _dptr(prim), _dptr(mask)), "cuharm_apply_floors")


def cuharm_cons_to_prim(h, U, prim_inout, flag=None):
    _check(lib().cuharm_cons_to_prim(h, _dptr(U), _dptr(prim_inout), _dptr(flag)), "cuharm_cons_to_prim")


def cuharm_repair(h, prim, flag):
    _check(lib().cuharm_repair(h, _dptr(prim), _dptr(flag)), "cuharm_repair")


def cuharm_invert_fallback(h, method: int, U, US, prim_inout, flag=None):
    _check(lib().cuharm_invert_fallback(h, int(method), _dptr(U), _dptr(US), _dptr(prim_inout), _dptr(flag)),
           "cuharm_invert_fallback")


def cuharm_prim_to_cons(h, prim, U):
    _check(lib().cuharm_prim_to_cons(h, _dptr(prim), _dptr(U)), "cuharm_prim_to_cons")


def cuharm_cfl_dt(h, xi: float) -> float:
    dt = C.c_double()
    _check(lib().cuharm_cfl_dt(h, float(xi), C.byref(dt)), "cuharm_cfl_dt")
    return dt.value


def cuharm_last_cfl_dt(h, xi: float) -> float:
    dt = C.c_double()
    _check(lib().cuharm_last_cfl_dt(h, float(xi), C.byref(dt)), "cuharm_last_cfl_dt")
    return dt.value


def cuharm_shell_fluxes(h, i):
    """(Mdot, phi_B, Ldot, Edot) through the shell of zone centres of radial index i (eqs. 43-46)."""
    out = (C.c_double * 4)()
    _check(lib().cuharm_shell_fluxes(h, C.c_int32(i), out), "cuharm_shell_fluxes")
    return tuple(out)


def cuharm_divb(h):
    a, n = C.c_double(), C.c_double()
    _check(lib().cuharm_divb(h, C.byref(a), C.byref(n)), "cuharm_divb")
    return a.value, n.value


def cuharm_divb_noalloc(prim, sqrtg, n1, n2, n3, ng, dx, periodic_x3, out, stream=None):
    """Eq. 23 maxima without a context, a workspace or any allocation (include/cuharm.h): for code that sits inside
    another program's time loop and may not touch the device allocator.  `prim`, `sqrtg` ([n1g, n2g]) and `out` (2
    doubles) are CUDA tensors of the current device; the result lands in `out` asynchronously on `stream`.  The scratch
    is one static array per device shared by all calls: do not let two calls overlap on the GPU; grids with more than
    CUHARM_DIVB_NOALLOC_MAX_ROWS corner rows are refused."""
    arr = (C.c_double * 3)(*[float(x) for x in dx])
    s = C.c_void_p(stream.cuda_stream if stream is not None else 0)
    rc = lib().cuharm_divb_noalloc(_dptr(prim), _dptr(sqrtg), int(n1), int(n2), int(n3), int(ng), arr,
                                   1 if periodic_x3 else 0, s, _dptr(out))
    if rc != 0:
        raise CuharmError(f"cuharm_divb_noalloc failed ({rc}): {lib().cuharm_divb_noalloc_errtext().decode()}")


def cuharm_get_geom(h, loc: int, out):
    _check(lib().cuharm_get_geom(h, int(loc), _dptr(out)), "cuharm_get_geom")


def cuharm_apply_bc(h, prim):
    _check(lib().cuharm_apply_bc(h, _dptr(prim)), "cuharm_apply_bc")


def cuharm_flux_dir(h, prim, direction: int, F, cw=None):
    _check(lib().cuharm_flux_dir(h, _dptr(prim), int(direction), _dptr(F), _dptr(cw)), "cuharm_flux_dir")


def cuharm_get_stats(h):
    out = (C.c_int64 * 8)()
    _check(lib().cuharm_get_stats(h, out), "cuharm_get_stats")
    return list(out)


def cuharm_set_dt(h, dt: float):
    _check(lib().cuharm_set_dt(h, float(dt)), "cuharm_set_dt")


def cuharm_substep(h, which: int):
    _check(lib().cuharm_substep(h, int(which)), "cuharm_substep")


def cuharm_substep_update(h, which: int):
    _check(lib().cuharm_substep_update(h, int(which)), "cuharm_substep_update")


def cuharm_repair_pass(h, which: int, npass: int):
    out = (C.c_int64 * 2)()
    _check(lib().cuharm_repair_pass(h, int(which), int(npass), out), "cuharm_repair_pass")
    return int(out[0]), int(out[1])


def cuharm_substep_finish(h, which: int):
    _check(lib().cuharm_substep_finish(h, int(which)), "cuharm_substep_finish")


def cuharm_flag_offset(h) -> int:
    return int(lib().cuharm_flag_offset(h))


def cuharm_half_offset(h) -> int:
    return int(lib().cuharm_half_offset(h))


def cuharm_last_cw(h):
    out = (C.c_double * 3)()
    _check(lib().cuharm_last_cw(h, out), "cuharm_last_cw")
    return list(out)


def cuharm_cfl_cw(h):
    out = (C.c_double * 3)()
    _check(lib().cuharm_cfl_cw(h, out), "cuharm_cfl_cw")
    return list(out)


def cuharm_dt_of_cw(h, xi: float, cw) -> float:
    arr = (C.c_double * 3)(*[float(x) for x in cw])
    dt = C.c_double()
    _check(lib().cuharm_dt_of_cw(h, float(xi), arr, C.byref(dt)), "cuharm_dt_of_cw")
    return dt.value


def cuharm_get_chain_stats(h):
    out = (C.c_int64 * 4)()
    _check(lib().cuharm_get_chain_stats(h, out), "cuharm_get_chain_stats")
    return list(out)


def cuharm_use_graph(h, on: bool):
    _check(lib().cuharm_use_graph(h, 1 if on else 0), "cuharm_use_graph")


def cuharm_launch_count(h) -> int:
    return int(lib().cuharm_launch_count(h))


KERNEL_CLASSES = ("flux1", "flux2", "flux3", "emf", "update", "bc", "fixup")


def cuharm_set_timing(h, on: bool):
    _check(lib().cuharm_set_timing(h, 1 if on else 0), "cuharm_set_timing")


def cuharm_get_timing(h) -> dict:
    ms = (C.c_double * 8)()
    n = (C.c_int64 * 8)()
    _check(lib().cuharm_get_timing(h, ms, n), "cuharm_get_timing")
    return {k: (ms[i], n[i]) for i, k in enumerate(KERNEL_CLASSES)}


def cuharm_destroy(h):
    if h:
        lib().cuharm_destroy(h)


class Solver:
    """Owns the torch tensors the library borrows and forwards to the C calls.

        s = Solver(params, prim_host_or_device)   # grid_init + bind + metric_precompute
        dt = s.cfl_dt(0.45); s.step(dt); s.prim   # torch.float64 CUDA tensor [8, n1g, n2g, n3g]
    """

    def __init__(self, params: dict, prim, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise CuharmError("no CUDA device: libcuharm has no CPU path")
        self.params = dict(params)
        ng = params["ng"]
        self.shape = (8, params["n1"] + 2 * ng, params["n2"] + 2 * ng, params["n3"] + 2 * ng)
        self.device = torch.device(device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        with torch.cuda.device(self.device):
            self.h = cuharm_grid_init(params, self.stream)
            self.prim = torch.as_tensor(prim, dtype=torch.float64).to(self.device).contiguous().clone()
            if tuple(self.prim.shape) != self.shape:
                raise CuharmError(f"prim has shape {tuple(self.prim.shape)}, expected {self.shape}")
            self.workspace = torch.empty(cuharm_workspace_bytes(self.h), dtype=torch.uint8, device=self.device)
            cuharm_bind(self.h, self.prim, self.workspace)
            cuharm_metric_precompute(self.h)

    def load(self, prim):
        """Replace the primitives (host or device array of the bound shape) and refill the ghost zones."""
        import torch
        self.prim.copy_(torch.as_tensor(prim, dtype=torch.float64), non_blocking=True)
        cuharm_bind(self.h, self.prim, self.workspace)

    def step(self, dt): cuharm_step(self.h, dt)
    def step_cfl(self, xi, dt_max=0.0): cuharm_step_cfl(self.h, xi, dt_max)
    def time(self): return cuharm_get_time(self.h)
    def cfl_dt(self, xi): return cuharm_cfl_dt(self.h, xi)
    def last_cfl_dt(self, xi): return cuharm_last_cfl_dt(self.h, xi)
    def divb(self): return cuharm_divb(self.h)
    def shell_fluxes(self, i): return cuharm_shell_fluxes(self.h, i)
    def stats(self): return cuharm_get_stats(self.h)
    def chain_stats(self): return cuharm_get_chain_stats(self.h)
    # split step and face-speed maxima (slab decomposition, paper_2205_02484_b200/slab.py)
    def set_dt(self, dt): cuharm_set_dt(self.h, dt)
    def substep(self, which): cuharm_substep(self.h, which)
    def substep_update(self, which): cuharm_substep_update(self.h, which)
    def repair_pass(self, which, npass): return cuharm_repair_pass(self.h, which, npass)
    def substep_finish(self, which): cuharm_substep_finish(self.h, which)
    def work(self, which): return self.half if which == 0 else self.prim   # the array substep `which` produces
    def end_step(self): pass

    @property
    def max_passes(self): return int(self.params["fixup_max_passes"])

    @property
    def flags(self):
        """The fail flags of the last substep (a view of the workspace; int32 [n1g, n2g, n3g])."""
        import torch
        off, n = cuharm_flag_offset(self.h), self.shape[1] * self.shape[2] * self.shape[3] * 4
        return self.workspace[off:off + n].view(torch.int32).view(self.shape[1:])
    def last_cw(self): return cuharm_last_cw(self.h)
    def cfl_cw(self): return cuharm_cfl_cw(self.h)
    def dt_of_cw(self, xi, cw): return cuharm_dt_of_cw(self.h, xi, cw)

    @property
    def half(self):
        """The half-step primitives (a view of the workspace; layout of `prim`)."""
        import torch
        off, n = cuharm_half_offset(self.h), 8 * self.shape[1] * self.shape[2] * self.shape[3] * 8
        return self.workspace[off:off + n].view(torch.float64).view(self.shape)
    def repair(self, prim, flag): cuharm_repair(self.h, prim, flag)
    def use_graph(self, on=True): cuharm_use_graph(self.h, on)
    def launch_count(self): return cuharm_launch_count(self.h)
    def set_timing(self, on=True): cuharm_set_timing(self.h, on)
    def get_timing(self): return cuharm_get_timing(self.h)

    def geom(self, loc):
        import torch
        out = torch.empty((40 if loc == 3 else 22, self.shape[1], self.shape[2]), dtype=torch.float64, device=self.device)
        cuharm_get_geom(self.h, loc, out)
        return out

    def prim_to_cons(self, prim=None):
        import torch
        prim = self.prim if prim is None else prim
        U = torch.empty_like(prim)
        cuharm_prim_to_cons(self.h, prim, U)
        return U

    def cons_to_prim(self, U, guess):
        import torch
        out = guess.clone()
        flag = torch.zeros(self.shape[1:], dtype=torch.int32, device=self.device)
        cuharm_cons_to_prim(self.h, U, out, flag)
        return out, flag

    def invert_fallback(self, method, U, guess, US=None):
        import torch
        out = guess.clone()
        flag = torch.zeros(self.shape[1:], dtype=torch.int32, device=self.device)
        cuharm_invert_fallback(self.h, method, U, US, out, flag)
        return out, flag

    def flux_dir(self, prim, direction):
        import torch
        F = torch.empty_like(prim)
        cw = torch.empty(self.shape[1:], dtype=torch.float64, device=self.device)
        cuharm_flux_dir(self.h, prim, direction, F, cw)
        return F, cw

    def apply_bc(self, prim): cuharm_apply_bc(self.h, prim)

    def apply_floors(self, prim):
        import torch
        mask = torch.zeros(self.shape[1:], dtype=torch.int32, device=self.device)
        cuharm_apply_floors(self.h, prim, mask)
        return mask

    def close(self):
        if getattr(self, "h", None):
            import torch
            torch.cuda.synchronize(self.device)
            cuharm_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
