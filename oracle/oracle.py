"""ctypes wrapper of liboracle.so (host numpy arrays in, numpy arrays out).

TEST INFRASTRUCTURE ONLY — see the header of oracle.cpp.  Argument marshalling only; all arithmetic
is in oracle.cpp.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class OracleParams(C.Structure):
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


def make_params(d: dict) -> OracleParams:
    p = OracleParams()
    p.struct_bytes = C.sizeof(OracleParams)
    for k, v in d.items():
        if k in ("xmin", "xmax"):
            setattr(p, k, (C.c_double * 3)(*v))
        else:
            setattr(p, k, v)
    return p


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def _d(a):
    return a.ctypes.data_as(_dp)


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        L = _lib
        L.oracle_slope_mc.restype = C.c_double
        L.oracle_slope_mc.argtypes = [C.c_double] * 3
        L.oracle_get_threads.restype = C.c_int
        L.oracle_entropy_cons.restype = C.c_double
    return _lib


def _arr(x, n=None):
    a = np.ascontiguousarray(x, dtype=np.float64)
    if n is not None:
        assert a.size == n, (a.shape, n)
    return a


# ------------------------------------------------------------------ point-level functions
def coord_map(params: dict, X1, X2):
    out = np.zeros(5)
    lib().oracle_coord_map(C.byref(make_params(params)), C.c_double(X1), C.c_double(X2), _d(out))
    return dict(r=out[0], th=out[1], drdX=out[2], dthdY=out[3], d2thdY2=out[4])


def radial_map(params: dict, X1):
    """r, dr/dX, d2r/dX2 of eq. 39's radial map at X1, and X_out = the X of r_out."""
    out = np.zeros(4)
    lib().oracle_radial_map(C.byref(make_params(params)), C.c_double(X1), _d(out))
    return dict(r=out[0], d1=out[1], d2=out[2], X_out=out[3])


def metric_at(params: dict, X1, X2, polar_face=0):
    gcov = np.zeros((4, 4)); gcon = np.zeros((4, 4))
    sg = C.c_double(); al = C.c_double()
    lib().oracle_metric_at(C.byref(make_params(params)), C.c_double(X1), C.c_double(X2), int(polar_face),
                           _d(gcov), _d(gcon), C.byref(sg), C.byref(al))
    return gcov, gcon, sg.value, al.value


def conn_at(params: dict, X1, X2):
    conn = np.zeros((4, 4, 4))
    lib().oracle_conn_at(C.byref(make_params(params)), C.c_double(X1), C.c_double(X2), _d(conn))
    return conn


def fluid_state(prim, gcov, gcon):
    prim = _arr(prim, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    ucon = np.zeros(4); ucov = np.zeros(4); bcon = np.zeros(4); bcov = np.zeros(4)
    bsq = C.c_double()
    lib().oracle_fluid_state(_d(prim), _d(gcov), _d(gcon), _d(ucon), _d(ucov), _d(bcon), _d(bcov), C.byref(bsq))
    return dict(ucon=ucon, ucov=ucov, bcon=bcon, bcov=bcov, bsq=bsq.value)


def flux_vector(prim, gcov, gcon, sqrtg, gam, direction):
    prim = _arr(prim, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    out = np.zeros(8)
    lib().oracle_flux_vector(_d(prim), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam), int(direction), _d(out))
    return out


def wave_speeds(prim, gcov, gcon, gam, direction):
    prim = _arr(prim, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    c1 = C.c_double(); c2 = C.c_double()
    lib().oracle_wave_speeds(_d(prim), _d(gcov), _d(gcon), C.c_double(gam), int(direction), C.byref(c1), C.byref(c2))
    return c1.value, c2.value


def slope_mc(qm, q0, qp):
    return lib().oracle_slope_mc(float(qm), float(q0), float(qp))


def recon_cell(recon, y5):
    y = _arr(y5, 5)
    l = C.c_double(); r = C.c_double()
    lib().oracle_recon_cell(int(recon), _d(y), C.byref(l), C.byref(r))
    return l.value, r.value


def face_flux(pl, pr, gcov, gcon, sqrtg, gam, direction, riemann):
    pl = _arr(pl, 8); pr = _arr(pr, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    F = np.zeros(8); cw = C.c_double()
    lib().oracle_face_flux(_d(pl), _d(pr), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam), int(direction),
                           int(riemann), _d(F), C.byref(cw))
    return F, cw.value


def source_term(prim, gcov, gcon, sqrtg, conn, gam):
    prim = _arr(prim, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16); conn = _arr(conn, 64)
    S = np.zeros(4)
    lib().oracle_source_term(_d(prim), _d(gcov), _d(gcon), C.c_double(sqrtg), _d(conn), C.c_double(gam), _d(S))
    return S


def invert_2d(U, gcov, gcon, sqrtg, gam, guess, tol=1e-10, maxit=30, extra=0):
    U = _arr(U, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    prim = np.array(guess, dtype=np.float64).copy()
    it = C.c_int()
    flag = lib().oracle_invert_2d(_d(U), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam), _d(prim),
                                  C.c_double(tol), int(maxit), int(extra), C.byref(it))
    return prim, flag, it.value


def invert_1dw(U, gcov, gcon, sqrtg, gam, guess, tol=1e-14, maxit=200):
    """(ii) of P:L204: the 1D method for W by Brent."""
    U = _arr(U, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    prim = np.array(guess, dtype=np.float64).copy()
    flag = lib().oracle_invert_1dw(_d(U), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam), _d(prim),
                                   C.c_double(tol), int(maxit))
    return prim, flag


def invert_entropy(U, US, gcov, gcon, sqrtg, gam, guess, tol=1e-14, maxit=200):
    """(iii) of P:L204: the entropy method (eq. 32 in eq. 29) by Brent.  US = sqrt(-g) S u^t."""
    U = _arr(U, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    prim = np.array(guess, dtype=np.float64).copy()
    flag = lib().oracle_invert_entropy(_d(U), C.c_double(US), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam),
                                       _d(prim), C.c_double(tol), int(maxit))
    return prim, flag


def entropy_cons(prim, gcov, gcon, sqrtg, gam):
    prim = _arr(prim, 8); gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    return lib().oracle_entropy_cons(_d(prim), _d(gcov), _d(gcon), C.c_double(sqrtg), C.c_double(gam))


def apply_floors(params: dict, r, gcov, gcon, sqrtg, prim):
    gcov = _arr(gcov, 16); gcon = _arr(gcon, 16)
    q = np.array(prim, dtype=np.float64).copy()
    mask = lib().oracle_apply_floors(C.byref(make_params(params)), C.c_double(r), _d(gcov), _d(gcon), C.c_double(sqrtg), _d(q))
    return q, mask


def set_threads(n: int):
    lib().oracle_set_threads(int(n))


def get_threads() -> int:
    return lib().oracle_get_threads()


# ------------------------------------------------------------------ grid-level object
class Grid:
    """Mirror of the library's handle-based calls, on host numpy arrays."""

    def __init__(self, params: dict):
        self.params = dict(params)
        self._p = make_params(params)
        self._h = C.c_void_p()
        rc = lib().oracle_grid_init(C.byref(self._h), C.byref(self._p))
        if rc != 0:
            raise ValueError(f"oracle_grid_init failed: {rc}")
        ng = self._p.ng
        self.shape = (self._p.n1 + 2 * ng, self._p.n2 + 2 * ng, self._p.n3 + 2 * ng)
        self.nz = int(np.prod(self.shape))
        self.prim = None

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def get_geom(self, loc):
        ncomp = 40 if loc == 3 else 22
        out = np.zeros((ncomp, self.shape[0], self.shape[1]))
        rc = lib().oracle_get_geom(self._h, int(loc), _d(out))
        assert rc == 0
        return out

    def bind(self, prim: np.ndarray):
        assert prim.dtype == np.float64 and prim.flags.c_contiguous and prim.shape == (8,) + self.shape
        self.prim = prim
        lib().oracle_bind(self._h, _d(prim))

    def apply_bc(self, prim: np.ndarray):
        assert prim.dtype == np.float64 and prim.flags.c_contiguous and prim.shape == (8,) + self.shape
        lib().oracle_apply_bc(self._h, _d(prim))

    # ---- slab decomposition: split step, half-step array, face-speed maxima
    def substep(self, which: int, dt: float):
        assert lib().oracle_substep(self._h, int(which), C.c_double(dt)) == 0

    def substep_update(self, which: int, dt: float):
        assert lib().oracle_substep_update(self._h, int(which), C.c_double(dt)) == 0

    def repair_pass(self, which: int, npass: int):
        out = np.zeros(2, dtype=np.int64)
        lib().oracle_repair_pass(self._h, int(which), int(npass), out.ctypes.data_as(C.POINTER(C.c_int64)))
        return int(out[0]), int(out[1])

    def substep_finish(self, which: int):
        lib().oracle_substep_finish(self._h, int(which))

    def commit(self):
        lib().oracle_commit(self._h)

    def new(self) -> np.ndarray:
        lib().oracle_new.restype = _dp
        return np.ctypeslib.as_array(lib().oracle_new(self._h), shape=(8,) + self.shape)

    def flags(self) -> np.ndarray:
        lib().oracle_flags.restype = _ip
        return np.ctypeslib.as_array(lib().oracle_flags(self._h), shape=self.shape)

    def half(self) -> np.ndarray:
        lib().oracle_half.restype = _dp
        ptr = lib().oracle_half(self._h)
        return np.ctypeslib.as_array(ptr, shape=(8,) + self.shape)

    def last_cw(self):
        out = np.zeros(3)
        lib().oracle_last_cw(self._h, _d(out))
        return out

    def cfl_cw(self):
        out = np.zeros(3)
        assert lib().oracle_cfl_cw(self._h, _d(out)) == 0
        return out

    def dt_of_cw(self, xi: float, cw) -> float:
        cw = np.ascontiguousarray(cw, dtype=np.float64)
        dt = C.c_double()
        lib().oracle_dt_of_cw(self._h, C.c_double(xi), _d(cw), C.byref(dt))
        return dt.value

    def polar_damp(self, prim: np.ndarray):
        """P:L311 (A16) as a stage: utilde^2 of the two zones nearest each pole interpolated to zero at the pole."""
        assert prim.dtype == np.float64 and prim.flags.c_contiguous and prim.shape == (8,) + self.shape
        lib().oracle_polar_damp(self._h, _d(prim))

    def step(self, dt: float):
        rc = lib().oracle_step(self._h, C.c_double(dt))
        assert rc == 0, rc

    def flux_dir(self, prim, direction):
        prim = _arr(prim, 8 * self.nz)
        F = np.zeros((8,) + self.shape); cw = np.zeros(self.shape); m = C.c_double()
        lib().oracle_flux_dir(self._h, _d(prim), int(direction), _d(F), _d(cw), C.byref(m))
        return F, cw, m.value

    def flux_ct(self, F1, F2, F3):
        F1 = _arr(F1).copy(); F2 = _arr(F2).copy(); F3 = _arr(F3).copy()
        E = np.zeros((3,) + self.shape)
        lib().oracle_flux_ct(self._h, _d(F1), _d(F2), _d(F3), _d(E))
        return F1, F2, F3, E

    def update_B_only(self, prim, F1, F2, F3, dtau):
        assert prim.dtype == np.float64 and prim.flags.c_contiguous
        F1 = _arr(F1); F2 = _arr(F2); F3 = _arr(F3)
        lib().oracle_update_B_only(self._h, _d(prim), _d(F1), _d(F2), _d(F3), C.c_double(dtau))

    def prim_to_cons(self, prim):
        prim = _arr(prim, 8 * self.nz)
        U = np.zeros((8,) + self.shape)
        lib().oracle_prim_to_cons(self._h, _d(prim), _d(U))
        return U

    def cons_to_prim(self, U, guess):
        U = _arr(U, 8 * self.nz)
        prim = np.array(guess, dtype=np.float64).copy()
        flag = np.zeros(self.shape, dtype=np.int32)
        lib().oracle_cons_to_prim(self._h, _d(U), _d(prim), flag.ctypes.data_as(_ip))
        return prim, flag

    def cfl_dt(self, xi: float) -> float:
        dt = C.c_double()
        rc = lib().oracle_cfl_dt(self._h, C.c_double(xi), C.byref(dt))
        assert rc == 0
        return dt.value

    def last_cfl_dt(self, xi: float) -> float:
        dt = C.c_double()
        lib().oracle_last_cfl_dt(self._h, C.c_double(xi), C.byref(dt))
        return dt.value

    def divb(self):
        a = C.c_double(); n = C.c_double()
        rc = lib().oracle_divb(self._h, C.byref(a), C.byref(n))
        assert rc == 0
        return a.value, n.value

    def shell_fluxes(self, i):
        """(Mdot, phi_B, Ldot, Edot) through the shell of zone centres of radial index i (eqs. 43-46)."""
        out = np.zeros(4)
        rc = lib().oracle_shell_fluxes(self._h, C.c_int32(i), out.ctypes.data_as(C.POINTER(C.c_double)))
        assert rc == 0, rc
        return out

    def get_stats(self):
        out = np.zeros(8, dtype=np.int64)
        lib().oracle_get_stats(self._h, out.ctypes.data_as(C.POINTER(C.c_int64)))
        return out

    def get_chain_stats(self):
        out = np.zeros(4, dtype=np.int64)
        lib().oracle_get_chain_stats(self._h, out.ctypes.data_as(C.POINTER(C.c_int64)))
        return out

    def entropy_flux_dir(self, prim, direction):
        prim = _arr(prim, 8 * self.nz)
        FS = np.zeros(self.shape)
        lib().oracle_entropy_flux_dir(self._h, _d(prim), int(direction), _d(FS))
        return FS

    def get_flags(self):
        out = np.zeros(self.shape, dtype=np.int32)
        lib().oracle_get_flags(self._h, out.ctypes.data_as(_ip))
        return out

    def apply_floors(self, prim):
        """C-12 on every interior zone of prim, in place; returns the per-zone bit mask."""
        assert prim.dtype == np.float64 and prim.flags.c_contiguous and prim.shape == (8,) + self.shape
        mask = np.zeros(self.shape, dtype=np.int32)
        lib().oracle_apply_floors_grid(self._h, _d(prim), mask.ctypes.data_as(_ip))
        return mask

    def fixup(self, prim, flag):
        assert prim.dtype == np.float64 and prim.flags.c_contiguous
        flag = np.ascontiguousarray(flag, dtype=np.int32)
        lib().oracle_fixup(self._h, _d(prim), flag.ctypes.data_as(_ip))
