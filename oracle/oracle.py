"""ctypes binding of the fp64 CPU oracle (oracle/hhrr_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py.  The product package
(paper_2510_13726_b200) never imports this module and this module never imports
the product package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "hhrr_oracle.c"
_LIB = _HERE / "libhhrr_oracle.so"
# the same oracle on the paper's own velocity set: a second translation unit, a second library
_SRC19 = _HERE / "hhrr_oracle_q19.c"
_LIB19 = _HERE / "libhhrr_oracle_q19.so"

Q = 27
MAX_TAGS = 16
T_FLUID, T_GROWTH, T_FRONTIER, T_SOLID, T_FRINGE = 0, 1, 2, 3, 4
PERIODIC, MIRROR = 0, 1


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc.  -ffp-contract=off: the geometry classification
    is defined by its operation order (bit-exact cell types)."""
    for src, out in ((_SRC, _LIB), (_SRC19, _LIB19)):
        newest = max(_SRC.stat().st_mtime, src.stat().st_mtime)
        if force or not out.exists() or out.stat().st_mtime < newest:
            cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
                   "-shared", "-fPIC", "-o", str(out), str(src), "-lm"]
            subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("mode", C.c_int32 * 3),
                ("tau0", C.c_double), ("sigma", C.c_double), ("smagorinsky_cs", C.c_double),
                ("body_force", C.c_double * 3),
                ("eps_cells", C.c_double),
                ("kappa", C.c_double), ("E", C.c_double),
                ("newton_max_iter", C.c_int32), ("newton_tol", C.c_double),
                ("sampling_distance", C.c_double)]


class RotorDesc(C.Structure):
    _fields_ = [("sdf", C.c_void_p), ("tag", C.c_void_p),
                ("gx", C.c_int32), ("gy", C.c_int32), ("gz", C.c_int32),
                ("spacing", C.c_double), ("origin", C.c_double * 3),
                ("centre", C.c_double * 3), ("axis", C.c_double * 3),
                ("omega", C.c_double), ("theta0", C.c_double), ("n_tags", C.c_int32)]


_libs = {}


def lib(q=27):
    if q not in _libs:
        build()
        _libs[q] = C.CDLL(str({27: _LIB, 19: _LIB19}[q]))
        L = _libs[q]
        assert L.ohrr_q() == q
        L.ohrr_create.restype = C.c_void_p
        L.ohrr_create.argtypes = [C.POINTER(Params)]
        L.ohrr_destroy.argtypes = [C.c_void_p]
        L.ohrr_rotor_coefficients.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_double,
                                              C.c_void_p, C.c_void_p]
        L.ohrr_spalding_f.restype = C.c_double
        L.ohrr_spalding_f.argtypes = [C.c_double] * 6
        L.ohrr_newton_utau.restype = C.c_double
        L.ohrr_newton_utau.argtypes = [C.c_double] * 6 + [C.c_int, C.c_double, C.POINTER(C.c_int32)]
        L.ohrr_musker_uplus.restype = C.c_double
        L.ohrr_musker_uplus.argtypes = [C.c_double]
        L.ohrr_musker_f.restype = C.c_double
        L.ohrr_musker_f.argtypes = [C.c_double] * 4
        L.ohrr_newton_utau_musker.restype = C.c_double
        L.ohrr_newton_utau_musker.argtypes = [C.c_double] * 4 + [C.c_int, C.c_double, C.POINTER(C.c_int32)]
        L.ohrr_spalding_uplus.restype = C.c_double
        L.ohrr_spalding_uplus.argtypes = [C.c_double] * 3
        L.ohrr_wall_uplus.restype = C.c_double
        L.ohrr_wall_uplus.argtypes = [C.c_int] + [C.c_double] * 3
        L.ohrr_wall_shear.restype = C.c_double
        L.ohrr_wall_shear.argtypes = [C.c_int] + [C.c_double] * 6
        L.ohrr_tau_eff.restype = C.c_double
        L.ohrr_tau_eff.argtypes = [C.c_double, C.c_double, C.c_double, C.c_void_p]
        L.ohrr_get_wall_list.restype = C.c_int64
        L.ohrr_step_count.restype = C.c_int64
        L.ohrr_step_count.argtypes = [C.c_void_p]
    return _libs[q]


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def make_params(nx, ny, nz, mode=(0, 0, 0), tau0=0.55, sigma=0.995, smagorinsky_cs=0.1,
                body_force=(0.0, 0.0, 0.0), eps_cells=2.0, kappa=0.41, E=9.8,
                newton_max_iter=10, newton_tol=1e-4, sampling_distance=2.0) -> Params:
    p = Params()
    p.nx, p.ny, p.nz = nx, ny, nz
    p.mode[:] = list(mode)
    p.tau0, p.sigma, p.smagorinsky_cs = tau0, sigma, smagorinsky_cs
    p.body_force[:] = list(body_force)
    p.eps_cells = eps_cells
    p.kappa, p.E = kappa, E
    p.newton_max_iter, p.newton_tol = newton_max_iter, newton_tol
    p.sampling_distance = sampling_distance
    return p


# ---- free functions (cell-model pieces, used by the pins) ---------------------------------
def lattice_tables(q=27):
    cx = np.zeros(q, np.int32); cy = np.zeros(q, np.int32); cz = np.zeros(q, np.int32)
    w = np.zeros(q, np.float64)
    lib(q).ohrr_lattice_tables(_p(cx), _p(cy), _p(cz), _p(w))
    return cx, cy, cz, w


def equilibrium(rho, u, q=27):
    u = _f64(u); out = np.zeros(q)
    lib(q).ohrr_equilibrium(C.c_double(rho), _p(u), _p(out))
    return out


def collide_cell(fin, g, d, uB, S, sigma, tau0, cs, q=27):
    fin = _f64(fin); g = _f64(g); uB = _f64(uB); S = _f64(S)
    out = np.zeros(q); diag = np.zeros(5)
    lib(q).ohrr_collide_cell(_p(fin), _p(g), C.c_double(d), _p(uB), _p(S), C.c_double(sigma),
                            C.c_double(tau0), C.c_double(cs), _p(out), _p(diag))
    return out, diag


def tau_eff(tau0, cs, rho, pi):
    pi = _f64(pi)
    return lib().ohrr_tau_eff(tau0, cs, rho, _p(pi))


def spalding_f(utau, U, y, nu, kappa=0.41, E=9.8):
    return lib().ohrr_spalding_f(utau, U, y, nu, kappa, E)


def spalding_uplus(yp, kappa=0.41, E=9.8):
    return lib().ohrr_spalding_uplus(float(yp), float(kappa), float(E))


def wall_uplus(kind, yp, kappa=0.41, E=9.8):
    return lib().ohrr_wall_uplus(int(kind), float(yp), float(kappa), float(E))


def wall_shear(kind, utau, U, y, nu, kappa=0.41, E=9.8):
    return lib().ohrr_wall_shear(int(kind), float(utau), float(U), float(y), float(nu), float(kappa), float(E))


def musker_uplus(yp):
    return lib().ohrr_musker_uplus(float(yp))


def musker_f(utau, U, y, nu):
    return lib().ohrr_musker_f(float(utau), float(U), float(y), float(nu))


def newton_utau_musker(u0, U, y, nu, max_iter=10, tol=1e-4):
    it = C.c_int32(0)
    u = lib().ohrr_newton_utau_musker(float(u0), float(U), float(y), float(nu), int(max_iter), float(tol), C.byref(it))
    return u, it.value


def newton_utau(u0, U, y, nu, kappa=0.41, E=9.8, max_iter=10, tol=1e-4):
    it = C.c_int32(0)
    r = lib().ohrr_newton_utau(u0, U, y, nu, kappa, E, max_iter, tol, C.byref(it))
    return r, it.value


# ---- lattice object -------------------------------------------------------------------------
class Lattice:
    def __init__(self, params: Params, q=27):
        self.p = params
        self.q = q
        self.lib = lib(q)
        self.nx, self.ny, self.nz = params.nx, params.ny, params.nz
        self.n = self.nx * self.ny * self.nz
        self.h = self.lib.ohrr_create(C.byref(params))
        if not self.h:
            raise RuntimeError("ohrr_create failed")
        self._keep = []

    def close(self):
        if self.h:
            self.lib.ohrr_destroy(C.c_void_p(self.h))
            self.h = None

    def __del__(self):
        self.close()

    @property
    def _h(self):
        return C.c_void_p(self.h)

    def init_equilibrium(self, rho, u, with_neq=False):
        rho = _f64(rho).ravel(); u = _f64(u).reshape(3, -1)
        assert rho.size == self.n and u.shape[1] == self.n
        self.lib.ohrr_init_equilibrium(self._h, _p(rho), _p(u), int(with_neq))

    def set_static_geometry(self, phi, tag=None, d_override=None):
        phi = _f64(phi).ravel()
        tag = None if tag is None else np.ascontiguousarray(tag, np.uint8).ravel()
        dov = None if d_override is None else _f64(d_override).ravel()
        self.lib.ohrr_set_static_geometry(self._h, _p(phi), _p(tag), _p(dov))

    def set_body(self, tag, centre=(0, 0, 0), omega=(0, 0, 0), vel=(0, 0, 0)):
        c = _f64(centre); o = _f64(omega); v = _f64(vel)
        self.lib.ohrr_set_body(self._h, int(tag), _p(c), _p(o), _p(v))

    def set_fringe(self, x0, x1, u_in):
        u = _f64(u_in)
        self.lib.ohrr_set_fringe(self._h, int(x0), int(x1), _p(u))

    def set_rotor(self, sdf, tag, spacing, origin, centre, axis, omega, theta0, n_tags):
        sdf = np.ascontiguousarray(sdf, np.float32); tag = np.ascontiguousarray(tag, np.uint8)
        gz, gy, gx = sdf.shape
        r = RotorDesc()
        r.sdf = sdf.ctypes.data; r.tag = tag.ctypes.data
        r.gx, r.gy, r.gz = gx, gy, gz
        r.spacing = spacing
        r.origin[:] = list(origin); r.centre[:] = list(centre); r.axis[:] = list(axis)
        r.omega, r.theta0, r.n_tags = omega, theta0, n_tags
        rc = self.lib.ohrr_set_rotor(self._h, C.byref(r))
        if rc:
            raise RuntimeError("ohrr_set_rotor failed")

    def enable_wall_model(self, enable=True):
        self.lib.ohrr_enable_wall_model(self._h, int(enable))

    def set_fsi_region(self, boxes):
        """boxes: iterable of (x0, x1, y0, y1, z0, z1), half-open; empty = HHRRLBM everywhere."""
        b = np.ascontiguousarray(np.asarray(list(boxes), np.int32).reshape(-1, 6))
        rc = self.lib.ohrr_set_fsi_region(self._h, int(b.shape[0]), _p(b) if b.size else None)
        if rc:
            raise RuntimeError("ohrr_set_fsi_region failed")

    def set_wall_model_variant(self, slip=0, shear=0):
        if self.lib.ohrr_set_wall_model_variant(self._h, int(slip), int(shear)):
            raise RuntimeError("ohrr_set_wall_model_variant failed")

    def set_wall_function(self, kind):
        if self.lib.ohrr_set_wall_function(self._h, int(kind)):
            raise RuntimeError("ohrr_set_wall_function failed")

    def region_violation(self):
        return bool(self.lib.ohrr_region_violation(self._h))

    def update_geometry(self):
        self.lib.ohrr_update_geometry(self._h)

    def wall_model_only(self):
        self.lib.ohrr_wall_model_only(self._h)

    def force_only(self):
        F = np.zeros((MAX_TAGS, 3))
        self.lib.ohrr_force_only(self._h, _p(F))
        return F

    def torque_only(self):
        M = np.zeros((MAX_TAGS, 3))
        self.lib.ohrr_torque_only(self._h, _p(M))
        return M

    def step(self, n=1):
        self.lib.ohrr_step(self._h, int(n))

    def moments(self):
        rho = np.zeros(self.n); v = np.zeros((3, self.n))
        self.lib.ohrr_get_moments(self._h, _p(rho), _p(v))
        return rho, v

    def forces(self, first=0, count=None):
        if count is None:
            count = self.lib.ohrr_step_count(self._h) - first
        F = np.zeros((count, MAX_TAGS, 3))
        rc = self.lib.ohrr_get_forces(self._h, C.c_int64(first), C.c_int64(count), _p(F))
        if rc:
            raise RuntimeError("ohrr_get_forces: range")
        return F

    def torques(self, first=0, count=None):
        if count is None:
            count = self.lib.ohrr_step_count(self._h) - first
        M = np.zeros((count, MAX_TAGS, 3))
        rc = self.lib.ohrr_get_torques(self._h, C.c_int64(first), C.c_int64(count), _p(M))
        if rc:
            raise RuntimeError("ohrr_get_torques: range")
        return M

    def rotor_coefficients(self, rho, u_inf, radius, first=0, count=None):
        """(C_T, C_P) per step: Definition 3 / Eq. 26 and the power coefficient of the same rotor."""
        if count is None:
            count = self.lib.ohrr_step_count(self._h) - first
        ct = np.zeros(count); cp = np.zeros(count)
        rc = self.lib.ohrr_rotor_coefficients(self._h, first, count, rho, u_inf, radius, _p(ct), _p(cp))
        if rc:
            raise RuntimeError("ohrr_rotor_coefficients: no rotor, bad range or bad argument")
        return ct, cp

    def cell_types(self):
        t = np.zeros(self.n, np.uint8); g = np.zeros(self.n, np.uint8); d = np.zeros(self.n)
        self.lib.ohrr_get_cell_types(self._h, _p(t), _p(g), _p(d))
        return t, g, d

    def wall_list(self):
        k = self.lib.ohrr_get_wall_list(self._h, None, None, None, None, C.c_int64(0))
        idx = np.zeros(k, np.int32); y1n = np.zeros((k, 3)); ut = np.zeros(k); va = np.zeros(k, np.uint8)
        if k:
            self.lib.ohrr_get_wall_list(self._h, _p(idx), _p(y1n), _p(ut), _p(va), C.c_int64(k))
        return idx, y1n, ut, va

    def wall_state(self, cell):
        ut = C.c_double(0); u = np.zeros(3); s = np.zeros(6)
        valid = self.lib.ohrr_get_wall_state(self._h, C.c_int64(cell), C.byref(ut), _p(u), _p(s))
        return valid, ut.value, u, s

    def populations(self):
        f = np.zeros((self.q, self.n))
        self.lib.ohrr_get_populations(self._h, _p(f))
        return f

    def set_populations(self, f):
        f = _f64(f).reshape(self.q, self.n)
        self.lib.ohrr_set_populations(self._h, _p(f))

    def uhat(self):
        u = np.zeros((3, self.n))
        self.lib.ohrr_get_uhat(self._h, _p(u))
        return u


class View:
    """The oracle on one velocity set with the module's own names: view(19).Lattice(p), .equilibrium(rho, u), ..."""

    def __init__(self, q):
        self.Q = self.q = q

    def __getattr__(self, name):
        import functools
        obj = globals()[name]
        if name in ("lattice_tables", "equilibrium", "collide_cell", "Lattice"):
            return functools.partial(obj, q=self.q)
        return obj


def view(q):
    return View(q)


def threads() -> int:
    return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
