"""Thin ctypes binding of libhhrr.so (include/hhrr.h).  Argument marshalling only: every step
of the path runs in the CUDA kernels behind the C ABI.  PyTorch is used for the device
workspace allocation and the CUDA stream, nothing else.

There is no CPU fallback: importing works without a GPU (so the symbol table can be
checked), but creating a Lattice without the built library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libhhrr.so"
LIB_PATHS = {27: LIB_PATH, 19: _HERE / "libhhrr_q19.so"}   # one library build per velocity set (HHRR_Q)

Q = 27
MAX_TAGS = 16
FLUID, GROWTH, FRONTIER, SOLID, FRINGE = 0, 1, 2, 3, 4
PERIODIC, MIRROR = 0, 1

# every symbol include/hhrr.h declares (tests check the library exports exactly these)
SYMBOLS = [
    "hhrr_workspace_bytes", "hhrr_create", "hhrr_destroy", "hhrr_init_equilibrium",
    "hhrr_set_static_geometry", "hhrr_set_body", "hhrr_set_fringe", "hhrr_set_rotor",
    "hhrr_enable_wall_model", "hhrr_update_geometry", "hhrr_step", "hhrr_step_count",
    "hhrr_get_moments", "hhrr_get_moments_device", "hhrr_get_forces", "hhrr_get_torques", "hhrr_get_rotor_coefficients", "hhrr_force_history",
    "hhrr_get_cell_types", "hhrr_get_wall_list", "hhrr_get_wall_state", "hhrr_get_populations",
    "hhrr_set_populations", "hhrr_get_cell_populations", "hhrr_get_uhat", "hhrr_check_finite", "hhrr_set_kernel_variant",
    "hhrr_population_storage", "hhrr_set_fsi_region", "hhrr_set_wall_function", "hhrr_set_wall_model_variant",
    "hhrr_get_wall_model_state", "hhrr_set_wall_model_state", "hhrr_set_step_count",
    "hhrr_set_timing", "hhrr_get_timing", "hhrr_set_lookahead", "hhrr_set_launch_shape", "hhrr_launch_count", "hhrr_last_error", "hhrr_version",
    "hhrr_velocity_set", "hhrr_halo_floats", "hhrr_halo_pack", "hhrr_halo_unpack", "hhrr_wall_model_noalloc",
]


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


class HhrrError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"hhrr error {code}: {msg}")
        self.code = code


_libs = {}


def lib(q=27):
    """Loads libhhrr.so (D3Q27) or libhhrr_q19.so (D3Q19); raises if it has not been built (no fallback)."""
    if q not in _libs:
        path = LIB_PATHS[q]
        if not path.exists():
            raise RuntimeError(f"{path} missing: run `python -m paper_2510_13726_b200.build` "
                               "(the CUDA library is the only implementation; there is no fallback)")
        L = C.CDLL(str(path))
        vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
        L.hhrr_workspace_bytes.restype = C.c_size_t
        L.hhrr_workspace_bytes.argtypes = [C.POINTER(Params), C.POINTER(RotorDesc)]
        L.hhrr_create.argtypes = [C.POINTER(Params), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.hhrr_destroy.argtypes = [vp]
        L.hhrr_init_equilibrium.argtypes = [vp, vp, vp, C.c_int]
        L.hhrr_set_static_geometry.argtypes = [vp, vp, vp, vp]
        L.hhrr_set_body.argtypes = [vp, i32, vp, vp, vp]
        L.hhrr_set_fringe.argtypes = [vp, i32, i32, vp]
        L.hhrr_set_rotor.argtypes = [vp, C.POINTER(RotorDesc)]
        L.hhrr_enable_wall_model.argtypes = [vp, C.c_int]
        L.hhrr_update_geometry.argtypes = [vp]
        L.hhrr_set_fsi_region.argtypes = [vp, i32, vp]
        L.hhrr_set_wall_function.argtypes = [vp, i32]
        L.hhrr_set_wall_model_variant.argtypes = [vp, i32, i32]
        L.hhrr_population_storage.argtypes = [vp]
        L.hhrr_step.argtypes = [vp, i32]
        L.hhrr_step_count.restype = i64
        L.hhrr_step_count.argtypes = [vp]
        L.hhrr_get_moments.argtypes = [vp, vp, vp]
        L.hhrr_get_moments_device.argtypes = [vp, vp, vp]
        L.hhrr_get_forces.argtypes = [vp, i64, i64, vp]
        L.hhrr_get_torques.argtypes = [vp, i64, i64, vp]
        L.hhrr_get_rotor_coefficients.argtypes = [vp, i64, i64, C.c_double, C.c_double, C.c_double, vp, vp]
        L.hhrr_force_history.restype = i64
        L.hhrr_get_cell_types.argtypes = [vp, vp, vp, vp]
        L.hhrr_get_wall_list.argtypes = [vp, i64, vp, vp, vp, vp, C.POINTER(i64)]
        L.hhrr_get_wall_state.argtypes = [vp, i64, C.POINTER(dbl), vp, vp, C.POINTER(i32)]
        L.hhrr_get_populations.argtypes = [vp, vp]
        L.hhrr_set_populations.argtypes = [vp, vp]
        L.hhrr_get_cell_populations.argtypes = [vp, i64, vp, vp, vp]
        L.hhrr_get_uhat.argtypes = [vp, vp]
        L.hhrr_get_wall_model_state.argtypes = [vp, i64, vp, vp, vp, vp, vp, C.POINTER(i64)]
        L.hhrr_set_wall_model_state.argtypes = [vp, i64, vp, vp, vp, vp, vp]
        L.hhrr_set_step_count.argtypes = [vp, i64]
        L.hhrr_check_finite.argtypes = [vp]
        L.hhrr_set_kernel_variant.argtypes = [vp, i32]
        L.hhrr_set_lookahead.argtypes = [vp, C.c_int]
        L.hhrr_set_launch_shape.argtypes = [vp, i32, i32]
        L.hhrr_set_timing.argtypes = [vp, C.c_int]
        L.hhrr_get_timing.argtypes = [vp, C.POINTER(dbl), C.POINTER(i64)]
        L.hhrr_launch_count.restype = i64
        L.hhrr_launch_count.argtypes = [vp]
        L.hhrr_last_error.restype = C.c_char_p
        L.hhrr_version.restype = C.c_char_p
        L.hhrr_velocity_set.restype = i32
        L.hhrr_halo_floats.restype = i64
        L.hhrr_halo_floats.argtypes = [vp]
        L.hhrr_halo_pack.argtypes = [vp, i32, vp]
        L.hhrr_halo_unpack.argtypes = [vp, i32, vp]
        L.hhrr_wall_model_noalloc.argtypes = [vp, i64, vp, vp, vp, vp]
        if L.hhrr_velocity_set() != q:
            raise RuntimeError(f"{path} was built for D3Q{L.hhrr_velocity_set()}, not D3Q{q}")
        _libs[q] = L
    return _libs[q]


W_FALLBACK = 1   # hhrr_set_kernel_variant: the default kernel cannot tile this lattice, variant 2 runs


def _check(rc, q=27):
    if rc < 0:
        raise HhrrError(rc, lib(q).hhrr_last_error().decode())
    return rc


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


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


def _rotor_desc(sdf, tag, spacing, origin, centre, axis, omega, theta0, n_tags):
    sdf = np.ascontiguousarray(sdf, np.float32)
    tag = np.ascontiguousarray(tag, np.uint8)
    gz, gy, gx = sdf.shape
    r = RotorDesc()
    r.sdf, r.tag = sdf.ctypes.data, tag.ctypes.data
    r.gx, r.gy, r.gz = gx, gy, gz
    r.spacing = spacing
    r.origin[:] = list(origin)
    r.centre[:] = list(centre)
    r.axis[:] = list(axis)
    r.omega, r.theta0, r.n_tags = omega, theta0, n_tags
    return r, (sdf, tag)


def workspace_bytes(params: Params, rotor_shape=None, q=27) -> int:
    r = None
    if rotor_shape is not None:
        r = RotorDesc()
        r.gz, r.gy, r.gx = rotor_shape
    n = lib(q).hhrr_workspace_bytes(C.byref(params), C.byref(r) if r is not None else None)
    if n == 0:
        raise HhrrError(-1, "hhrr_workspace_bytes: invalid parameters")
    return n


class Lattice:
    """One lattice on one GPU.  Method names mirror include/hhrr.h without the prefix."""

    def __init__(self, params: Params, rotor_shape=None, device="cuda:0", stream=None, q=27, guard_bytes=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2510_13726_b200 needs a CUDA device (no CPU fallback)")
        self.p = params
        self.q = q                      # velocity set: 27 (libhhrr.so) or 19 (libhhrr_q19.so)
        self.lib = lib(q)
        self.nx, self.ny, self.nz = params.nx, params.ny, params.nz
        self.n = self.nx * self.ny * self.nz
        self.device = torch.device(device)
        nbytes = workspace_bytes(params, rotor_shape, q)
        with torch.cuda.device(self.device):
            # guard_bytes > 0 (tests): canary regions of 0xA5 before and after the workspace handed to the library
            self.guard_bytes = int(guard_bytes)
            self._alloc = torch.empty(nbytes + 2 * self.guard_bytes, dtype=torch.uint8, device=self.device)
            if self.guard_bytes:
                self._alloc[:self.guard_bytes] = 0xA5
                self._alloc[self.guard_bytes + nbytes:] = 0xA5
            self.workspace = self._alloc[self.guard_bytes:self.guard_bytes + nbytes]
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            self._check(self.lib.hhrr_create(C.byref(params), C.c_void_p(self.workspace.data_ptr()), nbytes,
                                     C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self.h = h

    def _check(self, rc):
        return _check(rc, self.q)

    def guards_intact(self):
        """True if no kernel wrote outside the workspace (only meaningful with guard_bytes > 0)."""
        import torch
        self.synchronize()
        torch.cuda.synchronize(self.device)
        g, n = self.guard_bytes, self.workspace.numel()
        return bool((self._alloc[:g] == 0xA5).all().item() and (self._alloc[g + n:] == 0xA5).all().item())

    def close(self):
        if getattr(self, "h", None):
            self.lib.hhrr_destroy(self.h)
            self.h = None
            self.workspace = None
            self._alloc = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- setup
    def init_equilibrium(self, rho, u, with_neq=False):
        rho = _f32(rho).ravel()
        u = _f32(u).reshape(3, -1)
        assert rho.size == self.n and u.shape[1] == self.n
        self._check(self.lib.hhrr_init_equilibrium(self.h, _p(rho), _p(u), int(with_neq)))

    def set_static_geometry(self, phi, tag=None, d_override=None):
        phi = None if phi is None else _f32(phi).ravel()
        tag = None if tag is None else np.ascontiguousarray(tag, np.uint8).ravel()
        dov = None if d_override is None else _f32(d_override).ravel()
        self._check(self.lib.hhrr_set_static_geometry(self.h, _p(phi), _p(tag), _p(dov)))

    def set_body(self, tag, centre=(0, 0, 0), omega=(0, 0, 0), vel=(0, 0, 0)):
        c, o, v = _f64(centre), _f64(omega), _f64(vel)
        self._check(self.lib.hhrr_set_body(self.h, int(tag), _p(c), _p(o), _p(v)))

    def set_fringe(self, x0, x1, u_in):
        u = _f64(u_in)
        self._check(self.lib.hhrr_set_fringe(self.h, int(x0), int(x1), _p(u)))

    def set_rotor(self, sdf, tag, spacing, origin, centre, axis, omega, theta0, n_tags):
        r, keep = _rotor_desc(sdf, tag, spacing, origin, centre, axis, omega, theta0, n_tags)
        self._check(self.lib.hhrr_set_rotor(self.h, C.byref(r)))
        del keep

    def enable_wall_model(self, enable=True):
        self._check(self.lib.hhrr_enable_wall_model(self.h, int(enable)))

    def set_fsi_region(self, boxes):
        """boxes: iterable of (x0, x1, y0, y1, z0, z1), half-open; empty = HHRRLBM everywhere."""
        b = np.ascontiguousarray(np.asarray(list(boxes), np.int32).reshape(-1, 6))
        self._check(self.lib.hhrr_set_fsi_region(self.h, int(b.shape[0]), _p(b) if b.size else None))

    def set_wall_model_variant(self, slip=0, shear=0):
        """Second readings of PAPER.md:314 / :324 (include/hhrr.h)."""
        self._check(self.lib.hhrr_set_wall_model_variant(self.h, int(slip), int(shear)))

    def set_wall_function(self, kind):
        """0: truncated Spalding (Eq. 18, default); 1: Musker's profile."""
        self._check(self.lib.hhrr_set_wall_function(self.h, int(kind)))

    def update_geometry(self):
        self._check(self.lib.hhrr_update_geometry(self.h))

    def set_kernel_variant(self, variant):
        """Returns HHRR_OK (0) or the notice W_FALLBACK (1): variant 5 cannot tile the lattice, variant 2 runs."""
        return self._check(self.lib.hhrr_set_kernel_variant(self.h, int(variant)))

    def set_launch_shape(self, chunk_planes=0, cluster=0):
        self._check(self.lib.hhrr_set_launch_shape(self.h, int(chunk_planes), int(cluster)))

    def set_lookahead(self, enable=True):
        self._check(self.lib.hhrr_set_lookahead(self.h, int(bool(enable))))

    def population_storage(self):
        return int(self.lib.hhrr_population_storage(self.h))

    # ---- time loop
    def step(self, n=1):
        self._check(self.lib.hhrr_step(self.h, int(n)))

    def step_count(self):
        return self.lib.hhrr_step_count(self.h)

    def launch_count(self):
        return self.lib.hhrr_launch_count(self.h)

    def set_timing(self, enable=True):
        self._check(self.lib.hhrr_set_timing(self.h, int(enable)))

    def timing(self):
        """(summed collide-stream device ms, launches covered) since the last call."""
        ms, k = C.c_double(0), C.c_int64(0)
        self._check(self.lib.hhrr_get_timing(self.h, C.byref(ms), C.byref(k)))
        return ms.value, k.value

    def check_finite(self):
        self._check(self.lib.hhrr_check_finite(self.h))

    # ---- outputs
    def moments(self):
        rho = np.empty(self.n, np.float32)
        v = np.empty((3, self.n), np.float32)
        self._check(self.lib.hhrr_get_moments(self.h, _p(rho), _p(v)))
        return rho, v

    def moments_device(self, rho_t, v_t):
        """rho_t: float32 CUDA tensor [n]; v_t: float32 CUDA tensor [3, n]; asynchronous."""
        self._check(self.lib.hhrr_get_moments_device(self.h, C.c_void_p(rho_t.data_ptr()), C.c_void_p(v_t.data_ptr())))

    def forces(self, first=0, count=None):
        if count is None:
            count = self.step_count() - first
        F = np.zeros((count, MAX_TAGS, 3))
        if count:
            self._check(self.lib.hhrr_get_forces(self.h, int(first), int(count), _p(F)))
        return F

    def torques(self, first=0, count=None):
        if count is None:
            count = self.step_count() - first
        M = np.zeros((count, MAX_TAGS, 3))
        if count:
            self._check(self.lib.hhrr_get_torques(self.h, int(first), int(count), _p(M)))
        return M

    def rotor_coefficients(self, rho, u_inf, radius, first=0, count=None):
        """(C_T, C_P) per step: thrust coefficient of Eq. 26 and power coefficient (include/hhrr.h)."""
        if count is None:
            count = self.step_count() - first
        ct = np.zeros(count)
        cp = np.zeros(count)
        self._check(self.lib.hhrr_get_rotor_coefficients(self.h, int(first), int(count), float(rho), float(u_inf),
                                                         float(radius), _p(ct), _p(cp)))
        return ct, cp

    def cell_types(self):
        t = np.empty(self.n, np.uint8)
        g = np.empty(self.n, np.uint8)
        d = np.empty(self.n, np.float32)
        self._check(self.lib.hhrr_get_cell_types(self.h, _p(t), _p(g), _p(d)))
        return t, g, d

    def wall_list(self):
        k = C.c_int64(0)
        self._check(self.lib.hhrr_get_wall_list(self.h, 0, None, None, None, None, C.byref(k)))
        k = k.value
        idx = np.zeros(k, np.int32)
        y1n = np.zeros((k, 3))
        ut = np.zeros(k)
        va = np.zeros(k, np.uint8)
        if k:
            kk = C.c_int64(0)
            self._check(self.lib.hhrr_get_wall_list(self.h, k, _p(idx), _p(y1n), _p(ut), _p(va), C.byref(kk)))
        return idx, y1n, ut, va

    def wall_state(self, cell):
        ut = C.c_double(0)
        valid = C.c_int32(0)
        u = np.zeros(3)
        s = np.zeros(6)
        self._check(self.lib.hhrr_get_wall_state(self.h, int(cell), C.byref(ut), _p(u), _p(s), C.byref(valid)))
        return valid.value, ut.value, u, s

    def wall_model_state(self):
        """(idx int32[k], u_tau f64[k], u_wm f32[k,3], s_wm f32[k,6], valid u8[k]) of the current wall list."""
        kk = C.c_int64(0)
        self._check(self.lib.hhrr_get_wall_model_state(self.h, 0, None, None, None, None, None, C.byref(kk)))
        k = kk.value
        idx = np.zeros(k, np.int32); ut = np.zeros(k); uw = np.zeros((k, 3), np.float32)
        sw = np.zeros((k, 6), np.float32); va = np.zeros(k, np.uint8)
        if k:
            self._check(self.lib.hhrr_get_wall_model_state(self.h, k, _p(idx), _p(ut), _p(uw), _p(sw), _p(va), C.byref(kk)))
        return idx, ut, uw, sw, va

    def set_wall_model_state(self, idx, u_tau, u_wm, s_wm, valid):
        idx = np.ascontiguousarray(idx, np.int32); ut = np.ascontiguousarray(u_tau, np.float64)
        uw = np.ascontiguousarray(u_wm, np.float32); sw = np.ascontiguousarray(s_wm, np.float32)
        va = np.ascontiguousarray(valid, np.uint8)
        self._check(self.lib.hhrr_set_wall_model_state(self.h, len(idx), _p(idx), _p(ut), _p(uw), _p(sw), _p(va)))

    def wall_model_noalloc(self, capacity, start_t, utau_t, uwm_t, swm_t):
        """hhrr_wall_model_noalloc: CUDA tensors start_t (float64 [capacity] or None), utau_t (float64 [capacity]),
        uwm_t (float32 [capacity, 3]), swm_t (float32 [capacity, 6]); asynchronous, allocates nothing."""
        self._check(self.lib.hhrr_wall_model_noalloc(
            self.h, int(capacity), None if start_t is None else C.c_void_p(start_t.data_ptr()),
            C.c_void_p(utau_t.data_ptr()), C.c_void_p(uwm_t.data_ptr()), C.c_void_p(swm_t.data_ptr())))

    def halo_floats(self):
        return int(self.lib.hhrr_halo_floats(self.h))

    def halo_pack(self, face, buf_t):
        """buf_t: float32 CUDA tensor of halo_floats() elements (asynchronous on the lattice's stream)."""
        self._check(self.lib.hhrr_halo_pack(self.h, int(face), C.c_void_p(buf_t.data_ptr())))

    def halo_unpack(self, face, buf_t):
        self._check(self.lib.hhrr_halo_unpack(self.h, int(face), C.c_void_p(buf_t.data_ptr())))

    def set_step_count(self, step):
        self._check(self.lib.hhrr_set_step_count(self.h, int(step)))

    def populations(self):
        f = np.empty((self.q, self.n), np.float32)
        self._check(self.lib.hhrr_get_populations(self.h, _p(f)))
        return f

    def set_populations(self, f_minus_w):
        f = _f32(f_minus_w).reshape(self.q, self.n)
        self._check(self.lib.hhrr_set_populations(self.h, _p(f)))

    def cell_populations(self, cells):
        """(f - w)[k, 27] and the stored flag bytes of the given cell indices."""
        cells = np.ascontiguousarray(cells, np.int64)
        out = np.empty((cells.size, self.q), np.float32)
        fl = np.empty(cells.size, np.uint8)
        self._check(self.lib.hhrr_get_cell_populations(self.h, cells.size, _p(cells), _p(out), _p(fl)))
        return out, fl

    def uhat(self):
        u = np.empty((3, self.n), np.float32)
        self._check(self.lib.hhrr_get_uhat(self.h, _p(u)))
        return u

    def synchronize(self):
        self.stream.synchronize()
