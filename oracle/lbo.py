"""ctypes binding of the fp64 CPU oracle (oracle/lbo.cpp) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_2005_12764_b200 and vice versa.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lbo.cpp")
# LBO_SANITIZE=1: the oracle is built with -fsanitize=address,undefined into its own library (run the CPU
# tests as  LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 LBO_SANITIZE=1
# python -m pytest tests -m "not gpu";  DESIGN.md section 7 records the outcome)
_SAN = os.environ.get("LBO_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "liblbo_san.so" if _SAN else "liblbo.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle/lbo.cpp to oracle/liblbo.so with g++ -O2 -fopenmp (no GPU needed)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SAN else ["-O2"]
        subprocess.check_call(
            ["g++", "-std=c++17"] + flags + ["-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        vp, dp, ip, u8p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_uint8)
        lib.lbo_create.argtypes = [C.c_int, C.c_int, C.c_int, dp, C.POINTER(vp)]
        lib.lbo_destroy.argtypes = [vp]
        lib.lbo_destroy.restype = None
        lib.lbo_set_geometry.argtypes = [vp, u8p]
        lib.lbo_set_body_force.argtypes = [vp, C.c_double, C.c_double, C.c_double]
        lib.lbo_set_wall_velocity.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_double]
        lib.lbo_set_nc_cutoff.argtypes = [vp, C.c_double]
        lib.lbo_set_nc_mode.argtypes = [vp, C.c_int]
        lib.lbo_set_nc_symmetric.argtypes = [vp, C.c_int]
        lib.lbo_set_wall_type.argtypes = [vp, C.c_int, C.c_int, C.c_double, C.c_double]
        lib.lbo_set_wall_phi.argtypes = [vp, C.c_int, C.c_double]
        lib.lbo_set_forcing.argtypes = [vp, C.c_int]
        lib.lbo_set_model.argtypes = [vp, C.c_int, C.c_double]
        lib.lbo_init.argtypes = [vp, dp, dp, dp]
        lib.lbo_step.argtypes = [vp, C.c_int]
        lib.lbo_get_macros.argtypes = [vp, dp, dp, dp]
        lib.lbo_get_populations.argtypes = [vp, C.c_int, dp]
        lib.lbo_set_populations.argtypes = [vp, C.c_int, dp]
        lib.lbo_get_fields.argtypes = [vp, dp, dp, dp, ip, dp]
        lib.lbo_set_particles.argtypes = [vp, C.c_int, dp]
        lib.lbo_get_particles.argtypes = [vp, dp, dp]
        lib.lbo_set_particle_options.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_int]
        lib.lbo_set_particle_force.argtypes = [vp, C.c_int, dp, dp]
        lib.lbo_get_node_map.argtypes = [vp, u8p, ip]
        lib.lbo_constants.argtypes = [ip, ip, dp, dp]
        lib.lbo_constants.restype = None
        _lib = lib
    return _lib


def _dptr(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def constants():
    """(c[19,3], opp[19], w[19], B[19]) as the oracle holds them."""
    lib = _load()
    c = np.zeros((19, 3), np.int32)
    opp = np.zeros(19, np.int32)
    w = np.zeros(19)
    b = np.zeros(19)
    lib.lbo_constants(c.ctypes.data_as(C.POINTER(C.c_int)), opp.ctypes.data_as(C.POINTER(C.c_int)),
                      _dptr(w), _dptr(b))
    return c, opp, w, b


class Oracle:
    """Scalar fields are [nz, ny, nx] (x fastest); u is [3, nz, ny, nx]; populations [19, nz, ny, nx]."""

    def __init__(self, nx, ny, nz, tau_r=1.0, tau_b=1.0, A=0.0, beta=0.0, A_nc=0.0):
        self.lib = _load()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.two = True
        p = np.array([tau_r, tau_b, A, beta, A_nc], np.float64)
        h = C.c_void_p()
        rc = self.lib.lbo_create(self.nx, self.ny, self.nz, _dptr(p), C.byref(h))
        if rc != 0:
            raise ValueError("lbo_create failed: %d" % rc)
        self.h = h

    def _ck(self, rc, what):
        if rc != 0:
            raise RuntimeError("%s failed: %d" % (what, rc))

    def close(self):
        if getattr(self, "h", None):
            self.lib.lbo_destroy(self.h)
            self.h = None

    __del__ = close

    def set_geometry(self, mask):
        if mask is None:
            self._ck(self.lib.lbo_set_geometry(self.h, None), "lbo_set_geometry")
            return
        m = np.ascontiguousarray(mask, dtype=np.uint8).reshape(self.shape)
        self._ck(self.lib.lbo_set_geometry(self.h, m.ctypes.data_as(C.POINTER(C.c_uint8))), "lbo_set_geometry")

    def set_wall_velocity(self, group, ux, uy, uz):
        """Velocity of the walls whose mask value is `group` (2 or 3)."""
        self._ck(self.lib.lbo_set_wall_velocity(self.h, group, ux, uy, uz), "lbo_set_wall_velocity")

    def set_wall_type(self, group, kind, rho_r=0.0, rho_b=0.0):
        """'wall' (moving wall), 'inlet' (velocity inlet), 'reservoir' (pressure boundary, both densities
        prescribed) or 'outlet' (pressure outlet, total density prescribed), G31."""
        t = {'wall': 0, 'inlet': 1, 'reservoir': 2, 'outlet': 3}.get(kind, kind)
        self._ck(self.lib.lbo_set_wall_type(self.h, group, t, float(rho_r), float(rho_b)), "lbo_set_wall_type")

    def set_body_force(self, gx, gy, gz):
        self._ck(self.lib.lbo_set_body_force(self.h, gx, gy, gz), "lbo_set_body_force")

    def set_nc_cutoff(self, phi_c):
        self._ck(self.lib.lbo_set_nc_cutoff(self.h, phi_c), "lbo_set_nc_cutoff")

    def set_model(self, model, G_C=0.0):
        """0 / 'cg' = colour gradient, 1 / 'sc' = Shan-Chen + exact difference (Eq. 5-10 of the paper)."""
        self._ck(self.lib.lbo_set_model(self.h, {'cg': 0, 'sc': 1}.get(model, model), float(G_C)), "lbo_set_model")

    def set_forcing(self, mode):
        """0 / 'guo' = Guo forcing, 1 / 'edm' = exact-difference forcing (Eq. 9)."""
        self._ck(self.lib.lbo_set_forcing(self.h, {'guo': 0, 'edm': 1}.get(mode, mode)), "lbo_set_forcing")

    def set_nc_symmetric(self, on):
        """Colour-symmetric near-contact probe (G29)."""
        self._ck(self.lib.lbo_set_nc_symmetric(self.h, int(bool(on))), "lbo_set_nc_symmetric")

    def set_wall_phi(self, phi_wall):
        """Prescribed phi at solid nodes (wetting, G30); None = neutral rule G8."""
        self._ck(self.lib.lbo_set_wall_phi(self.h, 0 if phi_wall is None else 1,
                                           0.0 if phi_wall is None else float(phi_wall)), "lbo_set_wall_phi")

    def set_nc_mode(self, mode):
        self._ck(self.lib.lbo_set_nc_mode(self.h, mode), "lbo_set_nc_mode")

    def init(self, rho_r, rho_b, u):
        rr = _f64(rho_r).reshape(self.shape)
        rb = None if rho_b is None else _f64(rho_b).reshape(self.shape)
        uu = _f64(u).reshape((3,) + self.shape)
        self.two = rb is not None
        self._ck(self.lib.lbo_init(self.h, _dptr(rr), _dptr(rb), _dptr(uu)), "lbo_init")

    def step(self, n=1):
        self._ck(self.lib.lbo_step(self.h, int(n)), "lbo_step")

    def get_macros(self):
        rr = np.zeros(self.shape)
        rb = np.zeros(self.shape) if self.two else None
        u = np.zeros((3,) + self.shape)
        self._ck(self.lib.lbo_get_macros(self.h, _dptr(rr), _dptr(rb), _dptr(u)), "lbo_get_macros")
        return rr, rb, u

    def get_populations(self, comp):
        f = np.zeros((19,) + self.shape)
        self._ck(self.lib.lbo_get_populations(self.h, comp, _dptr(f)), "lbo_get_populations")
        return f

    def set_populations(self, comp, f):
        ff = _f64(f).reshape((19,) + self.shape)
        self._ck(self.lib.lbo_set_populations(self.h, comp, _dptr(ff)), "lbo_set_populations")

    # ---- rigid particles (G32-G37)
    def set_particles(self, state):
        """state [n, 15]: r[3], u[3], w[3], q[4] (w, x, y, z), R, mass.  Before init."""
        st = np.ascontiguousarray(state, dtype=np.float64).reshape(-1, 15)
        self.npart = len(st)
        self._ck(self.lib.lbo_set_particles(self.h, self.npart, _dptr(st)), "lbo_set_particles")

    def get_particles(self):
        """(state [n, 15], force [n, 9]: F[3], T[3] from the fluid links of the last step, F_pp[3])."""
        st = np.zeros((self.npart, 15))
        fo = np.zeros((self.npart, 9))
        self._ck(self.lib.lbo_get_particles(self.h, _dptr(st), _dptr(fo)), "lbo_get_particles")
        return st, fo

    def set_particle_options(self, mobile=True, K=0.0, h_c=0.0, lubrication=False):
        self._ck(self.lib.lbo_set_particle_options(self.h, int(mobile), float(K), float(h_c), int(lubrication)), "lbo_set_particle_options")

    def set_particle_force(self, p, F=(0, 0, 0), T=(0, 0, 0)):
        f, t = np.array(F, np.float64), np.array(T, np.float64)
        self._ck(self.lib.lbo_set_particle_force(self.h, int(p), _dptr(f), _dptr(t)), "lbo_set_particle_force")

    def get_node_map(self):
        sol = np.zeros(self.shape, np.uint8)
        pid = np.zeros(self.shape, np.int32)
        self._ck(self.lib.lbo_get_node_map(self.h, sol.ctypes.data_as(C.POINTER(C.c_uint8)), pid.ctypes.data_as(C.POINTER(C.c_int))), "lbo_get_node_map")
        return sol, pid

    def get_fields(self):
        """dict(phi, G[3], F[3], h (contact distance, 0 = none), margin (G12))."""
        phi = np.zeros(self.shape)
        G = np.zeros((3,) + self.shape)
        F = np.zeros((3,) + self.shape)
        h = np.zeros(self.shape, np.int32)
        m = np.zeros(self.shape)
        self._ck(self.lib.lbo_get_fields(self.h, _dptr(phi), _dptr(G), _dptr(F),
                                         h.ctypes.data_as(C.POINTER(C.c_int)), _dptr(m)), "lbo_get_fields")
        return dict(phi=phi, G=G, F=F, h=h, margin=m)
