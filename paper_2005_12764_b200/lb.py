"""Thin ctypes binding of the C-ABI library (include/lb.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of liblb_b200.so.  PyTorch provides device
memory (the caching allocator is handed to the library through lb_set_allocator) and the
stream (lb_set_stream with torch's current stream).  There is no CPU fallback: if the library
is missing this module fails to import, and without a CUDA device the calls return LB_ECUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

LB_OK, LB_EINVAL, LB_ENOMEM, LB_ECUDA, LB_ESTATE = 0, -1, -2, -3, -4

SYMBOLS = [
    "lb_set_allocator", "lb_create", "lb_destroy", "lb_set_stream", "lb_set_geometry",
    "lb_set_wall_velocity", "lb_set_wall_type", "lb_set_body_force", "lb_set_model", "lb_set_forcing", "lb_set_nc_cutoff", "lb_set_nc_symmetric", "lb_set_wall_phi", "lb_set_storage", "lb_init", "lb_step",
    "lb_check_state", "lb_check_state_static", "lb_get_macros", "lb_get_populations", "lb_set_populations", "lb_get_phi", "lb_launch_count",
    "lb_device_bytes", "lb_last_error", "lb_set_profiling", "lb_last_step_ms", "lb_set_tuning",
    "lb_set_slab", "lb_slab_halo_bytes", "lb_slab_begin", "lb_slab_interior", "lb_slab_end",
    "lb_slab_pack_phi", "lb_slab_unpack_phi", "lb_slab_part_get", "lb_slab_part_put",
    "lb_set_particles", "lb_set_particle_options", "lb_set_particle_force", "lb_get_particles",
]


class lb_params(C.Structure):
    _fields_ = [("tau_r", C.c_float), ("tau_b", C.c_float), ("A", C.c_float), ("beta", C.c_float),
                ("A_nc", C.c_float)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


def _load():
    path = _build.LIB
    if not os.path.exists(path):
        raise ImportError(
            "CUDA extension %s is missing: run `python -m paper_2005_12764_b200.build` "
            "(there is no CPU fallback)" % path)
    lib = C.CDLL(path)
    vp, fp = C.c_void_p, C.c_void_p   # arrays are passed as raw addresses (host or device)
    lib.lb_set_allocator.argtypes = [ALLOC_FN, FREE_FN, vp]
    lib.lb_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(lb_params), C.POINTER(vp)]
    lib.lb_destroy.argtypes = [vp]
    lib.lb_destroy.restype = None
    lib.lb_set_stream.argtypes = [vp, vp]
    lib.lb_set_geometry.argtypes = [vp, fp]
    lib.lb_set_wall_velocity.argtypes = [vp, C.c_int, C.c_float, C.c_float, C.c_float]
    lib.lb_set_wall_type.argtypes = [vp, C.c_int, C.c_int, C.c_float, C.c_float]
    lib.lb_set_body_force.argtypes = [vp, C.c_float, C.c_float, C.c_float]
    lib.lb_set_model.argtypes = [vp, C.c_int, C.c_float]
    lib.lb_set_forcing.argtypes = [vp, C.c_int]
    lib.lb_set_nc_cutoff.argtypes = [vp, C.c_float]
    lib.lb_set_nc_symmetric.argtypes = [vp, C.c_int]
    lib.lb_set_wall_phi.argtypes = [vp, C.c_int, C.c_float]
    lib.lb_set_storage.argtypes = [vp, C.c_int]
    lib.lb_init.argtypes = [vp, fp, fp, fp]
    lib.lb_step.argtypes = [vp, C.c_int]
    lib.lb_check_state.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    lib.lb_check_state_static.argtypes = [vp, vp]
    lib.lb_get_macros.argtypes = [vp, fp, fp, fp]
    lib.lb_get_populations.argtypes = [vp, C.c_int, fp]
    lib.lb_set_populations.argtypes = [vp, C.c_int, fp]
    lib.lb_get_phi.argtypes = [vp, fp]
    lib.lb_launch_count.argtypes = [vp]
    lib.lb_launch_count.restype = C.c_longlong
    lib.lb_device_bytes.argtypes = [vp]
    lib.lb_device_bytes.restype = C.c_size_t
    lib.lb_last_error.argtypes = [vp]
    lib.lb_last_error.restype = C.c_char_p
    lib.lb_set_tuning.argtypes = [vp, C.c_char_p, C.c_int]
    lib.lb_set_profiling.argtypes = [vp, C.c_int]
    lib.lb_last_step_ms.argtypes = [vp, C.c_int, C.POINTER(C.c_float)]
    lib.lb_set_slab.argtypes = [vp, C.c_int, C.c_int]
    lib.lb_slab_halo_bytes.argtypes = [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]
    lib.lb_slab_begin.argtypes = [vp, fp, fp]
    lib.lb_slab_interior.argtypes = [vp]
    lib.lb_slab_end.argtypes = [vp, fp, fp]
    lib.lb_slab_pack_phi.argtypes = [vp, fp, fp]
    lib.lb_slab_unpack_phi.argtypes = [vp, fp, fp]
    lib.lb_slab_part_get.argtypes = [vp, vp]
    lib.lb_slab_part_put.argtypes = [vp, vp]
    lib.lb_set_particles.argtypes = [vp, C.c_int, fp]
    lib.lb_set_particle_options.argtypes = [vp, C.c_int, C.c_double, C.c_double, C.c_int]
    lib.lb_set_particle_force.argtypes = [vp, C.c_int, fp, fp]
    lib.lb_get_particles.argtypes = [vp, fp, fp]
    return lib


lib = _load()

_torch_alloc_installed = False
_keepalive = []


def use_torch_allocator():
    """Route the library's device allocations through PyTorch's CUDA caching allocator."""
    global _torch_alloc_installed
    if _torch_alloc_installed:
        return
    import torch

    def _alloc(nbytes, _user):
        try:
            return torch.cuda.caching_allocator_alloc(int(nbytes))
        except Exception:      # out of memory -> NULL -> LB_ENOMEM
            return None

    def _free(ptr, _user):
        try:
            torch.cuda.caching_allocator_delete(ptr)
        except AttributeError:      # interpreter shutdown: torch is already torn down, the context frees the memory
            pass

    a, f = ALLOC_FN(_alloc), FREE_FN(_free)
    _keepalive.extend([a, f])
    rc = lib.lb_set_allocator(a, f, None)
    if rc != LB_OK:
        raise RuntimeError("lb_set_allocator failed: %d" % rc)
    _torch_alloc_installed = True


class LBError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("lb error %d: %s" % (code, msg))
        self.code = code


def _addr(a):
    """Raw address of a numpy array (host) or a torch tensor (host or device), or None."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    assert a.is_contiguous()
    return a.data_ptr()


class LB:
    """One simulation.  Method names and argument order follow include/lb.h.

    Arrays may be numpy float32 arrays (host), or torch float32 tensors on the CPU or the GPU.
    Scalar fields [nz, ny, nx]; u [3, nz, ny, nx]; populations [19, nz, ny, nx]."""

    def __init__(self, nx, ny, nz, tau_r=1.0, tau_b=1.0, A=0.0, beta=0.0, A_nc=0.0, torch_allocator=True):
        if torch_allocator:
            use_torch_allocator()
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.two = True
        p = lb_params(tau_r, tau_b, A, beta, A_nc)
        h = C.c_void_p()
        rc = lib.lb_create(self.nx, self.ny, self.nz, C.byref(p), C.byref(h))
        if rc != LB_OK:
            raise LBError(rc, (lib.lb_last_error(None) or b"").decode())
        self.h = h
        self._sync_stream()

    def _ck(self, rc):
        if rc != LB_OK:
            raise LBError(rc, (lib.lb_last_error(self.h) or b"").decode())

    def _sync_stream(self):
        try:
            import torch
            if torch.cuda.is_available():
                self._ck(lib.lb_set_stream(self.h, C.c_void_p(torch.cuda.current_stream().cuda_stream)))
        except ImportError:
            pass

    def destroy(self):
        if getattr(self, "h", None) and lib is not None:   # lib is None at interpreter shutdown
            lib.lb_destroy(self.h)
            self.h = None

    __del__ = destroy

    def set_geometry(self, solid_mask):
        self._sync_stream()
        self._ck(lib.lb_set_geometry(self.h, _addr(solid_mask)))

    def set_wall_velocity(self, group, ux, uy, uz):
        self._ck(lib.lb_set_wall_velocity(self.h, int(group), ux, uy, uz))

    def set_wall_type(self, group, kind, rho_r=0.0, rho_b=0.0):
        t = {"wall": 0, "inlet": 1, "reservoir": 2, "outlet": 3}.get(kind, kind)
        self._ck(lib.lb_set_wall_type(self.h, int(group), int(t), float(rho_r), float(rho_b)))

    def set_body_force(self, gx, gy, gz):
        self._ck(lib.lb_set_body_force(self.h, gx, gy, gz))

    def set_model(self, model, G_C=0.0):
        self._ck(lib.lb_set_model(self.h, {"cg": 0, "sc": 1}.get(model, model), float(G_C)))

    def set_forcing(self, mode):
        self._ck(lib.lb_set_forcing(self.h, {"guo": 0, "edm": 1}.get(mode, mode)))

    def set_nc_cutoff(self, phi_c):
        self._ck(lib.lb_set_nc_cutoff(self.h, phi_c))

    def set_nc_symmetric(self, on):
        self._ck(lib.lb_set_nc_symmetric(self.h, int(bool(on))))

    def set_wall_phi(self, phi_wall):
        """Prescribed phi at solid nodes; None switches back to the neutral wall."""
        self._ck(lib.lb_set_wall_phi(self.h, 0 if phi_wall is None else 1, 0.0 if phi_wall is None else float(phi_wall)))

    def set_storage(self, mode):
        self._ck(lib.lb_set_storage(self.h, {"ab": 0, "aa": 1}.get(mode, mode)))

    def init(self, rho_r, rho_b, u):
        self._sync_stream()
        self.two = rho_b is not None
        self._ck(lib.lb_init(self.h, _addr(rho_r), _addr(rho_b), _addr(u)))

    def step(self, nsteps=1):
        self._sync_stream()
        self._ck(lib.lb_step(self.h, int(nsteps)))

    def check_state(self):
        """(mass_r, mass_b) summed on the device; raises LBError(LB_ESTATE) on a non-finite state."""
        self._sync_stream()
        mr, mb = C.c_double(), C.c_double()
        self._ck(lib.lb_check_state(self.h, C.byref(mr), C.byref(mb)))
        return float(mr.value), float(mb.value)

    def check_state_static(self, d_out):
        """{mass_r, mass_b, non-finite sites} into d_out (3 float64 on the device) on the handle's
        stream: no allocation, no synchronisation (include/lb.h)."""
        self._sync_stream()
        self._ck(lib.lb_check_state_static(self.h, _addr(d_out)))

    def get_macros(self, rho_r=None, rho_b=None, u=None):
        """Fills the given arrays (host or device); allocates numpy outputs when none given."""
        self._sync_stream()
        if rho_r is None and rho_b is None and u is None:
            rho_r = np.empty(self.shape, np.float32)
            rho_b = np.empty(self.shape, np.float32) if self.two else None
            u = np.empty((3,) + self.shape, np.float32)
        self._ck(lib.lb_get_macros(self.h, _addr(rho_r), _addr(rho_b), _addr(u)))
        return rho_r, rho_b, u

    def get_populations(self, comp, out=None):
        self._sync_stream()
        if out is None:
            out = np.empty((19,) + self.shape, np.float32)
        self._ck(lib.lb_get_populations(self.h, comp, _addr(out)))
        return out

    def set_populations(self, comp, f):
        self._sync_stream()
        self._ck(lib.lb_set_populations(self.h, comp, _addr(f)))

    def get_phi(self, out=None):
        self._sync_stream()
        if out is None:
            out = np.empty(self.shape, np.float32)
        self._ck(lib.lb_get_phi(self.h, _addr(out)))
        return out

    # ---- z slabs (include/lb.h "z-slab decomposition"); message buffers are device tensors
    def set_slab(self, z0, nz_global):
        self._ck(lib.lb_set_slab(self.h, int(z0), int(nz_global)))

    def slab_halo_bytes(self):
        a, b = C.c_size_t(), C.c_size_t()
        self._ck(lib.lb_slab_halo_bytes(self.h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def slab_begin(self, send_lo, send_hi):
        self._sync_stream()
        self._ck(lib.lb_slab_begin(self.h, _addr(send_lo), _addr(send_hi)))

    def slab_interior(self):
        self._sync_stream()
        self._ck(lib.lb_slab_interior(self.h))

    def slab_end(self, recv_lo, recv_hi):
        self._sync_stream()
        self._ck(lib.lb_slab_end(self.h, _addr(recv_lo), _addr(recv_hi)))

    def slab_pack_phi(self, send_lo, send_hi):
        self._sync_stream()
        self._ck(lib.lb_slab_pack_phi(self.h, _addr(send_lo), _addr(send_hi)))

    def slab_unpack_phi(self, recv_lo, recv_hi):
        self._sync_stream()
        self._ck(lib.lb_slab_unpack_phi(self.h, _addr(recv_lo), _addr(recv_hi)))

    def slab_part_get(self, d_sums):
        self._sync_stream()
        self._ck(lib.lb_slab_part_get(self.h, _addr(d_sums)))

    def slab_part_put(self, d_sums):
        self._sync_stream()
        self._ck(lib.lb_slab_part_put(self.h, _addr(d_sums)))

    # ---- rigid particles (include/lb.h "rigid spherical particles"); state rows = lb_particle:
    # r[3], u[3], w[3], q[4], R, mass (float64)
    def set_particles(self, state):
        st = np.ascontiguousarray(state, dtype=np.float64).reshape(-1, 15)
        self.npart = len(st)
        self._ck(lib.lb_set_particles(self.h, self.npart, st.ctypes.data))

    def set_particle_options(self, mobile=True, K=0.0, h_c=0.0, lubrication=False):
        self._ck(lib.lb_set_particle_options(self.h, int(mobile), float(K), float(h_c), int(lubrication)))

    def set_particle_force(self, p, F=(0, 0, 0), T=(0, 0, 0)):
        f, t = np.array(F, np.float64), np.array(T, np.float64)
        self._ck(lib.lb_set_particle_force(self.h, int(p), f.ctypes.data, t.ctypes.data))

    def get_particles(self):
        """(state [n, 15], force [n, 9]: F[3], T[3] from the fluid links of the last step, F_pp[3])."""
        self._sync_stream()
        st = np.zeros((self.npart, 15))
        fo = np.zeros((self.npart, 9))
        self._ck(lib.lb_get_particles(self.h, st.ctypes.data, fo.ctypes.data))
        return st, fo

    def launch_count(self):
        return int(lib.lb_launch_count(self.h))

    def device_bytes(self):
        return int(lib.lb_device_bytes(self.h))

    def set_tuning(self, **kw):
        for k, v in kw.items():
            self._ck(lib.lb_set_tuning(self.h, k.encode(), int(v)))

    def set_profiling(self, on):
        self._ck(lib.lb_set_profiling(self.h, int(on)))

    def last_step_ms(self, which=0):
        ms = C.c_float()
        self._ck(lib.lb_last_step_ms(self.h, which, C.byref(ms)))
        return float(ms.value)


def from_workload(w, storage="ab", torch_allocator=True):
    """Create and configure (not initialise) an LB for a workloads.Workload."""
    sim = LB(w.nx, w.ny, w.nz, w.tau_r, w.tau_b, w.A, w.beta, w.A_nc, torch_allocator=torch_allocator)
    sim.set_storage(storage)
    if w.solid is not None:
        sim.set_geometry(np.ascontiguousarray(w.solid, dtype=np.uint8))
    sim.set_body_force(*w.g)
    sim.set_nc_cutoff(w.phi_c)
    from . import workloads
    workloads.configure_walls(sim, w)      # wall groups of the workload (velocities, open boundaries)
    return sim
