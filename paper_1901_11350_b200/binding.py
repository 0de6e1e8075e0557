"""Thin ctypes binding of the C-ABI library (include/spinllg.h): argument marshalling only.

Every step of the hot path runs inside libspinllg.so's CUDA kernels; this module only converts numpy arrays /
torch device pointers to C pointers and raises SpinError on a non-zero return code.  There is no CPU fallback:
if the library is missing it is built with nvcc, and if that fails the import of the library raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_LIB = None

EXPORTS = [
    "spin_geometry_create", "spin_system_destroy", "spin_system_nspins", "spin_set_stream",
    "hamiltonian_set_mu_s", "hamiltonian_set_site_mu_s", "hamiltonian_set_field", "hamiltonian_set_anisotropy", "hamiltonian_set_pairs",
    "hamiltonian_set_exchange_shells", "hamiltonian_set_dmi_shells", "hamiltonian_set_quadruplets",
    "hamiltonian_set_ddi", "spin_set_images", "spin_select_image", "llg_set_image_temperatures", "gneb_forces", "gneb_iterate", "spins_set_pinned", "spins_set", "spins_get", "spins_set_device", "spins_get_device",
    "llg_configure", "llg_set_solver", "llg_set_damping_only", "minimise_vp", "minimise_vp_reset", "llg_iterate", "llg_get_step", "llg_set_step", "spin_synchronize",
    "effective_field", "effective_field_device", "energy", "observables", "topological_charge", "topological_charge_noalloc",
    "spin_set_slab", "spin_halo_doubles", "spin_halo_get", "spin_halo_put", "llg_slab_sweep", "llg_slab_step", "llg_slab_step_fused", "spin_slab_arrays", "llg_slab_advance",
    "spin_ipc_export", "spin_ipc_open", "spin_ipc_close", "spin_slab_flags", "spin_flag_signal", "spin_flag_wait",
    "spin_launch_counts", "spin_measure_fp64_tflops", "spin_profile_enable", "spin_profile_get", "spin_set_option",
    "spin_kernel_info", "spin_ddi_info", "spin_jit_compiler_info", "spin_jit_source", "spin_last_error", "spin_version",
]


class SpinError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"spinllg error {code}: {msg}")
        self.code = code


def lib() -> C.CDLL:
    """Load (building if stale) libspinllg.so and declare the prototypes of include/spinllg.h."""
    global _LIB
    if _LIB is not None:
        return _LIB
    path = _build.build()
    if not os.path.exists(path):
        raise ImportError("libspinllg.so is missing and could not be built; there is no CPU fallback")
    L = C.CDLL(path)
    dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
    i64p = C.POINTER(C.c_int64)
    proto = {
        "spin_geometry_create": (C.c_int, [dp, C.c_int, dp, ip, ip, C.c_double, C.POINTER(vp)]),
        "spin_system_destroy": (None, [vp]),
        "spin_system_nspins": (C.c_int64, [vp]),
        "spin_set_stream": (C.c_int, [vp, vp]),
        "hamiltonian_set_mu_s": (C.c_int, [vp, dp]),
        "hamiltonian_set_site_mu_s": (C.c_int, [vp, dp]),
        "hamiltonian_set_field": (C.c_int, [vp, C.c_double, dp]),
        "hamiltonian_set_anisotropy": (C.c_int, [vp, C.c_int, ip, dp, dp]),
        "hamiltonian_set_pairs": (C.c_int, [vp, C.c_int, ip, ip, ip, dp, dp]),
        "hamiltonian_set_exchange_shells": (C.c_int, [vp, C.c_int, dp]),
        "hamiltonian_set_dmi_shells": (C.c_int, [vp, C.c_int, dp, C.c_int]),
        "hamiltonian_set_quadruplets": (C.c_int, [vp, C.c_int, ip, ip, dp]),
        "hamiltonian_set_ddi": (C.c_int, [vp, C.c_int, ip]),
        "spins_set": (C.c_int, [vp, dp]),
        "spins_get": (C.c_int, [vp, dp]),
        "spins_set_device": (C.c_int, [vp, vp]),
        "spins_get_device": (C.c_int, [vp, vp]),
        "llg_configure": (C.c_int, [vp, C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_double, dp, C.c_double]),
        "llg_set_solver": (C.c_int, [vp, C.c_int]),
        "llg_set_damping_only": (C.c_int, [vp, C.c_int]),
        "spins_set_pinned": (C.c_int, [vp, C.c_void_p]),
        "spin_measure_fp64_tflops": (C.c_int, [vp, dp]),
        "spin_set_images": (C.c_int, [vp, C.c_int]),
        "gneb_forces": (C.c_int, [vp, C.c_double, C.c_int, dp, dp, dp]),
        "gneb_iterate": (C.c_int, [vp, C.c_int64, C.c_double, C.c_double, C.c_int]),
        "spin_select_image": (C.c_int, [vp, C.c_int]),
        "llg_set_image_temperatures": (C.c_int, [vp, dp]),
        "minimise_vp": (C.c_int, [vp, C.c_int64, C.c_double, C.c_double]),
        "minimise_vp_reset": (C.c_int, [vp]),
        "llg_iterate": (C.c_int, [vp, C.c_int64]),
        "llg_get_step": (C.c_int, [vp, C.POINTER(C.c_uint64)]),
        "llg_set_step": (C.c_int, [vp, C.c_uint64]),
        "spin_synchronize": (C.c_int, [vp]),
        "effective_field": (C.c_int, [vp, dp]),
        "effective_field_device": (C.c_int, [vp, vp]),
        "energy": (C.c_int, [vp, dp, dp]),
        "observables": (C.c_int, [vp, dp, dp]),
        "topological_charge": (C.c_int, [vp, dp]),
        "topological_charge_noalloc": (C.c_int, [vp, C.c_void_p]),
        "spin_launch_counts": (C.c_int, [vp, i64p, i64p]),
        "spin_set_slab": (C.c_int, [vp, C.c_int, C.c_int, C.c_int, C.c_int]),
        "spin_halo_doubles": (C.c_int, [vp, i64p, ip]),
        "spin_halo_get": (C.c_int, [vp, C.c_int, C.c_int, vp, vp]),
        "spin_halo_put": (C.c_int, [vp, C.c_int, C.c_int, vp, vp]),
        "llg_slab_sweep": (C.c_int, [vp, C.c_int, C.c_int]),
        "llg_slab_step": (C.c_int, [vp, C.c_int]),
        "llg_slab_step_fused": (C.c_int, [vp, C.c_void_p, C.c_int, C.c_void_p]),
        "spin_slab_arrays": (C.c_int, [vp, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p)]),
        "spin_ipc_export": (C.c_int, [C.c_void_p, C.c_char_p, C.POINTER(C.c_int64)]),
        "spin_ipc_open": (C.c_int, [C.c_char_p, C.c_int64, C.POINTER(C.c_void_p)]),
        "spin_ipc_close": (C.c_int, [C.c_void_p, C.c_int64]),
        "spin_slab_flags": (C.c_int, [vp, C.POINTER(C.c_void_p)]),
        "spin_flag_signal": (C.c_int, [vp, C.c_void_p, C.c_uint64]),
        "spin_flag_wait": (C.c_int, [vp, C.c_void_p, C.c_uint64]),
        "llg_slab_advance": (C.c_int, [vp]),
        "spin_profile_enable": (C.c_int, [vp, C.c_int]),
        "spin_profile_get": (C.c_int, [vp, C.c_int, dp, i64p]),
        "spin_set_option": (C.c_int, [vp, C.c_char_p, C.c_int]),
        "spin_kernel_info": (C.c_int, [vp, C.c_char_p, C.c_int]),
        "spin_jit_compiler_info": (C.c_int, [C.c_char_p, C.c_int]),
        "spin_ddi_info": (C.c_int, [vp, C.c_char_p, C.c_int]),
        "spin_jit_source": (C.c_int, [vp, C.c_char_p, C.c_int, C.c_int, i64p]),
        "spin_last_error": (C.c_char_p, []),
        "spin_version": (C.c_char_p, []),
    }
    for name, (res, args) in proto.items():
        fn = getattr(L, name)          # AttributeError here = a symbol of spinllg.h is not exported
        fn.restype = res
        fn.argtypes = args
    _LIB = L
    return L


def _check(rc):
    if rc != 0:
        raise SpinError(rc, lib().spin_last_error().decode())


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


class SpinSystem:
    """Python handle of a `spin_system*`; method names are the C-ABI names."""

    def __init__(self, bravais, basis, n_cells, periodic, lattice_constant=1.0):
        L = lib()
        basis = np.atleast_2d(np.asarray(basis, float))
        b_, bp = _d(np.asarray(bravais, float).reshape(9))
        s_, sp = _d(basis.reshape(-1))
        n_, npx = _i(n_cells)
        p_, pp = _i(periodic)
        h = C.c_void_p()
        _check(L.spin_geometry_create(bp, basis.shape[0], sp, npx, pp, float(lattice_constant), C.byref(h)))
        self._h = h
        self.n_basis = basis.shape[0]
        self.N = int(L.spin_system_nspins(h))
        self.n_images = 1

    def close(self):
        if getattr(self, "_h", None):
            lib().spin_system_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @classmethod
    def from_workload(cls, w, use_shell_helpers=False, stream=None, set_spins=True):
        s = cls(w.bravais, w.basis, w.n_cells, w.periodic, w.lattice_constant)
        if stream is not None:
            s.spin_set_stream(stream)
        s.hamiltonian_set_mu_s(w.mu_s)
        s.hamiltonian_set_field(w.B, w.B_dir)
        if w.aniso:
            s.hamiltonian_set_anisotropy([a[0] for a in w.aniso], [a[1] for a in w.aniso], [a[2] for a in w.aniso])
        if not use_shell_helpers:
            s.hamiltonian_set_pairs(w.pair_i, w.pair_j, w.pair_t, w.pair_J, w.pair_D)
        if len(w.quad_K):
            s.hamiltonian_set_quadruplets(w.quad_b, w.quad_t, w.quad_K)
        s.hamiltonian_set_ddi(w.ddi, w.ddi_images)
        s.llg_configure(w.dt_fs, w.alpha, w.T, w.seed, w.u, w.j_dir, w.beta)
        if set_spins:
            s.spins_set(w.initial_spins())
        return s

    # ---- C-ABI calls -----------------------------------------------------------------------------------
    def spin_set_stream(self, stream):
        """stream: int cudaStream_t handle (e.g. torch.cuda.current_stream().cuda_stream) or None."""
        _check(lib().spin_set_stream(self._h, C.c_void_p(int(stream) if stream else None)))

    def hamiltonian_set_mu_s(self, mu):
        a, p = _d(np.broadcast_to(np.asarray(mu, float), (self.n_basis,)))
        _check(lib().hamiltonian_set_mu_s(self._h, p))

    def hamiltonian_set_site_mu_s(self, mu_site):
        if mu_site is None:
            _check(lib().hamiltonian_set_site_mu_s(self._h, None))
            return
        a, p = _d(np.asarray(mu_site, float).reshape(self.N))
        _check(lib().hamiltonian_set_site_mu_s(self._h, p))

    def hamiltonian_set_field(self, B, direction):
        a, p = _d(direction)
        _check(lib().hamiltonian_set_field(self._h, float(B), p))

    def hamiltonian_set_anisotropy(self, basis_idx, K, axis):
        b, bp = _i(basis_idx)
        k, kp = _d(K)
        a, ap = _d(np.asarray(axis, float).reshape(-1))
        _check(lib().hamiltonian_set_anisotropy(self._h, len(b), bp, kp, ap))

    def hamiltonian_set_pairs(self, i, j, t, J, D=None):
        i_, ip = _i(i)
        j_, jp = _i(j)
        t_, tp = _i(np.asarray(t).reshape(-1))
        J_, Jp = _d(J)
        Dp = None
        if D is not None:
            D_, Dp = _d(np.asarray(D, float).reshape(-1))
        _check(lib().hamiltonian_set_pairs(self._h, len(i_), ip, jp, tp, Jp, Dp))

    def hamiltonian_set_exchange_shells(self, J):
        a, p = _d(J)
        _check(lib().hamiltonian_set_exchange_shells(self._h, len(a), p))

    def hamiltonian_set_dmi_shells(self, D, chirality):
        a, p = _d(D)
        _check(lib().hamiltonian_set_dmi_shells(self._h, len(a), p, int(chirality)))

    def hamiltonian_set_quadruplets(self, basis_ijkl, trans_jkl, K):
        b, bp = _i(np.asarray(basis_ijkl).reshape(-1))
        t, tp = _i(np.asarray(trans_jkl).reshape(-1))
        k, kp = _d(K)
        _check(lib().hamiltonian_set_quadruplets(self._h, len(k), bp, tp, kp))

    def hamiltonian_set_ddi(self, enabled, n_images=(0, 0, 0)):
        n, p = _i(n_images)
        _check(lib().hamiltonian_set_ddi(self._h, int(bool(enabled)), p))

    def spins_set(self, n):
        a, p = _d(np.asarray(n, float).reshape(-1))
        if a.size != 3 * self.N:
            raise ValueError("spins_set expects 3N doubles")
        _check(lib().spins_set(self._h, p))

    def spins_get(self, out=None):
        out = np.empty((self.N, 3)) if out is None else out
        _check(lib().spins_get(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def spins_set_device(self, dev_ptr):
        _check(lib().spins_set_device(self._h, C.c_void_p(int(dev_ptr))))

    def spins_get_device(self, dev_ptr):
        _check(lib().spins_get_device(self._h, C.c_void_p(int(dev_ptr))))

    def llg_configure(self, dt_fs, alpha, T=0.0, seed=0, u=0.0, j_dir=(1, 0, 0), beta=0.0):
        j, jp = _d(j_dir)
        _check(lib().llg_configure(self._h, float(dt_fs), float(alpha), float(T), int(seed), float(u), jp, float(beta)))

    def gneb_forces(self, kappa=1.0, climbing=-1):
        """Returns (F (M, N, 3), E (M,), l (M,)) of the chain held in the batched images."""
        M = self.n_images
        F = np.zeros((M, self.N, 3)); E = np.zeros(M); l = np.zeros(M)
        P_ = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
        _check(lib().gneb_forces(self._h, float(kappa), int(climbing), P_(F), P_(E), P_(l)))
        return F, E, l

    def gneb_iterate(self, n_iterations, step, kappa=1.0, climbing=-1):
        _check(lib().gneb_iterate(self._h, int(n_iterations), float(step), float(kappa), int(climbing)))

    def spin_set_images(self, n_images):
        self.n_images = int(n_images)
        _check(lib().spin_set_images(self._h, int(n_images)))

    def spin_select_image(self, image):
        _check(lib().spin_select_image(self._h, int(image)))

    def llg_set_image_temperatures(self, T):
        if T is None:
            _check(lib().llg_set_image_temperatures(self._h, None))
            return
        a = np.ascontiguousarray(np.asarray(T, dtype=np.float64).reshape(-1))
        _check(lib().llg_set_image_temperatures(self._h, a.ctypes.data_as(C.POINTER(C.c_double))))

    def spin_measure_fp64_tflops(self):
        v = C.c_double(0.0)
        _check(lib().spin_measure_fp64_tflops(self._h, C.byref(v)))
        return float(v.value)

    def minimise_vp(self, n_iterations, dt, mass=1.0):
        _check(lib().minimise_vp(self._h, int(n_iterations), float(dt), float(mass)))

    def minimise_vp_reset(self):
        _check(lib().minimise_vp_reset(self._h))

    def spins_set_pinned(self, mask):
        """mask: N flags (boundary order) or None.  Pinned spins never move; a pinned zero vector is a vacancy."""
        if mask is None:
            _check(lib().spins_set_pinned(self._h, None))
            return
        m = np.ascontiguousarray(np.asarray(mask).astype(np.uint8).reshape(-1))
        if m.size != self.N:
            raise ValueError("mask must have N entries")
        _check(lib().spins_set_pinned(self._h, m.ctypes.data_as(C.c_void_p)))

    def topological_charge(self):
        q = C.c_double(0.0)
        _check(lib().topological_charge(self._h, C.byref(q)))
        return float(q.value)

    def topological_charge_noalloc(self, d_out_ptr):
        """Q into the DEVICE double at address `d_out_ptr` (e.g. tensor.data_ptr()); asynchronous on the system's stream; allocates nothing."""
        _check(lib().topological_charge_noalloc(self._h, C.c_void_p(int(d_out_ptr))))

    def llg_set_damping_only(self, enabled):
        _check(lib().llg_set_damping_only(self._h, int(bool(enabled))))

    def llg_set_solver(self, solver):
        """0 Depondt, 1 Heun, 2 SIB (include/spinllg.h SPIN_SOLVER_*)."""
        _check(lib().llg_set_solver(self._h, int(solver)))

    def llg_iterate(self, n_steps):
        _check(lib().llg_iterate(self._h, int(n_steps)))

    def llg_get_step(self):
        v = C.c_uint64(0)
        _check(lib().llg_get_step(self._h, C.byref(v)))
        return int(v.value)

    def llg_set_step(self, step):
        _check(lib().llg_set_step(self._h, int(step)))

    def spin_synchronize(self):
        _check(lib().spin_synchronize(self._h))

    def effective_field(self, out=None):
        out = np.empty((self.N, 3)) if out is None else out
        _check(lib().effective_field(self._h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def effective_field_device(self, dev_ptr):
        _check(lib().effective_field_device(self._h, C.c_void_p(int(dev_ptr))))

    def energy(self):
        tot = C.c_double(0.0)
        terms = np.zeros(6)
        _check(lib().energy(self._h, C.byref(tot), terms.ctypes.data_as(C.POINTER(C.c_double))))
        return float(tot.value), terms

    def observables(self):
        M = np.zeros(3)
        mt = C.c_double(0.0)
        _check(lib().observables(self._h, M.ctypes.data_as(C.POINTER(C.c_double)), C.byref(mt)))
        return M, float(mt.value)

    # ---- slab decomposition (device pointers and streams are plain integers here: torch's data_ptr() / cuda_stream)
    def spin_set_slab(self, enabled, c_offset=0, global_cells_c=0, global_periodic_c=0):
        _check(lib().spin_set_slab(self._h, int(bool(enabled)), int(c_offset), int(global_cells_c), int(bool(global_periodic_c))))

    def spin_halo_doubles(self):
        """(doubles per side of the halo, reach along c in planes)"""
        n, r = C.c_int64(0), C.c_int(0)
        _check(lib().spin_halo_doubles(self._h, C.byref(n), C.byref(r)))
        return int(n.value), int(r.value)

    def spin_halo_get(self, array, side, dst_device_ptr, stream=0):
        _check(lib().spin_halo_get(self._h, int(array), int(side), C.c_void_p(int(dst_device_ptr)), C.c_void_p(int(stream) or None)))

    def spin_halo_put(self, array, side, src_device_ptr, stream=0):
        _check(lib().spin_halo_put(self._h, int(array), int(side), C.c_void_p(int(src_device_ptr)), C.c_void_p(int(stream) or None)))

    def llg_slab_sweep(self, stage, part=0):
        _check(lib().llg_slab_sweep(self._h, int(stage), int(part)))

    def llg_slab_step(self, part=0):
        _check(lib().llg_slab_step(self._h, int(part)))

    def llg_slab_step_fused(self, peer_lo_next, peer_lo_cells_c, peer_hi_next):
        """peer_*_next: device addresses (int) of the neighbours' next-configuration arrays, or None at an open end"""
        _check(lib().llg_slab_step_fused(self._h, C.c_void_p(peer_lo_next or None), int(peer_lo_cells_c), C.c_void_p(peer_hi_next or None)))

    def spin_slab_arrays(self):
        """(current, next): device addresses of the configuration arrays (they swap at every llg_slab_advance)"""
        a, b = C.c_void_p(0), C.c_void_p(0)
        _check(lib().spin_slab_arrays(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def spin_slab_flags(self):
        """device address of the slab's two step flags ([0] written by the lower, [1] by the upper neighbour)"""
        p = C.c_void_p(0)
        _check(lib().spin_slab_flags(self._h, C.byref(p)))
        return int(p.value)

    def spin_flag_signal(self, flag_addr, value):
        _check(lib().spin_flag_signal(self._h, C.c_void_p(int(flag_addr)), int(value)))

    def spin_flag_wait(self, flag_addr, value):
        _check(lib().spin_flag_wait(self._h, C.c_void_p(int(flag_addr)), int(value)))

    def llg_slab_advance(self):
        _check(lib().llg_slab_advance(self._h))

    def spin_launch_counts(self):
        a, b = C.c_int64(0), C.c_int64(0)
        _check(lib().spin_launch_counts(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def spin_profile_enable(self, on=True):
        _check(lib().spin_profile_enable(self._h, int(bool(on))))

    def spin_profile_get(self, kind):
        ms, n = C.c_double(0.0), C.c_int64(0)
        _check(lib().spin_profile_get(self._h, int(kind), C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def spin_set_option(self, name, value):
        _check(lib().spin_set_option(self._h, name.encode(), int(value)))

    def spin_kernel_info(self):
        buf = C.create_string_buffer(1024)
        _check(lib().spin_kernel_info(self._h, buf, 1024))
        return buf.value.decode()

    def spin_ddi_info(self):
        buf = C.create_string_buffer(64)
        _check(lib().spin_ddi_info(self._h, buf, 64))
        return buf.value.decode()

    def spin_jit_source(self, compile=False):
        buf = C.create_string_buffer(1 << 18)
        nbytes = C.c_int64(0)
        _check(lib().spin_jit_source(self._h, buf, 1 << 18, int(bool(compile)), C.byref(nbytes)))
        return buf.value.decode(), int(nbytes.value)


def version() -> str:
    return lib().spin_version().decode()


def spin_jit_compiler_info() -> str:
    buf = C.create_string_buffer(1024)
    _check(lib().spin_jit_compiler_info(buf, 1024))
    return buf.value.decode()


def spin_ipc_export(device_addr):
    """(64-byte CUDA IPC handle, offset) of the allocation that holds the device address: picklable, for the neighbour's process"""
    h = C.create_string_buffer(64)
    off = C.c_int64(0)
    _check(lib().spin_ipc_export(C.c_void_p(int(device_addr)), h, C.byref(off)))
    return bytes(h.raw), int(off.value)


def spin_ipc_open(handle, offset):
    """device address in THIS process of what another process exported"""
    p = C.c_void_p(0)
    _check(lib().spin_ipc_open(C.c_char_p(bytes(handle)), int(offset), C.byref(p)))
    return int(p.value)


def spin_ipc_close(device_addr, offset):
    _check(lib().spin_ipc_close(C.c_void_p(int(device_addr)), int(offset)))

