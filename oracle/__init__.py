"""ctypes front end of the CPU oracle (oracle/spin_oracle.c).

TEST INFRASTRUCTURE ONLY -- the oracle is the independent checker written from the paper (arXiv 1901.11350,
/root/reference/PAPER.md).  Only tests/, bench.py's `cpu_baseline` / `--impl reference` legs and
`__graft_entry__.smoke()` may import this package; the product (paper_1901_11350_b200) never does.
All arithmetic lives in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MU_B = 0.057883818060      # meV/T   (CODATA 2018)
K_B = 0.08617333262        # meV/K
GAMMA = 0.176085963023     # rad/(ps T)
C_DD = 0.0536815112        # meV, mu0 mu_B^2 / (4 pi Angstrom^3)

T_ZEE, T_ANI, T_EXC, T_DMI, T_QUAD, T_DDI, T_ALL = 1, 2, 4, 8, 16, 32, 63

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.orc_create.restype = vp
        L.orc_create.argtypes = [dp, C.c_int, dp, ip, ip, C.c_double]
        L.orc_destroy.argtypes = [vp]
        L.orc_nspins.restype = C.c_long
        L.orc_nspins.argtypes = [vp]
        L.orc_threads.restype = C.c_int
        L.orc_threads.argtypes = [vp]
        L.orc_set_threads.argtypes = [vp, C.c_int]
        L.orc_set_mu_s.argtypes = [vp, dp]
        L.orc_set_site_mu_s.argtypes = [vp, dp]
        L.orc_set_field.argtypes = [vp, C.c_double, dp]
        L.orc_set_anisotropy.argtypes = [vp, C.c_int, ip, dp, dp]
        L.orc_set_pairs.argtypes = [vp, C.c_int, ip, ip, ip, dp, dp]
        L.orc_set_quadruplets.argtypes = [vp, C.c_int, ip, ip, dp]
        L.orc_set_ddi.argtypes = [vp, C.c_int, ip, C.c_int]
        L.orc_set_spins.argtypes = [vp, dp]
        L.orc_get_spins.argtypes = [vp, dp]
        L.orc_llg_configure.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_double, dp, C.c_double]
        L.orc_get_step.restype = C.c_uint64
        L.orc_get_step.argtypes = [vp]
        L.orc_set_step.argtypes = [vp, C.c_uint64]
        L.orc_energy.argtypes = [vp, dp, dp]
        L.orc_energy_ddi_pairsum.restype = C.c_double
        L.orc_energy_ddi_pairsum.argtypes = [vp, dp]
        L.orc_gradient.argtypes = [vp, dp, dp, C.c_int]
        L.orc_gradient_scatter.argtypes = [vp, dp, dp, C.c_int]
        L.orc_ddi_direct.argtypes = [vp, dp, dp]
        L.orc_ddi_fft.argtypes = [vp, dp, dp]
        L.orc_fft3d.argtypes = [dp, ip, C.c_int]
        L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_thermal_xi.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, dp]
        L.orc_thermal_xi_image.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, dp]
        L.orc_thermal_sigma.restype = C.c_double
        L.orc_thermal_sigma.argtypes = [vp, C.c_int]
        L.orc_stt_gradient.argtypes = [vp, dp, dp]
        L.orc_llg_step.argtypes = [vp]
        L.orc_llg_iterate.argtypes = [vp, C.c_long]
        L.orc_heun_step.argtypes = [vp]
        L.orc_set_solver.argtypes = [vp, C.c_int]
        L.orc_set_image.argtypes = [vp, C.c_uint32]
        L.orc_set_damping_only.argtypes = [vp, C.c_int]
        L.orc_gneb_forces.argtypes = [vp, C.c_int, dp, C.c_double, C.c_int, dp, dp, dp]
        L.orc_gneb_iterate.argtypes = [vp, C.c_int, dp, C.c_long, C.c_double, C.c_double, C.c_int]
        L.orc_geodesic_distance.argtypes = [vp, dp, dp]
        L.orc_geodesic_distance.restype = C.c_double
        L.orc_set_pinned.argtypes = [vp, C.c_void_p]
        L.orc_vp_iterate.argtypes = [vp, C.c_long, C.c_double, C.c_double]
        L.orc_vp_reset.argtypes = [vp]
        L.orc_topological_charge.argtypes = [vp, dp]
        L.orc_topological_charge.restype = C.c_double
        L.orc_spherical_area.argtypes = [dp, dp, dp]
        L.orc_spherical_area.restype = C.c_double
        L.orc_effective_field.argtypes = [vp, dp]
        L.orc_observables.argtypes = [vp, dp, dp]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int))


class OracleSystem:
    """One spin system in the oracle.  Arrays are (N,3) float64 in boundary index order."""

    def __init__(self, bravais, basis, n_cells, periodic, lattice_constant=1.0):
        L = lib()
        basis = np.atleast_2d(np.asarray(basis, float))
        self.n_basis = basis.shape[0]
        self.n_cells = tuple(int(x) for x in n_cells)
        self.periodic = tuple(int(x) for x in periodic)
        b_, bp = _d(np.asarray(bravais, float).reshape(9))
        s_, sp = _d(basis.reshape(-1))
        n_, np_ = _i(self.n_cells)
        p_, pp = _i(self.periodic)
        self._h = C.c_void_p(L.orc_create(bp, self.n_basis, sp, np_, pp, float(lattice_constant)))
        self.N = int(L.orc_nspins(self._h))

    def __del__(self):
        try:
            if self._h:
                lib().orc_destroy(self._h)
                self._h = None
        except Exception:
            pass

    @classmethod
    def from_workload(cls, w, ddi_direct=False):
        s = cls(w.bravais, w.basis, w.n_cells, w.periodic, w.lattice_constant)
        s.set_mu_s(w.mu_s)
        s.set_field(w.B, w.B_dir)
        if w.aniso:
            s.set_anisotropy([a[0] for a in w.aniso], [a[1] for a in w.aniso], [a[2] for a in w.aniso])
        s.set_pairs(w.pair_i, w.pair_j, w.pair_t, w.pair_J, w.pair_D)
        if len(w.quad_K):
            s.set_quadruplets(w.quad_b, w.quad_t, w.quad_K)
        s.set_ddi(w.ddi, w.ddi_images, direct=ddi_direct)
        s.llg_configure(w.dt_fs, w.alpha, w.T, w.seed, w.u, w.j_dir, w.beta)
        s.set_spins(w.initial_spins())
        return s

    # ---- setters
    def set_threads(self, n):
        lib().orc_set_threads(self._h, int(n))

    @property
    def threads(self):
        return int(lib().orc_threads(self._h))

    def set_mu_s(self, mu):
        a, p = _d(np.broadcast_to(np.asarray(mu, float), (self.n_basis,)))
        lib().orc_set_mu_s(self._h, p)

    def set_site_mu_s(self, mu_site):
        """Per-site moments (PAPER.md:79 'atoms of different types'), N values in boundary order; None clears."""
        if mu_site is None:
            lib().orc_set_site_mu_s(self._h, None)
            return
        a, p = _d(np.asarray(mu_site, float).reshape(self.N))
        lib().orc_set_site_mu_s(self._h, p)

    def set_field(self, B, direction):
        a, p = _d(direction)
        lib().orc_set_field(self._h, float(B), p)

    def set_anisotropy(self, basis_idx, K, axis):
        b, bp = _i(basis_idx)
        k, kp = _d(K)
        a, ap = _d(np.asarray(axis, float).reshape(-1))
        lib().orc_set_anisotropy(self._h, len(b), bp, kp, ap)

    def set_pairs(self, i, j, t, J, D=None):
        i_, ip = _i(i)
        j_, jp = _i(j)
        t_, tp = _i(np.asarray(t).reshape(-1))
        J_, Jp = _d(J)
        if D is None:
            D = np.zeros((len(i_), 3))
        D_, Dp = _d(np.asarray(D, float).reshape(-1))
        lib().orc_set_pairs(self._h, len(i_), ip, jp, tp, Jp, Dp)

    def set_quadruplets(self, basis_ijkl, trans_jkl, K):
        b, bp = _i(np.asarray(basis_ijkl).reshape(-1))
        t, tp = _i(np.asarray(trans_jkl).reshape(-1))
        k, kp = _d(K)
        lib().orc_set_quadruplets(self._h, len(k), bp, tp, kp)

    def set_ddi(self, enabled, n_images=(0, 0, 0), direct=False):
        n, p = _i(n_images)
        lib().orc_set_ddi(self._h, int(bool(enabled)), p, int(bool(direct)))

    def llg_configure(self, dt_fs, alpha, T=0.0, seed=0, u=0.0, j_dir=(1, 0, 0), beta=0.0):
        j, jp = _d(j_dir)
        lib().orc_llg_configure(self._h, float(dt_fs), float(alpha), float(T), int(seed), float(u), jp, float(beta))

    def set_spins(self, n):
        a, p = _d(np.asarray(n, float).reshape(-1))
        assert a.size == 3 * self.N
        lib().orc_set_spins(self._h, p)

    # ---- getters / computations
    def spins(self):
        out = np.empty((self.N, 3))
        lib().orc_get_spins(self._h, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    @property
    def step(self):
        return int(lib().orc_get_step(self._h))

    @step.setter
    def step(self, v):
        lib().orc_set_step(self._h, int(v))

    def energy_terms(self, n=None):
        """(Zeeman, anisotropy, exchange, DMI, quadruplet, DDI) in meV, from the sums of Eq. 1 / Eq. 2."""
        a, p = _d(self.spins() if n is None else np.asarray(n, float).reshape(-1))
        out = np.zeros(6)
        lib().orc_energy(self._h, p, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def energy(self, n=None):
        return float(self.energy_terms(n).sum())

    def energy_ddi_pairsum(self, n=None):
        a, p = _d(self.spins() if n is None else np.asarray(n, float).reshape(-1))
        return float(lib().orc_energy_ddi_pairsum(self._h, p))

    def gradient(self, n=None, mask=T_ALL, scatter=False):
        """F = -dH/dn (meV), (N,3)."""
        a, p = _d(self.spins() if n is None else np.asarray(n, float).reshape(-1))
        out = np.zeros((self.N, 3))
        fn = lib().orc_gradient_scatter if scatter else lib().orc_gradient
        fn(self._h, p, out.ctypes.data_as(C.POINTER(C.c_double)), int(mask))
        return out

    def ddi_field(self, n=None, direct=False):
        a, p = _d(self.spins() if n is None else np.asarray(n, float).reshape(-1))
        out = np.zeros((self.N, 3))
        fn = lib().orc_ddi_direct if direct else lib().orc_ddi_fft
        fn(self._h, p, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def stt_gradient(self, n=None):
        a, p = _d(self.spins() if n is None else np.asarray(n, float).reshape(-1))
        out = np.zeros((self.N, 3))
        lib().orc_stt_gradient(self._h, p, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def thermal_sigma(self, b=0):
        return float(lib().orc_thermal_sigma(self._h, int(b)))

    def effective_field(self):
        out = np.zeros((self.N, 3))
        lib().orc_effective_field(self._h, out.ctypes.data_as(C.POINTER(C.c_double)))
        return out

    def observables(self):
        M = np.zeros(3)
        mt = C.c_double(0.0)
        lib().orc_observables(self._h, M.ctypes.data_as(C.POINTER(C.c_double)), C.byref(mt))
        return M, float(mt.value)

    def iterate(self, n_steps):
        lib().orc_llg_iterate(self._h, int(n_steps))

    def topological_charge(self, n=None):
        """Q of App. A summed over the a-b planes (one basis atom)."""
        a, p = _d(self.spins() if n is None else n)
        return float(lib().orc_topological_charge(self._h, p))

    def vp_iterate(self, n_iter, dt, mass=1.0):
        """Velocity-projection minimiser, App. D; velocity and previous force persist between calls (vp_reset clears them)."""
        lib().orc_vp_iterate(self._h, int(n_iter), float(dt), float(mass))

    def vp_reset(self):
        lib().orc_vp_reset(self._h)

    def set_pinned(self, mask):
        """mask: N flags (boundary order) or None.  Pinned spins never move; a pinned zero vector is a vacancy."""
        if mask is None:
            lib().orc_set_pinned(self._h, None)
            return
        m = np.ascontiguousarray(np.asarray(mask).astype(np.uint8).reshape(-1))
        assert m.size == self.N
        lib().orc_set_pinned(self._h, m.ctypes.data_as(C.c_void_p))

    def gneb_forces(self, chain, kappa=1.0, climbing=-1):
        """chain: (M, N, 3).  Returns (F (M, N, 3), E (M,), l (M,) with l[nu] = geodesic distance nu -> nu+1)."""
        ch = np.ascontiguousarray(np.asarray(chain, float)); M = ch.shape[0]
        F = np.zeros_like(ch); E = np.zeros(M); l = np.zeros(M)
        P = lambda a: a.ctypes.data_as(C.POINTER(C.c_double))
        lib().orc_gneb_forces(self._h, M, P(ch), float(kappa), int(climbing), P(F), P(E), P(l))
        return F, E, l

    def gneb_iterate(self, chain, n_iter, step, kappa=1.0, climbing=-1):
        ch = np.ascontiguousarray(np.asarray(chain, float)).copy(); M = ch.shape[0]
        lib().orc_gneb_iterate(self._h, M, ch.ctypes.data_as(C.POINTER(C.c_double)), int(n_iter), float(step), float(kappa), int(climbing))
        return ch

    def geodesic_distance(self, a, b):
        (x, px), (y, py) = _d(a), _d(b)
        return float(lib().orc_geodesic_distance(self._h, px, py))

    def set_damping_only(self, on):
        """Drop the precession term of Eq. 10: the LLG solvers then minimise the energy."""
        lib().orc_set_damping_only(self._h, int(bool(on)))

    def set_image(self, image):
        """Noise stream of image `image` (independent images of one batched system; 0 = single system)."""
        lib().orc_set_image(self._h, int(image))

    def set_solver(self, solver):
        """0 Depondt (App. B B5-B7), 1 Heun (B3-B4), 2 SIB semi-implicit midpoint (App. C)."""
        lib().orc_set_solver(self._h, int(solver))

    def heun_step(self):
        lib().orc_heun_step(self._h)


def spherical_area(ni, nj, nk):
    (a, pa), (b, pb), (c, pc) = _d(ni), _d(nj), _d(nk)
    return float(lib().orc_spherical_area(pa, pb, pc))


def philox4x32_10(counter, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in counter])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def thermal_xi(seed, step, spin, image=0):
    out = np.zeros(3)
    if image == 0:
        lib().orc_thermal_xi(int(seed), int(step), int(spin), out.ctypes.data_as(C.POINTER(C.c_double)))
    else:
        lib().orc_thermal_xi_image(int(seed), int(step), int(spin), int(image), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out


def fft3d(z, sign):
    """In-place style helper for the FFT pin: z complex array of shape (P2,P1,P0) (x fastest)."""
    z = np.ascontiguousarray(z, dtype=np.complex128)
    P = np.array(z.shape[::-1], np.int32)
    buf = z.view(np.float64).reshape(-1).copy()
    lib().orc_fft3d(buf.ctypes.data_as(C.POINTER(C.c_double)), P.ctypes.data_as(C.POINTER(C.c_int)), int(sign))
    return buf.view(np.complex128).reshape(z.shape)
