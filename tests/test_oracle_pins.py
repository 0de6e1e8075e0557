"""Pins of the CPU oracle against what the paper prints and what mathematics fixes.

None of these tests touches the CUDA path.  Each pin is chosen so that a plausible mistake in the oracle
(dropped term, wrong sign or index, transposed operand, wrong unit) fails at least one of them.
"""
import dataclasses
import json
import math
import os

import numpy as np
import pytest

import oracle as O
from oracle import OracleSystem
import workloads as W

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.json")))


def small(cfg, cells, steps=None):
    return W.CONFIGS[cfg]().resized(cells, steps)


def rand_spins(N, seed):
    v = np.random.default_rng(seed).standard_normal((N, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


# ------------------------------------------------------------------ O1 ferromagnetic closed forms
@pytest.mark.parametrize("cfg,cells,z_J", [
    (1, (8, 6, 1), [(4, 1.0)]),
    (2, (12, 10, 1), [(6, 1.0), (6, -0.3), (6, -0.1)]),
    (3, (6, 5, 4), [(6, 1.0)]),
])
def test_O1_ferromagnet_closed_form(cfg, cells, z_J):
    """All n = z, periodic: E = -N (mu_s mu_B B + K + 1/2 sum_shells z J), DMI energy 0, F uniform.
    Pins Eq. 1, readings R3, R4 (unique pairs, :69)."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w)
    n = np.tile([0.0, 0.0, 1.0], (s.N, 1))
    E = s.energy_terms(n)
    K = w.aniso[0][1] if w.aniso else 0.0
    mu = w.mu_s[0] * O.MU_B
    assert E[0] == pytest.approx(-s.N * mu * w.B, rel=1e-13)
    assert E[1] == pytest.approx(-s.N * K, rel=1e-13, abs=1e-13)
    assert E[2] == pytest.approx(-s.N * 0.5 * sum(z * J for z, J in z_J), rel=1e-13)
    assert abs(E[3]) < 1e-10
    F = s.gradient(n)
    Fz = mu * w.B + 2 * K + sum(z * J for z, J in z_J)
    assert np.allclose(F[:, 2], Fz, rtol=1e-13)
    # DMI contributions of +t and -t partners cancel for a uniform state
    assert np.abs(F[:, :2]).max() < 1e-13


def test_O1_honeycomb_ferromagnet_with_quadruplets():
    """cfg4 lattice, all n = z: per cell E_exc = -(3*(-2) + 6*0.5) = 3, E_quad = -2*K4 = 0.4, E_ani = -2*K = 0.2."""
    w = small(4, (6, 4, 1))
    s = OracleSystem.from_workload(w)
    n = np.tile([0.0, 0.0, 1.0], (s.N, 1))
    E = s.energy_terms(n)
    ncell = 24
    assert E[2] == pytest.approx(3.0 * ncell, rel=1e-13)
    assert E[4] == pytest.approx(0.4 * ncell, rel=1e-13)
    assert E[1] == pytest.approx(0.2 * ncell, rel=1e-13)
    assert E[0] == 0.0


def test_tc_constant_pins_kB():
    """T_c = 1.44 J/k_B = 16.71 K at J = 1 meV fixes k_B in meV/K."""
    g = GOLD["tc_simple_cubic"]
    assert g["J_over_kB"] * 1.0 / O.K_B == pytest.approx(g["kelvin_for_J_1meV"], abs=0.005)


# ------------------------------------------------------------------ O2 damped Larmor precession, Eq. 12
def _larmor_error(dt_fs, alpha, method, t_ps=100.0, mu_s=2.0, B=1.0):
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
    s.set_mu_s([mu_s]); s.set_field(B, (0, 0, 1)); s.llg_configure(dt_fs, alpha)
    s.set_spins([[1.0, 0.0, 0.0]])
    gp = O.GAMMA / (1 + alpha * alpha)
    err, dev = 0.0, 0.0
    for k in range(int(round(t_ps / (dt_fs * 1e-3)))):
        if method == "heun_standalone":
            s.heun_step()
        else:
            s.set_solver({"depondt": 0, "heun": 1, "sib": 2, "rk4": 3}[method]); s.iterate(1)
        t = (k + 1) * dt_fs * 1e-3
        nz = math.tanh(alpha * gp * B * t)
        ph = gp * B * t
        ex = np.array([math.cos(ph) * math.sqrt(1 - nz * nz), math.sin(ph) * math.sqrt(1 - nz * nz), nz])
        n = s.spins()[0]
        err = max(err, np.abs(n - ex).max())
        dev = max(dev, abs(np.linalg.norm(n) - 1))
    return err, dev


def test_O2_larmor_depondt_matches_paper_error():
    """Eq. 12; the paper prints the Depondt error ~3e-7 at B=1 T, alpha=0.1, dt=10 fs (:166).
    A wrong sign of gamma, a missing 1/(1+alpha^2), rotating n^p instead of n(t) (R8) or a non-Stratonovich
    predictor changes this number by orders of magnitude."""
    g = GOLD["larmor_depondt_error"]
    err, dev = _larmor_error(g["dt_fs"], g["alpha"], "depondt")
    assert abs(err - g["value"]) < g["rel_window"] * g["value"], err
    assert dev < 5e-16
    err_half, _ = _larmor_error(g["dt_fs"] / 2, g["alpha"], "depondt")
    assert err / err_half == pytest.approx(4.0, rel=0.1)          # second order


def test_O2_larmor_mu_independent_and_heun_order():
    e1, _ = _larmor_error(10.0, 0.1, "depondt", t_ps=20.0, mu_s=2.0)
    e2, _ = _larmor_error(10.0, 0.1, "depondt", t_ps=20.0, mu_s=5.0)
    assert e1 == pytest.approx(e2, rel=1e-6)                        # reading R2: mu cancels
    eh, _ = _larmor_error(10.0, 0.1, "heun")
    assert e1 < eh < 10 * GOLD["larmor_heun_error_order"]["value"]
    # the Heun branch of the general step (thermal field and current included) equals Heun written out on its own
    assert _larmor_error(10.0, 0.1, "heun_standalone")[0] == eh


def test_solvers_heun_and_sib_closed_forms():
    """Heun (App. B, B3-B4) and the semi-implicit midpoint solver SIB (App. C, C5-C11) against what mathematics fixes:
    second order on the damped Larmor problem of Eq. 12; SIB keeps |n| = 1 without renormalisation; and for alpha = 0 in a
    constant field both SIB stages see the same A, so one step is the Cayley rotation about the field by exactly
    2 atan(gamma B dt / 2) -- which pins the dt/2 in the skew matrix (reading R25) and the sense of rotation."""
    for m in ("heun", "sib"):
        e, dev = _larmor_error(10.0, 0.1, m, t_ps=20.0)
        eh, _ = _larmor_error(5.0, 0.1, m, t_ps=20.0)
        assert e / eh == pytest.approx(4.0, rel=0.15), (m, e, eh)
        assert e < 2e-5 and dev < 1e-14, (m, e, dev)
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
    B, dt_fs, steps = 3.0, 50.0, 40
    s.set_mu_s([2.0]); s.set_field(B, (0, 0, 1)); s.llg_configure(dt_fs, 0.0); s.set_solver(2)
    n0 = np.array([0.6, 0.0, 0.8])
    s.set_spins([n0]); s.iterate(steps)
    ph = steps * 2.0 * math.atan(O.GAMMA * B * dt_fs * 1e-3 / 2.0)       # Eq. 12 sense: phi grows with +gamma B t
    ex = np.array([0.6 * math.cos(ph), 0.6 * math.sin(ph), 0.8])
    assert np.abs(s.spins()[0] - ex).max() < 1e-14
    # no hidden renormalisation: a non-unit start keeps its length
    s.set_spins([1.5 * n0]); s.iterate(7)
    assert abs(np.linalg.norm(s.spins()[0]) - 1.5) < 1e-14


def test_solver_rk4_is_fourth_order():
    """"A 4th order Runge-Kutta solver": on the damped Larmor problem of Eq. 12 the error falls by 2^4 when the step
    is halved, and at dt = 10 fs it is orders below Heun's 1e-6 and Depondt's 3e-7 (:166)."""
    e1, dev = _larmor_error(40.0, 0.1, "rk4", t_ps=20.0)
    e2, _ = _larmor_error(20.0, 0.1, "rk4", t_ps=20.0)
    assert e1 / e2 == pytest.approx(16.0, rel=0.15), (e1, e2)
    e10, _ = _larmor_error(10.0, 0.1, "rk4", t_ps=20.0)
    assert e10 < 1e-10 and dev < 5e-16, (e10, dev)


@pytest.mark.parametrize("solver", [1, 2, 3])
def test_solvers_energy_decreases_and_split_invariance(solver):
    """alpha > 0, T = 0: the energy must not increase (Heun, SIB); with noise, iterate(a) + iterate(b) == iterate(a+b)."""
    w = small(3, (6, 6, 6))
    s = OracleSystem.from_workload(w); s.set_solver(solver)
    E = [s.energy()]
    for _ in range(6):
        s.iterate(50); E.append(s.energy())
    assert all(b <= a + 1e-10 * abs(a) for a, b in zip(E, E[1:])), E
    w2 = small(2, (8, 8, 1))
    a = OracleSystem.from_workload(w2); a.set_solver(solver); a.iterate(30)
    b = OracleSystem.from_workload(w2); b.set_solver(solver); b.iterate(11); b.iterate(19)
    assert np.array_equal(a.spins(), b.spins())


# ------------------------------------------------------------------ O3 gradient vs finite differences
def _fd_check(s, n, sites, h=1e-6, tol=5e-8):
    F = s.gradient(n)
    for i in sites:
        for k in range(3):
            npl, nmi = n.copy(), n.copy()
            npl[i, k] += h; nmi[i, k] -= h
            fd = -(s.energy(npl) - s.energy(nmi)) / (2 * h)
            assert abs(fd - F[i, k]) < tol * max(1.0, abs(F[i, k])), (i, k, fd, F[i, k])


@pytest.mark.parametrize("cfg,cells", [(1, (5, 4, 1)), (2, (6, 5, 1)), (3, (4, 3, 5)), (4, (4, 5, 1)), (5, (4, 3, 3))])
def test_O3_gradient_matches_finite_differences(cfg, cells):
    """F = -dH/dn against central differences of the energy sums, every term of Eq. 1/2,
    periodic and open edges, 1- and 2-atom basis, dipolar term via the direct sum."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w, ddi_direct=True)
    n = rand_spins(s.N, 10 + cfg)
    rng = np.random.default_rng(cfg)
    _fd_check(s, n, rng.choice(s.N, size=6, replace=False))


def test_O3_fd_three_site_and_biquadratic_quadruplets():
    """Quadruplets with repeated sites (4-spin-2-site and 3-site): product rule over roles."""
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (4, 3, 1), (1, 0, 0))
    qb = [[0, 0, 0, 0], [0, 0, 0, 0]]
    qt = [[1, 0, 0, 0, 0, 0, 1, 0, 0],      # (i, i+a, i, i+a): bi-quadratic
          [1, 0, 0, 0, 0, 0, 0, 1, 0]]      # (i, i+a, i, i+b): three sites
    s.set_quadruplets(qb, qt, [0.7, -0.4])
    n = rand_spins(s.N, 3)
    _fd_check(s, n, range(s.N))
    assert np.allclose(s.gradient(n), s.gradient(n, scatter=True), rtol=0, atol=1e-14)


# ------------------------------------------------------------------ gather form == scatter form
@pytest.mark.parametrize("cfg,cells", [(1, (5, 4, 1)), (2, (7, 5, 1)), (3, (3, 4, 5)), (4, (5, 3, 1)), (5, (5, 4, 3))])
def test_gather_equals_scatter(cfg, cells):
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w, ddi_direct=True)
    n = rand_spins(s.N, 77)
    a, b = s.gradient(n), s.gradient(n, scatter=True)
    assert np.abs(a - b).max() < 1e-13 * np.abs(a).max()


def test_open_edges_by_explicit_site_loop():
    """Reading R20: a bond whose partner is off an open edge does not exist.  Energy recomputed here by an
    explicit loop over sites in plain Python for a 4x3 open square lattice."""
    J, Dv = 1.3, np.array([0.2, -0.1, 0.4])
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (4, 3, 1), (0, 0, 0))
    s.set_pairs([0, 0], [0, 0], [[1, 0, 0], [0, 1, 0]], [J, J], [Dv, Dv])
    n = rand_spins(12, 5)
    e_exc = e_dmi = 0.0
    for y in range(3):
        for x in range(4):
            i = x + 4 * y
            for dx, dy in ((1, 0), (0, 1)):
                if x + dx < 4 and y + dy < 3:
                    j = (x + dx) + 4 * (y + dy)
                    e_exc -= J * n[i] @ n[j]
                    e_dmi -= Dv @ np.cross(n[i], n[j])
    E = s.energy_terms(n)
    assert E[2] == pytest.approx(e_exc, rel=1e-13)
    assert E[3] == pytest.approx(e_dmi, rel=1e-13)


# ------------------------------------------------------------------ O4 Euler identity per term
@pytest.mark.parametrize("cfg,cells", [(2, (6, 5, 1)), (4, (5, 4, 1)), (5, (4, 4, 2))])
def test_O4_euler_identity(cfg, cells):
    """E_k = -(1/k) sum_i n_i.F_i^(k): k=1 Zeeman, 2 anisotropy/exchange/DMI/DDI, 4 quadruplets.
    Ties the normalisation of the gradient to the energy, term by term."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w, ddi_direct=True)
    n = rand_spins(s.N, 4)
    E = s.energy_terms(n)
    for idx, (mask, k) in enumerate([(O.T_ZEE, 1), (O.T_ANI, 2), (O.T_EXC, 2), (O.T_DMI, 2), (O.T_QUAD, 4), (O.T_DDI, 2)]):
        F = s.gradient(n, mask=mask)
        assert -(n * F).sum() / k == pytest.approx(E[idx], rel=1e-12, abs=1e-12), idx


# ------------------------------------------------------------------ O5 / O6 dipole-dipole
def test_fft_matches_library_and_inverts():
    rng = np.random.default_rng(0)
    for shape in [(4, 6, 8), (1, 5, 16), (3, 1, 7)]:
        z = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
        f = O.fft3d(z, -1)
        assert np.abs(f - np.fft.fftn(z)).max() < 1e-12
        assert np.abs(O.fft3d(f, +1) / z.size - z).max() < 1e-13


def test_O6_two_dipole_closed_forms():
    """Reading R1 (Eq. 1's dipolar term is garbled): textbook form. Two moments mu at distance r:
    head-to-tail E = -2 C_dd mu^2/r^3, side-by-side parallel E = +C_dd mu^2/r^3."""
    mu, a = 1.7, 2.5
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (2, 1, 1), (0, 0, 0), lattice_constant=a)
    s.set_mu_s([mu]); s.set_ddi(True, (0, 0, 0), direct=True)
    x = np.array([[1.0, 0, 0], [1.0, 0, 0]]); z = np.array([[0, 0, 1.0], [0, 0, 1.0]])
    c = O.C_DD * mu * mu / a ** 3
    assert s.energy_terms(x)[5] == pytest.approx(-2 * c, rel=1e-13)
    assert s.energy_terms(z)[5] == pytest.approx(+c, rel=1e-13)
    assert s.energy_ddi_pairsum(x) == pytest.approx(-2 * c, rel=1e-13)
    # field of dipole j at site i: along the axis 2 mu/r^3, perpendicular -mu/r^3 (times mu_i C_dd)
    assert np.allclose(s.ddi_field(x, direct=True)[0], [2 * c, 0, 0], rtol=1e-13, atol=1e-18)
    assert np.allclose(s.ddi_field(z, direct=True)[0], [0, 0, -c], rtol=1e-13, atol=1e-18)
    s.set_ddi(True, (0, 0, 0), direct=False)
    assert np.allclose(s.ddi_field(x), [[2 * c, 0, 0]] * 2, rtol=1e-12, atol=1e-16)


DDI_CASES = [
    # bravais, basis, cells, periodic, images
    (np.eye(3), [[0, 0, 0]], (4, 3, 2), (1, 1, 0), (2, 2, 0)),
    (np.eye(3), [[0, 0, 0]], (3, 3, 3), (0, 0, 0), (0, 0, 0)),
    (np.eye(3), [[0, 0, 0]], (4, 4, 1), (1, 1, 0), (3, 3, 0)),
    (np.array([[1, 0, 0], [0.5, 0.8, 0], [0.1, 0.2, 1.1]]), [[0, 0, 0], [0.31, 0.17, 0.23]], (3, 2, 2), (1, 0, 1), (1, 0, 2)),
    (W._TRI, [[0, 0, 0], [1 / 3, 1 / 3, 0.2]], (5, 3, 1), (0, 1, 0), (0, 2, 0)),
]


@pytest.mark.parametrize("case", range(len(DDI_CASES)))
def test_O5_ddi_fft_equals_direct_sum(case):
    """'compared to the direct evaluation of the sum for random configurations with spatially
    non-symmetric basis cells'.  Padded FFT convolution (R17, R18) == O(N^2) sum with the same image set (R16)."""
    brav, basis, cells, per, img = DDI_CASES[case]
    s = OracleSystem(brav, basis, cells, per, lattice_constant=1.3)
    s.set_mu_s(np.linspace(1.0, 2.5, len(basis)))
    s.set_ddi(True, img)
    n = rand_spins(s.N, case)
    Fd, Ff = s.ddi_field(n, direct=True), s.ddi_field(n, direct=False)
    assert np.abs(Fd - Ff).max() < 2e-13 * np.abs(Fd).max()
    # the energy from the printed double sum equals -1/2 sum n.F
    assert s.energy_ddi_pairsum(n) == pytest.approx(-0.5 * (n * Fd).sum(), rel=1e-12)


def test_O6_dipole_tensor_traceless():
    """sum_alpha F_alpha(all spins along alpha) = 0 at every site (Laplace: the tensor is traceless)."""
    s = OracleSystem(np.eye(3), [[0, 0, 0], [0.4, 0.3, 0.2]], (3, 3, 2), (1, 1, 0))
    s.set_ddi(True, (2, 2, 0))
    tr = np.zeros(s.N)
    for k in range(3):
        n = np.zeros((s.N, 3)); n[:, k] = 1.0
        tr += s.ddi_field(n)[:, k]
    scale = np.abs(s.ddi_field(np.tile([0, 0, 1.0], (s.N, 1)))).max()
    assert np.abs(tr).max() < 1e-12 * scale


def test_O6_monolayer_lattice_sum():
    """PAPER.md:89 'convergence of the stray field of a homogeneously magnetized monolayer against the analytically
    known result': square monolayer, all moments parallel; F_z = -S C_dd mu^2/a^3 out of plane, F_x = +S/2 ... in
    plane with S = 9.0336217.  The finite image set converges like 1/n_img: Richardson-extrapolated."""
    S_exact = GOLD["square_lattice_dipole_sum"]["value"]
    mu, a = 2.0, 1.5
    vals = {}
    for nimg in (100, 200):
        s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (1, 1, 0), lattice_constant=a)
        s.set_mu_s([mu]); s.set_ddi(True, (nimg, nimg, 0))
        fz = s.ddi_field(np.array([[0, 0, 1.0]]))[0, 2]
        fx = s.ddi_field(np.array([[1.0, 0, 0]]))[0, 0]
        assert fx == pytest.approx(-fz / 2, rel=1e-12)
        vals[nimg] = -fz / (O.C_DD * mu * mu / a ** 3)
    assert vals[100] < vals[200] < S_exact
    assert 2 * vals[200] - vals[100] == pytest.approx(S_exact, abs=2e-4)


# ------------------------------------------------------------------ O7 invariants of the Depondt step
@pytest.mark.parametrize("cfg,cells", [(1, (12, 12, 1)), (3, (8, 8, 8)), (5, (6, 6, 3))])
def test_O7_unit_length_and_energy_decrease(cfg, cells):
    """alpha > 0, T = 0, u = 0: |n_i| = 1 and the energy never increases (sampled)."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w, ddi_direct=False)
    E_prev = s.energy()
    for _ in range(10):
        s.iterate(20)
        n = s.spins()
        assert np.abs(np.linalg.norm(n, axis=1) - 1).max() < 4e-16
        E = s.energy()
        assert E <= E_prev + 1e-9 * abs(E_prev)
        E_prev = E


# ------------------------------------------------------------------ O8 spin spiral
def test_O8_spin_spiral_closed_form():
    """Chain along x, n_i = (0, cos q x_i, sin q x_i), D = D x: E/N = -J cos(qa) - D sin(qa) (R15 sign of D.(ni x nj))."""
    N, J, D, a = 24, 1.0, 0.37, 1.0
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (N, 1, 1), (1, 0, 0), lattice_constant=a)
    s.set_pairs([0], [0], [[1, 0, 0]], [J], [[D, 0, 0]])
    for m in (1, 3, -2):
        q = 2 * math.pi * m / (N * a)
        x = np.arange(N) * a
        n = np.stack([np.zeros(N), np.cos(q * x), np.sin(q * x)], axis=1)
        assert s.energy(n) / N == pytest.approx(-J * math.cos(q * a) - D * math.sin(q * a), rel=1e-12)


# ------------------------------------------------------------------ O9 / O10 thermal noise
def _philox_py(ctr, key):
    """Independent big-int restatement of Philox4x32-10 for cross-checking the C oracle."""
    c = list(ctr); k = list(key); M32 = 0xFFFFFFFF
    for r in range(10):
        if r:
            k = [(k[0] + 0x9E3779B9) & M32, (k[1] + 0xBB67AE85) & M32]
        p0, p1 = 0xD2511F53 * c[0], 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & M32, (p0 >> 32) ^ c[3] ^ k[1], p0 & M32]
    return tuple(c)


def test_O10_philox_known_answers_and_second_implementation():
    for v in GOLD["philox4x32_10_known_answers"]["vectors"]:
        ctr = [int(x, 16) for x in v["counter"]]; key = [int(x, 16) for x in v["key"]]
        out = tuple(int(x, 16) for x in v["output"])
        assert O.philox4x32_10(ctr, key) == out
        assert _philox_py(ctr, key) == out
    rng = np.random.default_rng(1)
    for _ in range(50):
        ctr = [int(x) for x in rng.integers(0, 2 ** 32, 4)]; key = [int(x) for x in rng.integers(0, 2 ** 32, 2)]
        assert O.philox4x32_10(ctr, key) == _philox_py(ctr, key)


def test_O10_thermal_xi_layout_and_moments():
    """Reading R13: key = seed, counter = (spin, block, step_lo, step_hi); 53-bit uniforms; Box-Muller."""
    seed, step, spin = 0x1234567890ABCDEF, (7 << 32) + 5, 4242
    xi = O.thermal_xi(seed, step, spin)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    def u(hi, lo):
        return ((((hi << 32) | lo) >> 11) + 0.5) * 2.0 ** -53
    x = _philox_py((spin, 0, step & 0xFFFFFFFF, step >> 32), key)
    r = math.sqrt(-2 * math.log(u(x[0], x[1])))
    assert xi[0] == pytest.approx(r * math.cos(2 * math.pi * u(x[2], x[3])), rel=1e-14)
    assert xi[1] == pytest.approx(r * math.sin(2 * math.pi * u(x[2], x[3])), rel=1e-14)
    x = _philox_py((spin, 1, step & 0xFFFFFFFF, step >> 32), key)
    assert xi[2] == pytest.approx(math.sqrt(-2 * math.log(u(x[0], x[1]))) * math.cos(2 * math.pi * u(x[2], x[3])), rel=1e-14)
    z = np.array([O.thermal_xi(9, st, sp) for st in range(40) for sp in range(500)])
    m = z.size
    assert abs(z.mean()) < 4 / math.sqrt(m)
    assert abs(z.var() - 1) < 4 * math.sqrt(2 / m)
    assert abs((z ** 4).mean() - 3) < 0.15
    c = np.corrcoef(z.T)
    assert np.abs(c - np.eye(3)).max() < 4 / math.sqrt(m / 3)


def test_O10_split_invariance():
    """iterate(a) + iterate(b) == iterate(a+b) bit for bit (counter-based noise keyed by the global step)."""
    w = small(2, (8, 8, 1))
    s1, s2 = OracleSystem.from_workload(w), OracleSystem.from_workload(w)
    s1.iterate(7); s1.iterate(5)
    s2.iterate(12)
    assert np.array_equal(s1.spins(), s2.spins())
    assert s1.step == s2.step == 12


def test_O9_langevin_magnetisation():
    """Decoupled moments in a field at temperature T: <n_z> = coth(x) - 1/x, x = mu B / k_B T.
    Pins Eq. 11's amplitude (R10: no extra 1/(1+alpha^2)), the 1/sqrt(dt) scaling (:160), the same noise in
    predictor and corrector (R11) and noise entering both precession and damping (R12)."""
    mu_s, B, T, alpha = 2.0, 30.0, 20.0, 0.5
    x = mu_s * O.MU_B * B / (O.K_B * T)
    L = 1 / math.tanh(x) - 1 / x
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (40, 40, 1), (0, 0, 0))
    s.set_mu_s([mu_s]); s.set_field(B, (0, 0, 1)); s.llg_configure(5.0, alpha, T=T, seed=11)
    s.set_spins(rand_spins(s.N, 1))
    s.iterate(400)                 # thermalise: relaxation time 1/(alpha gamma' B) ~ 0.5 ps = 100 steps
    acc = []
    for _ in range(60):
        s.iterate(40)
        acc.append(s.spins()[:, 2].mean())
    got = float(np.mean(acc))
    wrong = 1 / math.tanh(x * (1 + alpha ** 2)) - 1 / (x * (1 + alpha ** 2))    # what an extra 1/(1+alpha^2) would give
    assert abs(got - L) < 0.01, (got, L)
    assert abs(wrong - L) > 0.04


# ------------------------------------------------------------------ O11 spin-transfer torque
def test_O11_stt_gradient_exact_on_linear_fields():
    """(j.grad) of a field linear in position is exact for central differences, also on a skewed 2-atom lattice."""
    w = small(4, (7, 6, 1))
    s = OracleSystem(w.bravais, w.basis, w.n_cells, (0, 0, 0), 1.7)
    pos = dataclass_positions(w, 1.7)
    G = np.array([[0.3, -0.2, 0.0], [0.1, 0.5, 0.0], [-0.4, 0.25, 0.0]])      # n_k = G_k . r
    n = pos @ G.T
    for jdir in [(1, 0, 0), (0, 1, 0), (0.6, 0.8, 0)]:
        s.llg_configure(1.0, 0.1, u=1.0, j_dir=jdir)
        sg = s.stt_gradient(n)
        expect = G @ (np.array(jdir) / np.linalg.norm(jdir))
        assert np.allclose(sg, expect, rtol=0, atol=1e-12)


def dataclass_positions(w, alat):
    import dataclasses
    return dataclasses.replace(w, lattice_constant=alat).positions()


def test_O11_beta_equals_alpha_translates_rigidly():
    """No Hamiltonian, beta = alpha: Eq. 10 reduces to dn/dt = -u (j.grad) n, so a smooth profile moves
    at velocity u along j (Zhang-Li adiabatic limit).  Checks the signs and prefactors of both current terms.
    The residual is the O((a/w)^2) dispersion of the central difference: it must shrink ~8x when the profile
    is twice as wide (error after a fixed distance ~ third derivative ~ w^-3)."""
    N, u, alpha, steps = 256, 2.0, 0.3, 2500                      # 2.5 ps * 2 A/ps = 5 sites
    x = np.arange(N, dtype=float)

    def profile(x0, wdt):
        th = math.pi * np.exp(-(((x - x0 + N / 2) % N - N / 2) / wdt) ** 2)
        return np.stack([np.sin(th), np.zeros(N), np.cos(th)], axis=1)

    errs = {}
    for wdt in (12.0, 24.0):
        s = OracleSystem(np.eye(3), [[0, 0, 0]], (N, 1, 1), (1, 0, 0))
        s.llg_configure(1.0, alpha, u=u, j_dir=(1, 0, 0), beta=alpha)
        s.set_spins(profile(80.0, wdt))
        s.iterate(steps)
        errs[wdt] = np.abs(s.spins() - profile(80.0 + u * steps * 1e-3, wdt)).max()
        assert np.abs(s.spins() - profile(80.0, wdt)).max() > 0.2          # it did move
        assert np.abs(s.spins() - profile(80.0 - u * steps * 1e-3, wdt)).max() > 0.4   # and not backwards
    assert errs[24.0] < 3e-3
    assert errs[12.0] / errs[24.0] > 5.0


# ------------------------------------------------------------------ O12 perturbation growth (documents attainable parity)
@pytest.mark.parametrize("cfg,cells,steps", [(1, (16, 16, 1), 300), (2, (16, 16, 1), 300), (3, (8, 8, 8), 300), (4, (8, 8, 1), 300), (5, (8, 8, 2), 100)])
def test_O12_perturbation_growth_is_bounded(cfg, cells, steps):
    """Two oracle runs 1e-13 apart: the amplification over a few hundred steps stays far below the 1e-9/1e-16
    budget of the parity tolerance.  The full-length figures are in DESIGN.md."""
    w = small(cfg, cells, steps)
    a, b = OracleSystem.from_workload(w), OracleSystem.from_workload(w)
    n0 = w.initial_spins()
    d = np.random.default_rng(0).standard_normal(n0.shape) * 1e-13
    n1 = n0 + d
    n1 /= np.linalg.norm(n1, axis=1, keepdims=True)
    b.set_spins(n1)
    a.iterate(steps); b.iterate(steps)
    growth = np.abs(a.spins() - b.spins()).max() / np.abs(n1 - n0).max()
    assert growth < 1e3, growth


# ------------------------------------------------------------------ workloads: neighbour counts by brute force
@pytest.mark.parametrize("cfg,expected", [(1, {1.0: 4}), (2, {1.0: 6, math.sqrt(3): 6, 2.0: 6}), (3, {1.0: 6}),
                                          (4, {1 / math.sqrt(3): 3, 1.0: 6}), (5, {1.0: 6})])
def test_workload_pair_lists_are_complete_shells(cfg, expected):
    """Every listed pair sits on the stated shell and each shell is complete: coordination numbers recounted by
    brute force over all lattice vectors (z = 4 / 6,6,6 / 6 / 3+6 / 6)."""
    w = W.CONFIGS[cfg]()
    for b in range(w.n_basis):
        count = {}
        for p in range(len(w.pair_J)):
            r = (w.pair_t[p] + w.basis[w.pair_j[p]] - w.basis[w.pair_i[p]]) @ w.bravais
            d = round(float(np.linalg.norm(r)), 9)
            count[d] = count.get(d, 0) + (w.pair_i[p] == b) + (w.pair_j[p] == b)
        brute = {}
        rng3 = range(-3, 4)
        zr = rng3 if w.n_cells[2] > 1 else [0]
        for bj in range(w.n_basis):
            for ta in rng3:
                for tb in rng3:
                    for tc in zr:
                        r = (np.array([ta, tb, tc]) + w.basis[bj] - w.basis[b]) @ w.bravais
                        d = round(float(np.linalg.norm(r)), 9)
                        if d > 0:
                            brute[d] = brute.get(d, 0) + 1
        for dist, z in expected.items():
            dist = round(dist, 9)
            assert count[dist] == z == brute[dist], (cfg, b, dist, count, brute.get(dist))
        assert set(count) == {round(k, 9) for k in expected}


# ------------------------------------------------------------------ topological charge, App. A
def _girard_area(a, b, c):
    """Spherical excess (Girard): area = alpha + beta + gamma - pi from the corner angles -- independent of Eq. A2."""
    def corner(p, q, r):
        u = np.cross(p, q); v = np.cross(p, r)
        return math.acos(np.clip(np.dot(u, v) / (np.linalg.norm(u) * np.linalg.norm(v)), -1, 1))
    return corner(a, b, c) + corner(b, c, a) + corner(c, a, b) - math.pi


def test_topological_charge_spherical_triangle_area():
    """Eq. A2: one octant of the sphere has area 4 pi / 8; orientation gives the sign; random triangles
    agree with Girard's spherical excess."""
    x, y, z = np.eye(3)
    assert O.spherical_area(x, y, z) == pytest.approx(math.pi / 2, abs=1e-15)
    assert O.spherical_area(x, z, y) == pytest.approx(-math.pi / 2, abs=1e-15)
    rng = np.random.default_rng(11)
    for _ in range(200):
        t = rng.standard_normal((3, 3)); t /= np.linalg.norm(t, axis=1, keepdims=True)
        sgn = np.sign(np.dot(t[0], np.cross(t[1], t[2])))
        assert O.spherical_area(*t) == pytest.approx(sgn * _girard_area(*t), abs=1e-9)


@pytest.mark.parametrize("cfg,cells", [(1, (40, 40, 1)), (2, (36, 36, 1))])
def test_topological_charge_of_textures(cfg, cells):
    """Q = -1 for a skyrmion in a +z background, +1 for the antiskyrmion, 0 for the ferromagnet, additive,
    odd under n -> -n; an integer to rounding on a periodic lattice (Berg-Luescher)."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w)
    fm = np.tile([0.0, 0.0, 1.0], (w.n_spins, 1))
    assert s.topological_charge(fm) == 0.0
    pos = w.positions()
    ctr = pos[:, :2].mean(axis=0)
    sk = W.skyrmion_spins(w, 9.0)
    assert s.topological_charge(sk) == pytest.approx(-1.0, abs=1e-12)
    anti = sk * np.array([1.0, -1.0, 1.0])
    assert s.topological_charge(anti) == pytest.approx(+1.0, abs=1e-12)
    assert s.topological_charge(-sk) == pytest.approx(+1.0, abs=1e-12)
    two = W.skyrmion_spins(w, 6.0, centre=ctr - [8.0, 0.0])
    other = W.skyrmion_spins(w, 6.0, centre=ctr + [8.0, 0.0])
    inside = np.linalg.norm(pos[:, :2] - (ctr + [8.0, 0.0]), axis=1) < 6.0
    two[inside] = other[inside]
    assert s.topological_charge(two) == pytest.approx(-2.0, abs=1e-12)
    # a random configuration on a periodic lattice still has an integer charge
    q = s.topological_charge(rand_spins(w.n_spins, 5))
    assert abs(q - round(q)) < 1e-9


# ------------------------------------------------------------------ pinned spins and vacancies
def _chain(n_sites, J=1.0, B=0.0, alpha=0.1, dt_fs=10.0, mu=2.0):
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (n_sites, 1, 1), (0, 0, 0))
    s.set_mu_s([mu]); s.set_field(B, (0, 0, 1)); s.llg_configure(dt_fs, alpha)
    s.set_pairs([0], [0], [[1, 0, 0]], [J])
    return s


def test_pinned_spin_acts_as_a_fixed_field_source():
    """Spin 0 pinned along x, spin 1 free, exchange J, no external field: spin 1 sees the constant field J x^ / (mu mu_B) and
    follows Eq. 12 in the frame whose polar axis is x; the pinned spin does not move by a single bit."""
    J, mu, alpha, dt_fs = 1.0, 2.0, 0.1, 10.0
    s = _chain(2, J=J, alpha=alpha, dt_fs=dt_fs, mu=mu)
    s.set_pinned([1, 0])
    s.set_spins([[1.0, 0.0, 0.0], [0.0, 1.0, 0.0]])
    Beff = J / (mu * O.MU_B)
    gp = O.GAMMA / (1 + alpha * alpha)
    err = 0.0
    for k in range(500):
        s.iterate(1)
        t = (k + 1) * dt_fs * 1e-3
        npar = math.tanh(alpha * gp * Beff * t); ph = gp * Beff * t; r = math.sqrt(1 - npar * npar)
        # polar axis x, azimuth from y towards z (right-handed about x, same sense as Eq. 12 about z)
        ex = np.array([npar, r * math.cos(ph), r * math.sin(ph)])
        n = s.spins()
        assert np.array_equal(n[0], [1.0, 0.0, 0.0])
        err = max(err, np.abs(n[1] - ex).max())
    assert err < 5e-5, err       # second-order error of the scheme at |A| dt = 0.15 rad per step


def test_vacancy_decouples_its_neighbours():
    """A vacancy (pinned zero vector) in the middle of a 3-site chain: the end spins are free spins, bit for bit the trajectory of
    a single spin in the same field; and the energy equals that of the Hamiltonian with the vacant site's bonds removed."""
    s = _chain(3, J=1.3, B=1.0)
    s.set_pinned([0, 1, 0])
    n0 = np.array([[1.0, 0.0, 0.0], [0.0, 0.0, 0.0], [0.6, 0.0, 0.8]])
    s.set_spins(n0); s.iterate(300)
    for site in (0, 2):
        f = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
        f.set_mu_s([2.0]); f.set_field(1.0, (0, 0, 1)); f.llg_configure(10.0, 0.1)
        f.set_spins([n0[site]]); f.iterate(300)
        assert np.array_equal(s.spins()[site], f.spins()[0])
    assert np.array_equal(s.spins()[1], [0.0, 0.0, 0.0])
    w = small(1, (6, 5, 1))
    a = OracleSystem.from_workload(w)
    n = rand_spins(w.n_spins, 3)
    vac = 13
    n[vac] = 0.0
    keep = np.ones(len(w.pair_J), bool)       # bonds are per cell: removing a site's bonds needs the explicit site loop instead
    E_vac = a.energy_terms(n)
    # explicit: energy of the full lattice minus every term that involves the vacant site, evaluated with the original spin
    m = rand_spins(w.n_spins, 3)
    E_full = a.energy_terms(m)
    F = a.gradient(m)                          # F_i = -dH/dn_i; pair terms are bilinear: E_pairs(site) = -n_i . F_i^{pairs}
    Fz = a.gradient(m, mask=O.T_ZEE)[vac]; Fa = a.gradient(m, mask=O.T_ANI)[vac]
    Fp = a.gradient(m, mask=O.T_EXC | O.T_DMI)[vac]
    expect = E_full.sum() + np.dot(m[vac], Fz) + 0.5 * np.dot(m[vac], Fa) + np.dot(m[vac], Fp)
    assert E_vac.sum() == pytest.approx(expect, rel=1e-12)


# ------------------------------------------------------------------ velocity-projection minimiser, App. D
def test_vp_constant_force_closed_form():
    """One spin in a field: F = mu mu_B B z^ is constant, so D1-D3 give v_k = k dt F / m (always parallel to F,
    the projection changes nothing) and the k-th iteration displaces by (k + 1/2) dt^2 F / m before the renormalisation (D5).
    Pins the 1/(2m) factors, the momentum accumulation and the order of D2 -> D3 -> D1."""
    mu, B, dt, m = 2.0, 1.5, 0.05, 0.7
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
    s.set_mu_s([mu]); s.set_field(B, (0, 0, 1))
    x = np.array([0.8, 0.0, 0.6]); s.set_spins([x])
    F = np.array([0.0, 0.0, mu * O.MU_B * B])
    for k in range(1, 12):
        s.vp_iterate(1, dt, m)
        x = x + (k + 0.5) * dt * dt / m * F
        x /= np.linalg.norm(x)
        assert np.abs(s.spins()[0] - x).max() < 1e-15, k


def test_vp_stops_on_overshoot_and_finds_the_ferromagnet():
    """D3: when v.F <= 0 the velocity is dropped, so the energy of a ferromagnet in a field goes down to the closed form
    E = -N (mu mu_B B + z J / 2) (D4: F = -dH/dn, a wrong sign would climb) from a random start."""
    w = dataclasses.replace(small(1, (8, 8, 1)), pair_D=small(1, (8, 8, 1)).pair_D * 0, aniso=[])    # K = 0: -z is not metastable
    s = OracleSystem.from_workload(w)
    E0 = s.energy()
    s.vp_iterate(4000, 0.1, 1.0)
    N = w.n_spins
    Efm = -N * (w.mu_s[0] * O.MU_B * w.B + 0.5 * 4 * 1.0)
    assert s.energy() < E0
    assert s.energy() == pytest.approx(Efm, rel=1e-10)
    assert np.abs(s.spins() - [0, 0, 1]).max() < 1e-6
    # split calls continue the same trajectory (velocity and previous force persist)
    a = OracleSystem.from_workload(w); a.vp_iterate(30, 0.1)
    b = OracleSystem.from_workload(w); b.vp_iterate(13, 0.1); b.vp_iterate(17, 0.1)
    assert np.array_equal(a.spins(), b.spins())


def test_image_noise_streams_are_independent():
    """Batched images (reading R30): image m draws from the Philox counter words block + 2 m.  Image 0 is the single-system stream;
    other images are standard normal and uncorrelated with it and with each other."""
    seed, n = 77, 4000
    x = {m: np.array([O.thermal_xi(seed, 3, i, image=m) for i in range(n)]) for m in (0, 1, 2)}
    assert np.array_equal(x[0], np.array([O.thermal_xi(seed, 3, i) for i in range(n)]))
    for m in (1, 2):
        assert abs(x[m].mean()) < 0.05 and abs(x[m].var() - 1.0) < 0.06
    for a, b in ((0, 1), (0, 2), (1, 2)):
        c = np.corrcoef(x[a].ravel(), x[b].ravel())[0, 1]
        assert abs(c) < 0.04, (a, b, c)
        assert not np.any(np.all(x[a] == x[b], axis=1))
    # the layout: image m's x/y pair comes from counter word 2 m, its z from 2 m + 1
    ctr = lambda blk: O.philox4x32_10([5, blk, 3, 0], [seed, 0])
    assert not np.array_equal(ctr(2), ctr(0))
    w = small(2, (8, 8, 1))
    a = OracleSystem.from_workload(w); a.set_image(1); a.iterate(5)
    b = OracleSystem.from_workload(w); b.iterate(5)
    assert np.abs(a.spins() - b.spins()).max() > 1e-6


# ------------------------------------------------------------------ GNEB forces (III.D Eqs. 14-17, App. F)
def _single_spin(K=0.0, B=0.0):
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
    s.set_mu_s([2.0]); s.set_field(B, (0, 0, 1))
    if K:
        s.set_anisotropy([0], [K], [[0, 0, 1]])
    return s


def _meridian(thetas, phi=0.3):
    return np.array([[[math.sin(t) * math.cos(phi), math.sin(t) * math.sin(phi), math.cos(t)]] for t in thetas])


def test_gneb_geodesic_distance_and_force_geometry():
    """l is the great-circle distance, in 3N dimensions the root of the summed squared angles; F^E is orthogonal to the
    tangent (Eq. 16), every force lies in the tangent space of its image (F2), end images get none."""
    s = _single_spin(K=0.7, B=0.4)
    a, b = _meridian([0.2])[0], _meridian([1.3])[0]
    assert s.geodesic_distance(a, b) == pytest.approx(1.1, abs=1e-14)
    w = small(1, (5, 4, 1))
    o = OracleSystem.from_workload(w)
    x, y = rand_spins(w.n_spins, 1), rand_spins(w.n_spins, 2)
    ang = np.arccos(np.clip((x * y).sum(1), -1, 1))
    assert o.geodesic_distance(x, y) == pytest.approx(math.sqrt((ang ** 2).sum()), rel=1e-12)
    chain = np.array([rand_spins(w.n_spins, 10 + k) for k in range(5)])
    F, E, l = o.gneb_forces(chain, kappa=0.0)
    assert np.all(F[0] == 0) and np.all(F[-1] == 0)
    for nu in (1, 2, 3):
        assert np.abs((F[nu] * chain[nu]).sum(1)).max() < 1e-13                   # tangent to every spin
        assert E[nu] == pytest.approx(o.energy(chain[nu]), rel=1e-14)
    # pure spring force (no Hamiltonian): parallel to the tangent, i.e. to the projected central difference when E is flat
    free = _single_spin()
    ch = _meridian([0.1, 0.5, 1.6])
    Fs, _, ls = free.gneb_forces(ch, kappa=2.0)
    t = ch[2, 0] - ch[0, 0]; t -= np.dot(t, ch[1, 0]) * ch[1, 0]; t /= np.linalg.norm(t)
    assert np.allclose(Fs[1, 0], 2.0 * (ls[1] - ls[0]) * t, atol=1e-14)             # towards the farther neighbour (reading R31)
    assert ls[0] == pytest.approx(0.4, abs=1e-14) and ls[1] == pytest.approx(1.1, abs=1e-14)


def test_gneb_springs_make_the_chain_equidistant():
    """Eq. 15 "gives an equidistant distribution of images": on a flat energy surface unevenly spaced images relax to
    equal geodesic spacing.  With the two lengths in the printed order the chain bunches up instead (reading R31)."""
    free = _single_spin()
    ch = _meridian([0.1, 0.2, 0.35, 1.9, 2.4])
    out = free.gneb_iterate(ch, 400, 0.2, kappa=1.0)
    l = [free.geodesic_distance(out[k], out[k + 1]) for k in range(4)]
    assert max(l) - min(l) < 1e-6 and sum(l) == pytest.approx(2.3, abs=1e-9)


def test_gneb_climbing_image_finds_the_anisotropy_barrier():
    """One spin with easy axis z: the minimum-energy path from +z to -z is a meridian, the saddle is on the equator and the barrier
    is exactly K (E = -K n_z^2).  The climbing image (Eq. 17) converges onto it."""
    K = 0.8
    s = _single_spin(K=K)
    ch = _meridian(np.linspace(0.02, math.pi - 0.02, 9) + np.array([0, .05, -.04, .06, .1, -.03, .02, -.05, 0]))
    ch[0, 0] = [0, 0, 1]; ch[-1, 0] = [0, 0, -1]
    out = s.gneb_iterate(ch, 300, 0.2, kappa=1.0)
    _, E, _ = s.gneb_forces(out)
    ci = int(np.argmax(E))
    out = s.gneb_iterate(out, 600, 0.2, kappa=1.0, climbing=ci)
    F, E, l = s.gneb_forces(out, climbing=ci)
    assert E[ci] - E[0] == pytest.approx(K, abs=1e-10)
    assert abs(out[ci, 0, 2]) < 1e-6
    assert np.abs(F).max() < 1e-6
    assert max(l[:3]) - min(l[:3]) < 1e-3


def test_several_anisotropy_axes_per_atom():
    """Eq. 1 sums the anisotropy over axes j as well as over spins: -sum_i sum_j K_j (K^_j . n_i)^2.  Two axes on one atom:
    the closed form of the biaxial energy (the form of Eq. 13, :187), the gradient against finite differences, and the equivalence of
    two equal axes with one of double strength."""
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (3, 2, 1), (0, 0, 0))
    s.set_mu_s([2.0])
    K1, K2 = 0.7, -0.3
    s.set_anisotropy([0, 0], [K1, K2], [[1, 0, 0], [0, 2, 0]])
    n = rand_spins(6, 4)
    assert s.energy_terms(n)[1] == pytest.approx(-(K1 * n[:, 0] ** 2 + K2 * n[:, 1] ** 2).sum(), rel=1e-14)
    F = s.gradient(n)
    assert np.allclose(F, np.stack([2 * K1 * n[:, 0], 2 * K2 * n[:, 1], 0 * n[:, 2]], axis=1), atol=1e-15)
    _fd_check(s, n, [0, 3, 5])
    a = OracleSystem(np.eye(3), [[0, 0, 0]], (3, 2, 1), (0, 0, 0)); a.set_anisotropy([0, 0], [0.2, 0.2], [[0, 0, 1], [0, 0, 1]])
    b = OracleSystem(np.eye(3), [[0, 0, 0]], (3, 2, 1), (0, 0, 0)); b.set_anisotropy([0], [0.4], [[0, 0, 1]])
    assert a.energy(n) == pytest.approx(b.energy(n), rel=1e-15)


def test_damping_only_dynamics_closed_form():
    """"considering only the damping part of the LLG equation".  One spin in a field: without the precession term the
    azimuth stays put and n_z follows the same tanh as in Eq. 12 (:178), n_z(t) = tanh(alpha gamma' B t + atanh n_z0)."""
    alpha, B, dt_fs = 0.3, 2.0, 5.0
    for solver in (0, 1, 2, 3):
        s = OracleSystem(np.eye(3), [[0, 0, 0]], (1, 1, 1), (0, 0, 0))
        s.set_mu_s([2.0]); s.set_field(B, (0, 0, 1)); s.llg_configure(dt_fs, alpha); s.set_solver(solver); s.set_damping_only(True)
        n0 = np.array([0.6 * math.cos(0.7), 0.6 * math.sin(0.7), -0.8])
        s.set_spins([n0])
        gp = O.GAMMA / (1 + alpha * alpha)
        for k in range(1, 401):
            s.iterate(1)
            n = s.spins()[0]
            nz = math.tanh(alpha * gp * B * k * dt_fs * 1e-3 + math.atanh(-0.8))
            assert abs(n[2] - nz) < 2e-6, (solver, k, n[2], nz)
            assert abs(math.atan2(n[1], n[0]) - 0.7) < 1e-12
    # a coupled system runs downhill
    w = small(1, (8, 8, 1))
    c = OracleSystem.from_workload(w); c.set_damping_only(True)
    E = [c.energy()]
    for _ in range(5):
        c.iterate(100); E.append(c.energy())
    assert all(b < a for a, b in zip(E, E[1:]))


def test_current_driven_domain_wall_moves_at_beta_over_alpha_u():
    """The experiment of Fig. 6: head-to-head wall in a chain along x with the biaxial Hamiltonian of Eq. 13 and the
    end spins pinned.  Below the Walker breakdown the wall moves steadily ("linear fits" of Fig. 6) at the Zhang-Li / Thiaville (Ref. 53)
    velocity v = (beta / alpha) u -- which pins both current terms of Eq. 10 for beta != alpha (O11 only covers beta = alpha), several
    anisotropy axes per atom and pinning together.  Lattice discreteness and the approach to the steady state leave 2 %."""
    N, alpha, beta, u = 240, 0.1, 0.2, 0.02
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (N, 1, 1), (0, 0, 0))
    s.set_mu_s([2.0])
    s.set_anisotropy([0, 0], [0.05, -0.03], [[1, 0, 0], [0, 1, 0]])        # easy axis x, hard axis y
    s.set_pairs([0], [0], [[1, 0, 0]], [1.0])
    s.llg_configure(10.0, alpha, 0.0, 0, u, (1, 0, 0), beta)
    x = np.arange(N)
    w = math.sqrt(1.0 / (2 * 0.05))
    n0 = np.stack([-np.tanh((x - N / 2) / w), np.zeros(N), 1.0 / np.cosh((x - N / 2) / w)], axis=1)
    n0 /= np.linalg.norm(n0, axis=1, keepdims=True)
    mask = np.zeros(N, np.uint8); mask[0] = mask[-1] = 1
    s.set_pinned(mask); s.set_spins(n0)
    ts, xs = [], []
    for k in range(160):
        s.iterate(500)
        ts.append((k + 1) * 5.0); xs.append(0.5 * (N + s.spins()[:, 0].sum()))      # wall position from sum n_x
    v = np.polyfit(ts[120:], xs[120:], 1)[0]
    assert v == pytest.approx(beta / alpha * u, rel=0.04), v
    assert np.array_equal(s.spins()[0], n0[0]) and np.array_equal(s.spins()[-1], n0[-1])


# ------------------------------------------------------------------ what the boundary returns: effective field in Tesla, observables
@pytest.mark.parametrize("mu_s", [2.0, 5.0])
def test_effective_field_of_free_spins_is_the_applied_field_in_tesla(mu_s):
    """PAPER.md:155 "B_eff = -dH/dn_i", reading R2: the boundary returns F / (mu_s mu_B) in Tesla.  Free spins in a field B: the Zeeman
    force is mu_s mu_B B (Eq. 1 :61), so the effective field is B itself whatever the moment -- a dropped or doubled mu_B, or a
    field left in meV, fails this."""
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (4, 3, 2), (0, 0, 0))
    s.set_mu_s([mu_s])
    d = np.array([1.0, 2.0, -2.0]) / 3.0
    s.set_field(1.7, d)
    s.set_spins(rand_spins(s.N, 11))
    B = s.effective_field()
    assert np.allclose(B, 1.7 * d, rtol=0, atol=1e-15)
    # the force itself (meV) does scale with the moment
    F = s.gradient()
    assert np.allclose(F, mu_s * O.MU_B * 1.7 * d, rtol=1e-15, atol=0)


@pytest.mark.parametrize("cfg,cells,z", [(1, (8, 6, 1), 4), (3, (6, 5, 4), 6)])
def test_effective_field_of_the_ferromagnet_in_tesla(cfg, cells, z):
    """All n = z, periodic (O1): F_z = mu_s mu_B B + 2 K + z J (unique pairs, each bond felt from both ends), DMI cancels, so
    B_eff,z = B + (2 K + z J) / (mu_s mu_B) in Tesla, to 1e-13 (readings R2-R4)."""
    w = small(cfg, cells)
    s = OracleSystem.from_workload(w)
    s.set_spins(np.tile([0.0, 0.0, 1.0], (s.N, 1)))
    K = w.aniso[0][1] if w.aniso else 0.0
    mu = w.mu_s[0] * O.MU_B
    B = s.effective_field()
    expect = w.B + (2.0 * K + z * 1.0) / mu
    assert np.allclose(B[:, 2], expect, rtol=1e-13, atol=0)
    assert np.abs(B[:, :2]).max() < 1e-12 * expect


def test_effective_field_uses_the_moment_of_each_basis_atom():
    """Two sublattices with different moments in the same applied field: both see B Tesla, and the pair term J n_j enters as
    J / (mu_b mu_B), with the moment of the atom the field acts ON."""
    s = OracleSystem(np.eye(3), [[0, 0, 0], [0.5, 0.5, 0.5]], (3, 3, 3), (1, 1, 1))
    s.set_mu_s([2.0, 5.0])
    s.set_field(0.5, (0, 0, 1))
    s.set_pairs([0], [1], [[0, 0, 0]], [1.5])
    s.set_spins(np.tile([0.0, 0.0, 1.0], (s.N, 1)))
    B = s.effective_field()
    assert np.allclose(B[0::2, 2], 0.5 + 1.5 / (2.0 * O.MU_B), rtol=1e-14)
    assert np.allclose(B[1::2, 2], 0.5 + 1.5 / (5.0 * O.MU_B), rtol=1e-14)


def test_observables_magnetisation_and_max_torque_closed_forms():
    """PAPER.md:131 m = (1/N) sum_i n_i; reading R22: max torque = max_i |F_i - (F_i . n_i) n_i| in meV.  One spin tilted by theta away
    from the field among aligned free spins: M is known exactly and the largest torque is mu_s mu_B B sin(theta) (= |n x F|)."""
    mu_s, Bf, theta = 3.0, 2.0, 0.4
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (5, 4, 1), (0, 0, 0))
    s.set_mu_s([mu_s]); s.set_field(Bf, (0, 0, 1))
    n = np.tile([0.0, 0.0, 1.0], (s.N, 1))
    n[7] = [math.sin(theta), 0.0, math.cos(theta)]
    n[3] = [0.0, 0.0, -1.0]                         # antiparallel: no torque, but it counts in M
    s.set_spins(n)
    M, tq = s.observables()
    assert M[0] == pytest.approx(math.sin(theta) / s.N, rel=1e-14)
    assert M[1] == 0.0
    assert M[2] == pytest.approx((s.N - 2 + math.cos(theta) - 1.0) / s.N, rel=1e-14)
    assert tq == pytest.approx(mu_s * O.MU_B * Bf * math.sin(theta), rel=1e-13)
    # with an exchange bond the torque on the pair is |n x (F_Zeeman + J n_j)|
    s.set_pairs([0], [0], [[1, 0, 0]], [0.8])
    F = s.gradient()
    expect = max(np.linalg.norm(np.cross(n[i], F[i])) for i in range(s.N))
    M2, tq2 = s.observables()
    assert tq2 == pytest.approx(expect, rel=1e-13) and np.array_equal(M, M2)


# ------------------------------------------------------------------ atoms of different types: per-site moments (reading R32)
def test_site_moments_zeeman_energy_and_larmor_frequency():
    """A chain of free spins of two species (mu = 1.5 and 4 mu_B, alternating along the chain although the basis has one atom) in a field:
    E = -sum_i mu_i mu_B B . n_i (Eq. 1 :61) depends on the moments; the effective field in Tesla and the whole trajectory (Eq. 12: the
    precession and damping rates are gamma' B and alpha gamma' B, the moment cancels between Eq. 1 and the 1/mu_i of Eq. 10) do not."""
    N = 6
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (N, 1, 1), (0, 0, 0))
    s.set_mu_s([2.0]); s.set_field(1.3, (0, 0, 1))
    mu = np.array([1.5, 4.0] * 3)
    s.set_site_mu_s(mu)
    n0 = rand_spins(N, 4)
    s.set_spins(n0)
    assert s.energy_terms()[0] == pytest.approx(-(mu * O.MU_B * 1.3 * n0[:, 2]).sum(), rel=1e-14)
    assert np.allclose(s.gradient(), (mu * O.MU_B * 1.3)[:, None] * [0, 0, 1], rtol=1e-15)
    assert np.allclose(s.effective_field(), [0.0, 0.0, 1.3], rtol=0, atol=1e-15)
    s.llg_configure(10.0, 0.1)
    s.iterate(500)
    alpha, t = 0.1, 5.0
    gp = O.GAMMA / (1 + alpha * alpha)
    nz = np.tanh(alpha * gp * 1.3 * t + np.arctanh(n0[:, 2]))
    assert np.abs(s.spins()[:, 2] - nz).max() < 5e-7                      # both species follow Eq. 12
    r = OracleSystem(np.eye(3), [[0, 0, 0]], (N, 1, 1), (0, 0, 0))       # the same chain with one species
    r.set_mu_s([2.0]); r.set_field(1.3, (0, 0, 1)); r.llg_configure(10.0, 0.1); r.set_spins(n0); r.iterate(500)
    assert np.abs(s.spins() - r.spins()).max() < 1e-12
    s.set_site_mu_s(None)                                                 # cleared: the basis atom's moment again
    s.set_spins(n0)
    assert s.energy_terms()[0] == pytest.approx(-(2.0 * O.MU_B * 1.3 * n0[:, 2]).sum(), rel=1e-14)


def test_site_moments_in_the_exchange_field_and_the_dipolar_sum():
    """(i) A bond J between two sites of different moment: the field ON site i in Tesla is J n_j / (mu_i mu_B), so with a field the
    precession rates of the two species differ.  (ii) Two dipoles mu_1 != mu_2 head to tail at distance r: E = -2 C_dd mu_1 mu_2 / r^3,
    force on each C_dd mu_1 mu_2 2 / r^3 along the axis (the product of BOTH moments).  (iii) the padded-FFT path equals the direct sum
    with per-site moments on a periodic lattice."""
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (2, 1, 1), (0, 0, 0))
    s.set_mu_s([1.0]); s.set_site_mu_s([2.0, 5.0])
    s.set_pairs([0], [0], [[1, 0, 0]], [0.7])
    s.set_spins([[0, 0, 1.0], [1.0, 0, 0]])
    B = s.effective_field()
    assert np.allclose(B[0], np.array([0.7, 0, 0]) / (2.0 * O.MU_B), rtol=1e-15)
    assert np.allclose(B[1], np.array([0, 0, 0.7]) / (5.0 * O.MU_B), rtol=1e-15)
    d = OracleSystem(np.eye(3), [[0, 0, 0]], (2, 1, 1), (0, 0, 0), 2.0)
    d.set_mu_s([1.0]); d.set_site_mu_s([2.0, 5.0]); d.set_ddi(True, (0, 0, 0), direct=True)
    n = np.array([[1.0, 0, 0], [1.0, 0, 0]])
    d.set_spins(n)
    r3 = 8.0
    assert d.energy_terms()[5] == pytest.approx(-2 * O.C_DD * 10.0 / r3, rel=1e-14)
    assert d.energy_ddi_pairsum() == pytest.approx(-2 * O.C_DD * 10.0 / r3, rel=1e-14)
    assert np.allclose(d.ddi_field(direct=True), [[2 * O.C_DD * 10.0 / r3, 0, 0]] * 2, rtol=1e-14)
    assert np.allclose(d.ddi_field(direct=False), d.ddi_field(direct=True), rtol=1e-13)
    p = OracleSystem([[1, 0, 0], [0.3, 0.9, 0], [0, 0.1, 1.2]], [[0, 0, 0], [0.4, 0.3, 0.2]], (4, 3, 2), (1, 1, 0), 1.1)
    p.set_mu_s([1.0, 2.0]); p.set_ddi(True, (2, 1, 0))
    mu = np.random.default_rng(5).uniform(0.5, 3.0, p.N)
    p.set_site_mu_s(mu)
    nn = rand_spins(p.N, 6)
    Ff, Fd = p.ddi_field(nn, direct=False), p.ddi_field(nn, direct=True)
    assert np.abs(Ff - Fd).max() <= 1e-13 * np.abs(Fd).max()
    # Euler identity with per-site moments: E_ddi = -(1/2) sum n . F_ddi
    p.set_spins(nn)
    assert p.energy_terms()[5] == pytest.approx(-0.5 * (nn * Fd).sum(), rel=1e-12)


def test_site_moments_set_the_thermal_amplitude():
    """Eq. 11 (:157): sigma_i = sqrt(2 alpha k_B T mu_i mu_B / (gamma dt)).  Two decoupled species in the same field at the same temperature
    equilibrate to their own Langevin magnetisation coth(x_i) - 1/x_i, x_i = mu_i mu_B B / (k_B T)."""
    B, T, alpha = 30.0, 20.0, 0.5
    s = OracleSystem(np.eye(3), [[0, 0, 0]], (48, 40, 1), (0, 0, 0))
    s.set_mu_s([1.0]); s.set_field(B, (0, 0, 1)); s.llg_configure(5.0, alpha, T=T, seed=12)
    mu = np.where(np.arange(s.N) % 2 == 0, 1.0, 3.0)
    s.set_site_mu_s(mu)
    s.set_spins(rand_spins(s.N, 2))
    s.iterate(800)
    acc = [[], []]
    for _ in range(60):
        s.iterate(40)
        nz = s.spins()[:, 2]
        acc[0].append(nz[0::2].mean()); acc[1].append(nz[1::2].mean())
    for k, m in enumerate((1.0, 3.0)):
        x = m * O.MU_B * B / (O.K_B * T)
        L = 1 / math.tanh(x) - 1 / x
        assert abs(float(np.mean(acc[k])) - L) < 0.012, (m, np.mean(acc[k]), L)
