"""Seeded synthetic inputs shared by the oracle and the CUDA library.

This module holds INPUTS only: lattice descriptions, interaction lists, LLG parameters and the seeded
initial spin configurations of the five BASELINE.json configurations (restated in SURVEY.md 8(d) and
DESIGN.md "Input recipe").  It contains none of the method's arithmetic (no energies, fields, rotations
or random-number transforms of the method) and imports neither `oracle` nor `paper_1901_11350_b200`.

The paper measures on no public dataset: its workloads are parameterised lattices, so these
descriptions *are* the workloads.  Choices BASELINE.json leaves open are marked "fill-in".
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Sequence, Tuple

import numpy as np

SQ3 = math.sqrt(3.0)


@dataclasses.dataclass
class Workload:
    name: str
    bravais: np.ndarray            # (3,3) rows a, b, c in units of the lattice constant
    basis: np.ndarray              # (n_basis,3) fractional coordinates
    n_cells: Tuple[int, int, int]
    periodic: Tuple[int, int, int]
    lattice_constant: float        # Angstrom
    mu_s: np.ndarray               # (n_basis,) in mu_B
    B: float                       # Tesla
    B_dir: Tuple[float, float, float]
    aniso: List[Tuple[int, float, Tuple[float, float, float]]]   # (basis atom, K meV, axis)
    pair_i: np.ndarray             # (n_pairs,) basis atom of i
    pair_j: np.ndarray             # (n_pairs,) basis atom of j
    pair_t: np.ndarray             # (n_pairs,3) cell translation of j relative to i
    pair_J: np.ndarray             # (n_pairs,) meV
    pair_D: np.ndarray             # (n_pairs,3) meV
    quad_b: np.ndarray             # (n_quads,4) basis atoms i,j,k,l
    quad_t: np.ndarray             # (n_quads,9) translations of j,k,l relative to i
    quad_K: np.ndarray             # (n_quads,) meV
    ddi: bool
    ddi_images: Tuple[int, int, int]
    dt_fs: float
    alpha: float
    T: float
    seed: int
    u: float                       # Angstrom / ps
    j_dir: Tuple[float, float, float]
    beta: float
    steps: int
    note: str = ""

    @property
    def n_basis(self) -> int:
        return int(self.basis.shape[0])

    @property
    def n_spins(self) -> int:
        return self.n_basis * int(np.prod(self.n_cells))

    def resized(self, n_cells: Sequence[int], steps: int | None = None, name: str | None = None) -> "Workload":
        """Same physics on a lattice of a different size (parity-test replicas)."""
        return dataclasses.replace(self, n_cells=tuple(int(x) for x in n_cells),
                                   steps=self.steps if steps is None else int(steps),
                                   name=name or f"{self.name}@{'x'.join(str(int(x)) for x in n_cells)}")

    def initial_spins(self) -> np.ndarray:
        """Random unit vectors uniform on the sphere, (N,3) float64, boundary index order
        i = b + n_basis*(ia + Na*(ib + Nb*ic)).  numpy's default bit generator seeded with `seed`."""
        rng = np.random.default_rng(self.seed)
        v = rng.standard_normal((self.n_spins, 3))
        v /= np.linalg.norm(v, axis=1, keepdims=True)
        return np.ascontiguousarray(v)

    def positions(self) -> np.ndarray:
        """Cartesian positions (Angstrom) in boundary index order, for structured starts and tests."""
        na, nb_, nc = self.n_cells
        idx = np.arange(na * nb_ * nc)
        cells = np.stack([idx % na, (idx // na) % nb_, idx // (na * nb_)], axis=1).astype(float)
        frac = cells[:, None, :] + self.basis[None, :, :]
        return (frac.reshape(-1, 3) @ self.bravais) * self.lattice_constant


def _bond_dir(w_bravais, basis, bi, bj, t):
    r = (np.asarray(t, float) + basis[bj] - basis[bi]) @ w_bravais
    return r / np.linalg.norm(r)


def _pairs(bravais, basis, entries, dmi_kind):
    """entries: list of (bi, bj, (ta,tb,tc), J, D).  dmi_kind: 'interfacial' D_ij = D (z x r_ij), 'bulk'
    D_ij = D r_ij (conventions)."""
    pi, pj, pt, J, Dv = [], [], [], [], []
    for bi, bj, t, j, d in entries:
        rh = _bond_dir(bravais, basis, bi, bj, t)
        if dmi_kind == "interfacial":
            dv = d * np.cross([0.0, 0.0, 1.0], rh)
        elif dmi_kind == "bulk":
            dv = d * rh
        else:
            dv = np.zeros(3)
        pi.append(bi); pj.append(bj); pt.append(t); J.append(j); Dv.append(dv)
    return (np.array(pi, np.int32), np.array(pj, np.int32), np.array(pt, np.int32).reshape(-1, 3),
            np.array(J, float), np.array(Dv, float).reshape(-1, 3))


_NOQ = (np.zeros((0, 4), np.int32), np.zeros((0, 9), np.int32), np.zeros((0,), float))
_SC = np.eye(3)
_TRI = np.array([[1.0, 0.0, 0.0], [0.5, SQ3 / 2, 0.0], [0.0, 0.0, 1.0]])
_ONE = np.zeros((1, 3))


def config1() -> Workload:
    """2D square 32x32, J=1, interfacial D=0.3, K=0.1 z, B=1 T z, mu_s=2; dt=1 fs, alpha=0.3, T=0, 1000 steps."""
    p = _pairs(_SC, _ONE, [(0, 0, (1, 0, 0), 1.0, 0.3), (0, 0, (0, 1, 0), 1.0, 0.3)], "interfacial")
    return Workload("cfg1_square32", _SC, _ONE, (32, 32, 1), (1, 1, 0), 1.0, np.array([2.0]), 1.0, (0, 0, 1),
                    [(0, 0.1, (0, 0, 1))], *p, *_NOQ, False, (0, 0, 0), 1.0, 0.3, 0.0, 1, 0.0, (1, 0, 0), 0.0, 1000)


def config2() -> Workload:
    """2D triangular 256x256, shells J1=1, J2=-0.3, J3=-0.1, interfacial D=0.2 on shell 1, K=0.05 z, B=2 T z,
    mu_s=3; dt=0.5 fs, alpha=0.1, T=10 K, 10^4 steps."""
    s1 = [(1, 0, 0), (0, 1, 0), (-1, 1, 0)]
    s2 = [(1, 1, 0), (-1, 2, 0), (-2, 1, 0)]
    s3 = [(2, 0, 0), (0, 2, 0), (-2, 2, 0)]
    ent = [(0, 0, t, 1.0, 0.2) for t in s1] + [(0, 0, t, -0.3, 0.0) for t in s2] + [(0, 0, t, -0.1, 0.0) for t in s3]
    p = _pairs(_TRI, _ONE, ent, "interfacial")
    return Workload("cfg2_triangular256", _TRI, _ONE, (256, 256, 1), (1, 1, 0), 1.0, np.array([3.0]), 2.0, (0, 0, 1),
                    [(0, 0.05, (0, 0, 1))], *p, *_NOQ, False, (0, 0, 0), 0.5, 0.1, 10.0, 2, 0.0, (1, 0, 0), 0.0, 10000)


def config3() -> Workload:
    """3D simple cubic 128^3 (2,097,152 spins), J=1, bulk D=0.2, B=1 T z, mu_s=2; dt=1 fs, alpha=0.05, T=0,
    2000 steps -- the bandwidth headline."""
    ent = [(0, 0, (1, 0, 0), 1.0, 0.2), (0, 0, (0, 1, 0), 1.0, 0.2), (0, 0, (0, 0, 1), 1.0, 0.2)]
    p = _pairs(_SC, _ONE, ent, "bulk")
    return Workload("cfg3_cubic128", _SC, _ONE, (128, 128, 128), (1, 1, 1), 1.0, np.array([2.0]), 1.0, (0, 0, 1),
                    [], *p, *_NOQ, False, (0, 0, 0), 1.0, 0.05, 0.0, 3, 0.0, (1, 0, 0), 0.0, 2000)


def config4() -> Workload:
    """2D honeycomb (2-atom basis) 512x512 cells (524,288 spins): inter-sublattice J=-2 with interfacial D=0.1,
    intra-sublattice J=0.5, quadruplet K4=-0.2 on the nearest-neighbour zig-zag A(c) B(c) A(c+a_d) B(c+a_d),
    easy-plane K=-0.1 z; T=50 K, alpha=0.2, beta=0.1, j along x, 5000 steps.
    fill-ins: dt=0.5 fs, mu_s=2 mu_B, u=0.1 A/ps, B=0."""
    basis = np.array([[0.0, 0.0, 0.0], [1.0 / 3, 1.0 / 3, 0.0]])
    ent = [(0, 1, t, -2.0, 0.1) for t in [(0, 0, 0), (-1, 0, 0), (0, -1, 0)]]
    ent += [(b, b, t, 0.5, 0.0) for b in (0, 1) for t in [(1, 0, 0), (0, 1, 0), (-1, 1, 0)]]
    p = _pairs(_TRI, basis, ent, "interfacial")
    qb = np.array([[0, 1, 0, 1], [0, 1, 0, 1]], np.int32)
    qt = np.array([[0, 0, 0, 1, 0, 0, 1, 0, 0], [0, 0, 0, 0, 1, 0, 0, 1, 0]], np.int32)
    qK = np.array([-0.2, -0.2])
    return Workload("cfg4_honeycomb512", _TRI, basis, (512, 512, 1), (1, 1, 0), 1.0, np.array([2.0, 2.0]), 0.0, (0, 0, 1),
                    [(0, -0.1, (0, 0, 1)), (1, -0.1, (0, 0, 1))], *p, qb, qt, qK, False, (0, 0, 0),
                    0.5, 0.2, 50.0, 4, 0.1, (1, 0, 0), 0.1, 5000)


def config5() -> Workload:
    """Thin film simple cubic 256x256x8 (524,288 spins), periodic in-plane, open along z: J=1, interfacial D=0.3
    (in-plane bonds; z x z = 0 on the c bond), mu_s=2, dipole-dipole on (padded 512x512x16);
    dt=1 fs, alpha=0.3, T=0, 1000 steps.  fill-in: 4 periodic images in each in-plane direction."""
    ent = [(0, 0, (1, 0, 0), 1.0, 0.3), (0, 0, (0, 1, 0), 1.0, 0.3), (0, 0, (0, 0, 1), 1.0, 0.3)]
    p = _pairs(_SC, _ONE, ent, "interfacial")
    return Workload("cfg5_film256x8_ddi", _SC, _ONE, (256, 256, 8), (1, 1, 0), 1.0, np.array([2.0]), 0.0, (0, 0, 1),
                    [], *p, *_NOQ, True, (4, 4, 0), 1.0, 0.3, 0.0, 5, 0.0, (1, 0, 0), 0.0, 1000)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def all_configs() -> List[Workload]:
    return [CONFIGS[k]() for k in sorted(CONFIGS)]


# ---------------------------------------------------------------- structured starts (reporting only)
def skyrmion_spins(w: Workload, radius: float, centre=None) -> np.ndarray:
    """Neel skyrmion ansatz theta(r) = pi (1 - r/R) for r < R in a +z background (paper Fig. 10 workload shape)."""
    pos = w.positions()
    c = pos[:, :2].mean(axis=0) if centre is None else np.asarray(centre, float)
    d = pos[:, :2] - c
    r = np.linalg.norm(d, axis=1)
    theta = np.where(r < radius, math.pi * (1.0 - r / radius), 0.0)
    phi = np.arctan2(d[:, 1], d[:, 0])
    n = np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)], axis=1)
    return np.ascontiguousarray(n)


def domain_wall_spins(w: Workload, x0: float | None = None, width: float = 5.0) -> np.ndarray:
    """Head-to-head wall along x: n_x = -tanh((x-x0)/w), n_y = sech((x-x0)/w) (paper Fig. 6 workload shape)."""
    pos = w.positions()
    x0 = pos[:, 0].mean() if x0 is None else x0
    a = (pos[:, 0] - x0) / width
    n = np.stack([-np.tanh(a), 1.0 / np.cosh(a), np.zeros_like(a)], axis=1)
    return np.ascontiguousarray(n)


def bobber_spins(w: Workload, radius: float, depth_layers: int) -> np.ndarray:
    """Skyrmion tube truncated in depth (chiral bobber shape, paper Figs. 8-9): skyrmion in the top
    `depth_layers` layers with a radius shrinking linearly to zero, +z below."""
    pos = w.positions()
    zmax = pos[:, 2].max()
    c = pos[:, :2].mean(axis=0)
    d = pos[:, :2] - c
    r = np.linalg.norm(d, axis=1)
    below = (zmax - pos[:, 2]) / max(w.lattice_constant, 1e-30)
    rad = np.clip(radius * (1.0 - below / max(depth_layers, 1)), 0.0, None)
    theta = np.where(r < rad, math.pi * (1.0 - r / np.maximum(rad, 1e-30)), 0.0)
    phi = np.arctan2(d[:, 1], d[:, 0])
    n = np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)], axis=1)
    return np.ascontiguousarray(n)
