"""Seeded synthetic workloads (BASELINE.json `configs`; recipe in DESIGN.md §5).

This module holds NONE of the method's arithmetic: it only draws initial particle states and source
histories with ``numpy.random.default_rng`` and converts them to the units of the C-ABI (positions in grid
units, momenta u = gamma v / c).  It is the one module shared by the CUDA path's harness and the tests'
oracle harness; it imports neither.  The inputs stand in for the paper's own set-ups (§3), which
are self-defined simulations, not a public dataset.
"""
from __future__ import annotations

import math
from dataclasses import dataclass
from typing import Dict, Iterator, Optional

import numpy as np

# Physical constants (DESIGN.md §3 reading A18)
C_SI = 299792458.0
EPS0_SI = 8.8541878128e-12
E_CHARGE = 1.602176634e-19
M_E = 9.1093837015e-31
M_P = 1.67262192369e-27
SEED0 = 20220907


@dataclass(frozen=True)
class Workload:
    """Grid + run description of one BASELINE.json config."""

    name: str
    config: int
    n: int  # cubic grid n^3
    dx: float
    steps: int
    field_only: bool = False

    @property
    def dt(self) -> float:
        return self.dx / (2.0 * C_SI)  # dt = dx/(2c) in every config

    @property
    def N(self) -> int:
        return self.n ** 3

    @property
    def H(self) -> int:
        # BASELINE.json: H = ceil(sqrt(3) * n * dx / (c dt)) + 2
        return int(math.ceil(math.sqrt(3.0 * (self.n * self.dx) ** 2) / (C_SI * self.dt))) + 2

    @property
    def seed(self) -> int:
        return SEED0 + self.config


WORKLOADS: Dict[int, Workload] = {
    1: Workload("cfg1_16c_electron_cloud", 1, 16, 1e-4, 64),
    2: Workload("cfg2_32c_neutral_plasma", 2, 32, 1e-4, 100),
    3: Workload("cfg3_64c_electron_beam", 3, 64, 5e-5, 200),
    4: Workload("cfg4_96c_field_only", 4, 96, 1e-4, 1, field_only=True),
    5: Workload("cfg5_128c_two_stream", 5, 128, 5e-5, 50),
}


def _sigma_u(kT_eV: float, mass: float) -> float:
    """Maxwellian: each momentum component u = gamma v/c is Gaussian with sigma = sqrt(kT/(m c^2))."""
    return math.sqrt(kT_eV * E_CHARGE / (mass * C_SI * C_SI))


def _gauss_inside(rng, mean, sigma, n, lo, hi):
    """Gaussian draws, rejecting and redrawing values outside [lo, hi)."""
    out = rng.normal(mean, sigma, n)
    bad = (out < lo) | (out >= hi)
    while bad.any():
        out[bad] = rng.normal(mean, sigma, int(bad.sum()))
        bad = (out < lo) | (out >= hi)
    return out


def _species(x, y, z, ux, uy, uz, charge, mass, weight):
    n = x.shape[0]
    return dict(x=x, y=y, z=z, ux=ux, uy=uy, uz=uz,
                qw=np.full(n, charge * weight), qm=np.full(n, charge / mass))


def _concat(parts):
    keys = ("x", "y", "z", "ux", "uy", "uz", "qw", "qm")
    out = {k: np.concatenate([p[k] for p in parts]).astype(np.float32) for k in keys}
    out["alive"] = np.ones(out["x"].shape[0], dtype=np.uint8)
    return out


def particles(config: int, scale: float = 1.0) -> Dict[str, np.ndarray]:
    """Initial macro-particles of a PIC config as fp32 arrays (positions in grid units, u = gamma v/c).

    ``scale`` < 1 draws proportionally fewer macro-particles with proportionally larger weight (same total
    charge); used only by CPU-sized tests.  Keys: x y z ux uy uz qw (C per macro-particle) qm (q/m) alive.
    """
    w = WORKLOADS[config]
    rng = np.random.default_rng(w.seed)
    n = float(w.n)
    if config == 1:
        P = max(1, int(round(4096 * scale)))
        wt = 1e6 / scale
        su = _sigma_u(1000.0, M_E)
        pos = [_gauss_inside(rng, n / 2, 3.0, P, 0.0, n) for _ in range(3)]
        mom = [rng.normal(0.0, su, P) for _ in range(3)]
        return _concat([_species(*pos, *mom, -E_CHARGE, M_E, wt)])
    if config == 2:
        P = max(1, int(round(100000 * scale)))
        wt = 1e6 / scale
        parts = []
        for charge, mass, kT in ((-E_CHARGE, M_E, 1000.0), (E_CHARGE, M_P, 10.0)):
            su = _sigma_u(kT, mass)
            pos = [rng.uniform(n / 2 - 8.0, n / 2 + 8.0, P) for _ in range(3)]
            mom = [rng.normal(0.0, su, P) for _ in range(3)]
            parts.append(_species(*pos, *mom, charge, mass, wt))
        return _concat(parts)
    if config == 3:
        P = max(1, int(round(1000000 * scale)))
        wt = 5e4 / scale
        su = _sigma_u(10.0, M_E)
        x = _gauss_inside(rng, n / 2, 4.0, P, 0.0, n)
        y = _gauss_inside(rng, n / 2, 4.0, P, 0.0, n)
        z = rng.uniform(16.0, 48.0, P)
        beta = 0.5
        drift = beta / math.sqrt(1.0 - beta * beta)  # gamma_d * beta_d, added in u-space
        mom = [rng.normal(0.0, su, P), rng.normal(0.0, su, P), rng.normal(0.0, su, P) + drift]
        return _concat([_species(x, y, z, *mom, -E_CHARGE, M_E, wt)])
    if config == 5:
        Pb = max(1, int(round(2000000 * scale)))
        Pp = max(1, int(round(4000000 * scale)))
        wt = 2e5 / scale
        su = _sigma_u(100.0, M_E)
        parts = []
        for sign in (+1.0, -1.0):
            beta = 0.3
            drift = sign * beta / math.sqrt(1.0 - beta * beta)
            x = rng.uniform(0.0, n, Pb)
            y = _gauss_inside(rng, n / 2, 8.0, Pb, 0.0, n)
            z = _gauss_inside(rng, n / 2, 8.0, Pb, 0.0, n)
            mom = [rng.normal(0.0, su, Pb) + drift, rng.normal(0.0, su, Pb), rng.normal(0.0, su, Pb)]
            parts.append(_species(x, y, z, *mom, -E_CHARGE, M_E, wt))
        pos = [rng.uniform(0.0, n, Pp) for _ in range(3)]
        zero = [np.zeros(Pp) for _ in range(3)]
        parts.append(_species(*pos, *zero, E_CHARGE, M_P, wt))
        out = _concat(parts)
        # fp32 rounding of a draw just below n can land on n exactly; keep every start position inside [0, n)
        for k in ("x", "y", "z"):
            np.minimum(out[k], np.nextafter(np.float32(n), np.float32(0)), out=out[k])
        return out
    raise ValueError(f"config {config} has no particles")


# ---------------------------------------------------------------------------------------------------------------
# The paper's own slab set-ups (PAPER.md:243-250 grid and time step, :262 point emission, :288 zero-velocity column in
# a 10 T field): non-cubic grids, kappa = dx/(c dt) = 0.334 (neighbouring cells have delay 0),
# an external field.  The paper's seed and macro-particle count are unknown; these are seeded stand-ins.
# ---------------------------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class SlabWorkload:
    name: str
    shape: tuple  # (nx, ny, nz)
    dx: float
    dt: float
    Bext: tuple
    total_charge: float  # coulomb
    seed: int

    @property
    def N(self) -> int:
        return self.shape[0] * self.shape[1] * self.shape[2]


SLABS: Dict[str, SlabWorkload] = {
    "point_emission": SlabWorkload("slab_1x101x101_point_emission", (1, 101, 101), 1e-5, 1e-13, (0.0, 0.0, 0.0), -5e-14, SEED0 + 11),
    "column_in_By": SlabWorkload("slab_1x251x111_column_in_By", (1, 251, 111), 1e-5, 1e-13, (0.0, 10.0, 0.0), -5e-14, SEED0 + 12),
    # PAPER.md:356 (section 3.3.2, Fig. 14 caption at :368): electrons on the face y = 9 dy, z from 5 dz to 106 dz, speeds along
    # +y uniform in [0, v0] (v0 = 10 eV), 10 T B_y; Table 1 prints JefiPIC's maximum
    # displacement and velocity at 0.4 and 0.6 ns for this set-up.
    "planar_emission": SlabWorkload("slab_1x251x111_planar_emission", (1, 251, 111), 1e-5, 1e-13, (0.0, 10.0, 0.0), -5e-14, SEED0 + 13),
}
V0_10EV = math.sqrt(2.0 * 10.0 * E_CHARGE / M_E)  # "the energy corresponding to the velocities v0 ... equals to 10 eV"


def slab_particles(which: str, count: int, variant: str = "") -> Dict[str, np.ndarray]:
    """`count` macro-electrons of total charge -5e-14 C.
    point_emission (Fig. 5): uniform in the cell j = k = 50, velocity in the yz plane, speed Gaussian about
    v0 (10 eV) with sigma 0.2 v0, direction uniform.  column_in_By (Fig. 8): uniform in the column
    j = 124, k = 5..105, at rest.  planar_emission (Fig. 14): on the face y = 9 dy, z in [5, 106) dz, speed
    along +y uniform in [0, v0]."""
    w = SLABS[which]
    rng = np.random.default_rng(w.seed)
    wt = w.total_charge / (-E_CHARGE) / count
    x = rng.uniform(0.0, 1.0, count)
    if which == "point_emission":
        y, z = rng.uniform(50.0, 51.0, count), rng.uniform(50.0, 51.0, count)
        v0 = math.sqrt(2.0 * 10.0 * E_CHARGE / M_E)
        speed = np.abs(rng.normal(v0, 0.2 * v0, count))
        ang = rng.uniform(0.0, 2.0 * math.pi, count)
        beta = speed / C_SI
        g = 1.0 / np.sqrt(1.0 - beta * beta)
        mom = [np.zeros(count), g * beta * np.cos(ang), g * beta * np.sin(ang)]
    elif which == "planar_emission":
        # variant: what Fig. 14 (an image) leaves open.  "" = on the plane y = 9 dy; "cell" = uniform in the cell layer
        # 9 dy <= y < 10 dy; "xcentre" = all at x = dx/2 (no charge on the virtual x nodes of the one-cell-thick grid)
        y = rng.uniform(9.0, 10.0, count) if variant == "cell" else np.full(count, 9.0)
        z = rng.uniform(5.0, 106.0, count)
        if variant == "xcentre":
            x = np.full(count, 0.5)
        beta = rng.uniform(0.0, V0_10EV, count) / C_SI
        mom = [np.zeros(count), beta / np.sqrt(1.0 - beta * beta), np.zeros(count)]
    else:
        y, z = rng.uniform(124.0, 125.0, count), rng.uniform(5.0, 106.0, count)
        mom = [np.zeros(count) for _ in range(3)]
    return _concat([_species(x, y, z, *mom, -E_CHARGE, M_E, wt)])


def history_slices(n_cells: int, H: int, seed: int, j_scale: float = 1.0) -> Iterator[np.ndarray]:
    """Config-4 style source history: H slices of [4][N] fp32, i.i.d. uniform in [-1, 1].

    Slot t uses its own generator ``default_rng([seed, t])`` so any slice can be regenerated alone.
    ``j_scale`` multiplies Jx,Jy,Jz (the parity-only variant uses j_scale = c so that the J-dot term of
    Eq. (2.4) is visible next to the rho terms; SURVEY.md §8(d) config 4 caveat).
    """
    for t in range(H):
        yield history_slice(n_cells, t, seed, j_scale)


def history_slice(n_cells: int, t: int, seed: int, j_scale: float = 1.0) -> np.ndarray:
    rng = np.random.default_rng([seed, t])
    s = rng.random((4, n_cells), dtype=np.float32)  # fp32 draws directly: the 96^3 x 335-slot history is 1.2e9 values
    s *= np.float32(2.0)
    s -= np.float32(1.0)
    if j_scale != 1.0:
        s[1:] *= np.float32(j_scale)
    return s


def sample_obs(n_cells_axis: int, count: int, seed: int) -> np.ndarray:
    """Seeded observation-cell sample for sampled parity: `count` random cells + 8 corners, 6 face centres
    and the centre cell."""
    n = n_cells_axis
    rng = np.random.default_rng([seed, 777])
    idx = rng.integers(0, n ** 3, size=count, dtype=np.int64)
    m, c = n - 1, n // 2
    special = []
    for k in (0, m):
        for j in (0, m):
            for i in (0, m):
                special.append((i, j, k))
    special += [(0, c, c), (m, c, c), (c, 0, c), (c, m, c), (c, c, 0), (c, c, m), (c, c, c)]
    sp = np.array([i + n * (j + n * k) for i, j, k in special], dtype=np.int64)
    return np.concatenate([idx, sp])


# ---------------------------------------------------------------------------------------------------------------
# Field-only workloads of bench.py (one jefi_push_sources + jefi_field_step per timed step).  "4" is BASELINE.json's
# configs[3], the one the metric is quoted on; the other two are the paper's own shapes (SURVEY.md section 8(f) NEXT-1 and
# NEXT-2): the 20^3 analytic-source example in units c = eps0 = mu0 = 1 with dx = 0.3, dt = 0.05, i.e. kappa = 6
# (Eqs. 3.4-3.5) and the 1 x 251 x 111 slab with dx = 1e-5 m, dt = 1e-13 s, kappa = 0.334
# (PAPER.md:243-250, 288, 356).  Numbers 1, 2, 3, 5 give a random history on that config's grid (used by CPU-sized tests).
# ---------------------------------------------------------------------------------------------------------------
def history_depth(shape, h, dt: float, c: float) -> int:
    """BASELINE.json / PAPER.md:211: H = ceil(L_max/(c dt)) + 2 with L_max the diagonal of the region."""
    lmax = math.sqrt(sum((n * d) ** 2 for n, d in zip(shape, h)))
    return int(math.ceil(lmax / (c * dt))) + 2


@dataclass(frozen=True)
class FieldWorkload:
    name: str
    config: Optional[int]  # BASELINE.json config number, None for the paper's own shapes
    shape: tuple           # (nx, ny, nz)
    h: tuple               # (dx, dy, dz)
    dt: float
    c: float               # 0 -> SI
    eps0: float            # 0 -> SI
    seed: int
    kind: str              # "random": i.i.d. uniform [-1, 1) in every cell and slot; "analytic": Eqs. (3.4)-(3.5)

    @property
    def N(self) -> int:
        return self.shape[0] * self.shape[1] * self.shape[2]

    @property
    def c_eff(self) -> float:
        return self.c if self.c > 0 else C_SI

    @property
    def H(self) -> int:
        return history_depth(self.shape, self.h, self.dt, self.c_eff)

    @property
    def kappa(self) -> float:
        return self.h[0] / (self.c_eff * self.dt)

    def slice(self, t: int, j_scale: float = 1.0) -> np.ndarray:
        """Sources of step t as the C-ABI takes them: fp32 [4][N] = rho, Jx, Jy, Jz."""
        if self.kind == "random":
            return history_slice(self.N, t, self.seed, j_scale)
        nx, ny, nz = self.shape
        k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
        u = ((i + 0.5) * self.h[0] + (j + 0.5) * self.h[1] + (k + 0.5) * self.h[2]).ravel()
        tt = t * self.dt
        jv = np.sin(u) * math.sin(tt)                                   # Eq. (3.4)
        rho = 3.0 * (math.cos(tt) - 1.0) * np.cos(u)                    # Eq. (3.5)
        return np.stack([rho, jv, jv, jv]).astype(np.float32)


def field_workload(key) -> FieldWorkload:
    key = str(key)
    if key in ("1", "2", "3", "4", "5"):
        w = WORKLOADS[int(key)]
        return FieldWorkload(w.name if w.field_only else w.name + "_random_history", w.config, (w.n,) * 3, (w.dx,) * 3, w.dt, 0.0, 0.0,
                             w.seed, "random")
    if key == "analytic20":
        return FieldWorkload("paper_analytic_20c_kappa6", None, (20, 20, 20), (0.3, 0.3, 0.3), 0.05, 1.0, 1.0, SEED0 + 21, "analytic")
    if key == "slab251":
        return FieldWorkload("paper_slab_1x251x111_field_only", None, (1, 251, 111), (1e-5,) * 3, 1e-13, 0.0, 0.0, SEED0 + 22, "random")
    if key == "slab101":
        return FieldWorkload("paper_slab_1x101x101_field_only", None, (1, 101, 101), (1e-5,) * 3, 1e-13, 0.0, 0.0, SEED0 + 23, "random")
    raise ValueError(f"unknown field workload {key!r} (1-5, analytic20, slab251, slab101)")
