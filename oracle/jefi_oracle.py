"""ctypes front end of oracle/jefi_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.

Every function here marshals numpy arrays into the plain-C fp64 oracle; the arithmetic of the method lives
in jefi_oracle.c only, each routine citing the PAPER.md passage it follows.  Nothing in this file imports
or loads the CUDA library.
"""
from __future__ import annotations

import ctypes as C
import math
import os
import subprocess
from dataclasses import dataclass, field as dc_field
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jefi_oracle.c")
_LIB = os.path.join(_HERE, "libjefi_oracle.so")

# Reading A18: SI constants used when the config leaves c / eps0 at 0.
C_SI = 299792458.0
EPS0_SI = 8.8541878128e-12
RULE_NEAREST, RULE_LINEAR = 0, 1


def build_oracle(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2, OpenMP, no fast-math).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c99", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


_lib = None


def _L():
    global _lib
    if _lib is None:
        build_oracle()
        lib = C.CDLL(_LIB)
        dbl, i32, i64 = C.c_double, C.c_int, C.c_long
        p = C.c_void_p
        lib.orc_num_threads.restype = C.c_int
        lib.orc_set_num_threads.argtypes = [C.c_int]
        lib.orc_num_dt.restype = C.c_long
        lib.orc_num_dt.argtypes = [i32, i32, i32, dbl, dbl, dbl, dbl, dbl, i64]
        lib.orc_delay.restype = C.c_long
        lib.orc_delay.argtypes = [dbl, dbl, dbl, dbl, dbl]
        lib.orc_delay_table.argtypes = [i32, i32, i32, dbl, dbl, dbl, dbl, dbl, p]
        for name in ("orc_field_f64", "orc_field_f32"):
            getattr(lib, name).argtypes = [i32, i32, i32, dbl, dbl, dbl, dbl, dbl, dbl, i32, i64, i64, p, i64, p, p, p]
            getattr(lib, name).restype = None
        lib.orc_cell_index.argtypes = [i64, p, p, p, p]
        lib.orc_deposit.argtypes = [i32, i32, i32, dbl, dbl, dbl, dbl, i64] + [p] * 12
        lib.orc_interp.argtypes = [i32, i32, i32, i64] + [p] * 7
        lib.orc_push.argtypes = [i32, i32, i32, dbl, dbl, dbl, dbl, dbl, i64] + [p] * 16 + [i32]
        lib.orc_cell_index_s2.argtypes = [i64, p, p, p, p]
        lib.orc_deposit_s2.argtypes = lib.orc_deposit.argtypes
        lib.orc_interp_s2.argtypes = lib.orc_interp.argtypes
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


@dataclass
class OracleConfig:
    """Grid and constants (one structured cuboid grid for sources and observation points)."""

    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    c: float = C_SI
    eps0: float = EPS0_SI
    H: int = 0  # 0 -> N_dt + 2 (DESIGN.md §3 A1: the derivative needs step n-m-1, so two more than N_dt)
    hist_cap: int = 10000
    Eext: Sequence[float] = (0.0, 0.0, 0.0)
    Bext: Sequence[float] = (0.0, 0.0, 0.0)
    delay_rule: int = 0  # RULE_NEAREST (reading A1) or RULE_LINEAR (reading A22)
    shape_order: int = 1  # 1 = linear / CIC weights (Eqs. 2.16, 2.20, what the paper uses); 2 = S^(2), Eq. (2.14) (NEXT-4)

    def __post_init__(self):
        if self.H == 0:
            self.H = num_dt(self) + 2

    @property
    def N(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def mu0(self) -> float:
        return 1.0 / (self.eps0 * self.c * self.c)


def num_threads() -> int:
    return int(_L().orc_num_threads())


def set_num_threads(n: int) -> None:
    _L().orc_set_num_threads(int(n))


def num_dt(cfg: OracleConfig) -> int:
    return int(_L().orc_num_dt(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.dt, cfg.c, cfg.hist_cap))


def delay(cfg: OracleConfig, di: int, dj: int, dk: int) -> int:
    return int(_L().orc_delay(di * cfg.dx, dj * cfg.dy, dk * cfg.dz, cfg.dt, cfg.c))


def delay_table(cfg: OracleConfig) -> np.ndarray:
    """m for every non-negative offset (a,b,c) -> array[nz][ny][nx] int32."""
    out = np.empty((cfg.nz, cfg.ny, cfg.nx), dtype=np.int32)
    _L().orc_delay_table(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.dt, cfg.c, _ptr(out))
    return out


def field(cfg: OracleConfig, n: int, ring: np.ndarray, obs_idx: Optional[np.ndarray] = None, rule: Optional[int] = None):
    """E, B at step n (Eqs. 2.4-2.6).  ring: [H][4][N] float64 or float32, slot = step mod H.
    rule: RULE_NEAREST / RULE_LINEAR (default: cfg.delay_rule).

    Returns (E, B), each float64 [3][nobs]; obs_idx None -> all cells.
    """
    H = ring.shape[0]
    assert ring.shape == (H, 4, cfg.N), ring.shape
    assert ring.flags["C_CONTIGUOUS"]
    if obs_idx is None:
        nobs, idx = cfg.N, None
    else:
        idx = np.ascontiguousarray(obs_idx, dtype=np.int64)
        nobs = idx.shape[0]
    E = np.empty((3, nobs), dtype=np.float64)
    B = np.empty((3, nobs), dtype=np.float64)
    fn = {np.dtype(np.float64): _L().orc_field_f64, np.dtype(np.float32): _L().orc_field_f32}[ring.dtype]
    fn(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.dt, cfg.c, cfg.eps0, int(cfg.delay_rule if rule is None else rule),
       int(n), int(H), _ptr(ring),
       int(nobs), _ptr(idx), _ptr(E), _ptr(B))
    return E, B


def cell_index(x, y, z, shape_order: int = 1) -> np.ndarray:
    """Base node floor(xi - 1/2) of the 8 linear weights (Eq. 2.15), or for shape_order 2 the centre node floor(xi) of the
    27 S^(2) weights."""
    x, y, z = _f64(x), _f64(y), _f64(z)
    out = np.empty((x.shape[0], 3), dtype=np.int32)
    fn = _L().orc_cell_index_s2 if shape_order == 2 else _L().orc_cell_index
    fn(x.shape[0], _ptr(x), _ptr(y), _ptr(z), _ptr(out))
    return out


def deposit(cfg: OracleConfig, x, y, z, ux, uy, uz, qw, alive=None):
    """CIC deposit (Eqs. 2.15-2.19; 27-node S^(2) weights of Eq. 2.14 when cfg.shape_order == 2).  Positions in grid
    units, u = gamma v / c.  Returns [4][N] float64."""
    x, y, z, ux, uy, uz, qw = map(_f64, (x, y, z, ux, uy, uz, qw))
    al = None if alive is None else np.ascontiguousarray(alive, dtype=np.uint8)
    out = np.empty((4, cfg.N), dtype=np.float64)
    fn = _L().orc_deposit_s2 if cfg.shape_order == 2 else _L().orc_deposit
    fn(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.c, x.shape[0], _ptr(x), _ptr(y), _ptr(z),
                     _ptr(ux), _ptr(uy), _ptr(uz), _ptr(qw), _ptr(al), _ptr(out[0]), _ptr(out[1]), _ptr(out[2]),
                     _ptr(out[3]))
    return out


def interp(cfg: OracleConfig, x, y, z, F):
    """Eq. (2.20): F [3][N] -> [np][3] at the particles (virtual nodes count as zero)."""
    x, y, z = map(_f64, (x, y, z))
    F = _f64(F)
    out = np.empty((x.shape[0], 3), dtype=np.float64)
    fn = _L().orc_interp_s2 if cfg.shape_order == 2 else _L().orc_interp
    fn(cfg.nx, cfg.ny, cfg.nz, x.shape[0], _ptr(x), _ptr(y), _ptr(z), _ptr(F[0]), _ptr(F[1]), _ptr(F[2]),
                    _ptr(out))
    return out


def push(cfg: OracleConfig, x, y, z, ux, uy, uz, q_over_m, alive, E, B):
    """Interpolation + relativistic Boris + kill, in place on float64 / uint8 arrays (Eqs. 2.7-2.11, 2.20)."""
    for a in (x, y, z, ux, uy, uz, q_over_m):
        assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    assert alive.dtype == np.uint8
    E, B = _f64(E), _f64(B)
    Eext, Bext = _f64(cfg.Eext), _f64(cfg.Bext)
    _L().orc_push(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.dt, cfg.c, x.shape[0], _ptr(x), _ptr(y), _ptr(z),
                  _ptr(ux), _ptr(uy), _ptr(uz), _ptr(q_over_m), _ptr(alive), _ptr(E[0]), _ptr(E[1]), _ptr(E[2]),
                  _ptr(B[0]), _ptr(B[1]), _ptr(B[2]), _ptr(Eext), _ptr(Bext), int(cfg.shape_order))


class OracleJefi:
    """The same logical calls as the C-ABI on host arrays, fp64, for closed-loop parity.

    PIC step n: deposit(r^n, u^{n-1/2}) -> push_sources -> field_step -> push_particles.
    """

    def __init__(self, cfg: OracleConfig, ring_dtype=np.float64):
        self.cfg = cfg
        self.ring = np.zeros((cfg.H, 4, cfg.N), dtype=ring_dtype)  # zero before t0
        self.n = -1

    def push_sources(self, rho, jx, jy, jz) -> None:
        self.n += 1
        s = self.n % self.cfg.H
        self.ring[s, 0] = rho
        self.ring[s, 1] = jx
        self.ring[s, 2] = jy
        self.ring[s, 3] = jz

    def field_step(self, obs_idx=None):
        assert self.n >= 0, "field_step before any push_sources"
        return field(self.cfg, self.n, self.ring, obs_idx)

    def deposit(self, x, y, z, ux, uy, uz, qw, alive=None):
        return deposit(self.cfg, x, y, z, ux, uy, uz, qw, alive)

    def push_particles(self, x, y, z, ux, uy, uz, q_over_m, alive, E, B) -> None:
        push(self.cfg, x, y, z, ux, uy, uz, q_over_m, alive, E, B)

    def pic_step(self, part) -> tuple:
        """One whole step on a particle dict of float64 arrays (x,y,z,ux,uy,uz,qw,qm) + uint8 alive."""
        S = self.deposit(part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
        self.push_sources(S[0], S[1], S[2], S[3])
        E, B = self.field_step()
        self.push_particles(part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qm"],
                            part["alive"], E, B)
        return S, E, B
