"""Thin Python binding of the libjefi C-ABI (include/jefi.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of ``libjefi.so``; PyTorch supplies device memory and the
stream.  There is no CPU fallback: if the library is missing or no CUDA device is present the calls raise.
The functions carry the names of the C entry points; ``JefiContext`` is a small convenience wrapper around them.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence

_HERE = os.path.dirname(os.path.abspath(__file__))
# JEFI_LIBRARY selects another build of the same library, e.g. libjefi_checked.so (build.py --checked: the library's own
# device-side memory checks; JefiContext.close() then raises if any check fired).
LIB_PATH = os.environ.get("JEFI_LIBRARY") or os.path.join(_HERE, "libjefi.so")

JEFI_OK, JEFI_EINVAL, JEFI_ENOMEM, JEFI_ECUDA, JEFI_ESTATE = 0, -1, -2, -3, -4
JEFI_FIELD_AUTO, JEFI_FIELD_REFERENCE, JEFI_FIELD_TILED = 0, 1, 2
JEFI_DEPOSIT_AUTO, JEFI_DEPOSIT_DIRECT, JEFI_DEPOSIT_SORTED, JEFI_DEPOSIT_RUNS = 0, 1, 2, 3
JEFI_DELAY_NEAREST, JEFI_DELAY_LINEAR = 0, 1
JEFI_TILE_AUTO, JEFI_TILE_CELL, JEFI_TILE_DYAD = 0, 1, 2
JEFI_STATIC_MAX_PARTICLES, JEFI_STATIC_MAX_BINS = 1048576, 524288  # limits of jefi_deposit_static (include/jefi.h)

EXPORTS = [
    "jefi_create", "jefi_destroy", "jefi_last_error", "jefi_get_info", "jefi_deposit", "jefi_push_sources",
    "jefi_field_step", "jefi_field_step_slab", "jefi_push_particles", "jefi_field_step_host", "jefi_launch_count",
    "jefi_last_field_kernel_ms", "jefi_debug_delay_table", "jefi_debug_cell_index", "jefi_debug_history_slot",
    "jefi_debug_cell_order", "jefi_sort_particles", "jefi_field_impl_reason", "jefi_get_tile_info", "jefi_field_step_packed",
    "jefi_push_particles_packed", "jefi_field_kernel_ms", "jefi_debug_fp32_peak", "jefi_debug_check_errors", "jefi_pic_step",
    "jefi_debug_lds128_cycles", "jefi_deposit_static", "jefi_config_init",
]


class JefiError(RuntimeError):
    pass


class jefi_config(C.Structure):
    _fields_ = [
        ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double), ("dt", C.c_double),
        ("c", C.c_double), ("eps0", C.c_double),
        ("H", C.c_int), ("hist_cap", C.c_int),
        ("Eext", C.c_double * 3), ("Bext", C.c_double * 3),
        ("device", C.c_int), ("stream", C.c_void_p), ("field_impl", C.c_int), ("deposit_mode", C.c_int),
        ("delay_rule", C.c_int), ("shape_order", C.c_int), ("field_chunk", C.c_int), ("field_tile", C.c_int),
    ]


_lib = None


def load_library() -> C.CDLL:
    """dlopen libjefi.so (built by paper_2209_07944_b200.build.build_lib); fails loudly if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise JefiError(f"{LIB_PATH} not found: build it with `python -m paper_2209_07944_b200.build` "
                        "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, f32p, u8p = C.c_void_p, C.c_void_p, C.c_void_p
    lib.jefi_create.argtypes = [C.POINTER(jefi_config), C.POINTER(vp)]
    lib.jefi_create.restype = C.c_int
    lib.jefi_config_init.argtypes = [C.POINTER(jefi_config), C.c_ulong]
    lib.jefi_config_init.restype = C.c_int
    lib.jefi_destroy.argtypes = [vp]
    lib.jefi_destroy.restype = None
    lib.jefi_last_error.argtypes = [vp]
    lib.jefi_last_error.restype = C.c_char_p
    lib.jefi_get_info.argtypes = [vp, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_long),
                                  C.POINTER(C.c_long)]
    lib.jefi_get_info.restype = C.c_int
    lib.jefi_deposit.argtypes = [vp, C.c_long] + [f32p] * 7 + [u8p] + [f32p] * 4
    lib.jefi_deposit.restype = C.c_int
    lib.jefi_push_sources.argtypes = [vp] + [f32p] * 4
    lib.jefi_push_sources.restype = C.c_int
    lib.jefi_field_step.argtypes = [vp] + [f32p] * 6
    lib.jefi_field_step.restype = C.c_int
    lib.jefi_field_step_slab.argtypes = [vp, C.c_int, C.c_int] + [f32p] * 6
    lib.jefi_field_step_slab.restype = C.c_int
    lib.jefi_push_particles.argtypes = [vp, C.c_long] + [f32p] * 7 + [u8p] + [f32p] * 6
    lib.jefi_push_particles.restype = C.c_int
    lib.jefi_field_step_host.argtypes = [vp, f32p, f32p]
    lib.jefi_field_step_host.restype = C.c_int
    lib.jefi_launch_count.argtypes = [vp]
    lib.jefi_launch_count.restype = C.c_long
    lib.jefi_last_field_kernel_ms.argtypes = [vp]
    lib.jefi_last_field_kernel_ms.restype = C.c_float
    lib.jefi_field_kernel_ms.argtypes = [vp, C.c_int]
    lib.jefi_field_kernel_ms.restype = C.c_float
    lib.jefi_pic_step.argtypes = [vp, C.c_long] + [f32p] * 8 + [u8p] + [f32p] * 11
    lib.jefi_pic_step.restype = C.c_int
    lib.jefi_debug_check_errors.argtypes = [vp, C.POINTER(C.c_long * 4)]
    lib.jefi_debug_check_errors.restype = C.c_int
    lib.jefi_debug_fp32_peak.argtypes = [vp, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    lib.jefi_debug_fp32_peak.restype = C.c_int
    lib.jefi_debug_lds128_cycles.argtypes = [vp, C.c_int, C.POINTER(C.c_double)]
    lib.jefi_debug_lds128_cycles.restype = C.c_int
    lib.jefi_debug_delay_table.argtypes = [vp, vp]
    lib.jefi_debug_delay_table.restype = C.c_int
    lib.jefi_debug_cell_index.argtypes = [vp, C.c_long, f32p, f32p, f32p, vp]
    lib.jefi_debug_cell_index.restype = C.c_int
    lib.jefi_sort_particles.argtypes = [vp, C.c_long] + [f32p] * 8 + [u8p, vp]
    lib.jefi_sort_particles.restype = C.c_int
    lib.jefi_debug_cell_order.argtypes = [vp, C.c_long, f32p, f32p, f32p, u8p, vp, C.POINTER(C.c_long)]
    lib.jefi_debug_cell_order.restype = C.c_int
    lib.jefi_debug_history_slot.argtypes = [vp, C.c_int, f32p]
    lib.jefi_debug_history_slot.restype = C.c_int
    lib.jefi_field_impl_reason.argtypes = [vp]
    lib.jefi_field_impl_reason.restype = C.c_char_p
    lib.jefi_get_tile_info.argtypes = [vp, C.POINTER(C.c_int * 3), C.POINTER(C.c_int * 3), C.POINTER(C.c_int), C.POINTER(C.c_int),
                                       C.POINTER(C.c_int)]
    lib.jefi_get_tile_info.restype = C.c_int
    lib.jefi_field_step_packed.argtypes = [vp] + [f32p] * 7
    lib.jefi_field_step_packed.restype = C.c_int
    lib.jefi_push_particles_packed.argtypes = [vp, C.c_long] + [f32p] * 7 + [u8p, f32p]
    lib.jefi_push_particles_packed.restype = C.c_int
    lib.jefi_deposit_static.argtypes = ([C.c_int, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                         C.c_long] + [f32p] * 7 + [u8p] + [f32p] * 4 + [C.c_char_p, C.c_int])
    lib.jefi_deposit_static.restype = C.c_int
    _lib = lib
    return lib


def _check(handle, rc: int, what: str) -> None:
    if rc != JEFI_OK:
        msg = load_library().jefi_last_error(handle)
        raise JefiError(f"{what} failed with code {rc}: {msg.decode() if msg else ''}")


def _dev(t, dtype, n: Optional[int], name: str) -> int:
    """Device pointer of a contiguous CUDA tensor of the given dtype (and length, if given)."""
    import torch

    if t is None:
        return 0
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise JefiError(f"{name}: expected a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise JefiError(f"{name}: expected contiguous {dtype}, got {t.dtype} contiguous={t.is_contiguous()}")
    if n is not None and t.numel() != n:
        raise JefiError(f"{name}: expected {n} elements, got {t.numel()}")
    return t.data_ptr()


# ------------------------------------------------------------------------------------------------ C entry points
def jefi_create(nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, dt: float, c: float = 0.0,
                eps0: float = 0.0, H: int = 0, hist_cap: int = 0, Eext: Sequence[float] = (0, 0, 0),
                Bext: Sequence[float] = (0, 0, 0), device: int = 0, stream: int = 0,
                field_impl: int = JEFI_FIELD_AUTO, deposit_mode: int = JEFI_DEPOSIT_AUTO,
                delay_rule: int = JEFI_DELAY_NEAREST, shape_order: int = 1, field_chunk: int = 0,
                field_tile: int = 0) -> int:
    lib = load_library()
    cfg = jefi_config()
    if lib.jefi_config_init(C.byref(cfg), C.sizeof(jefi_config)) != JEFI_OK:  # this binding's struct is not the library's
        msg = lib.jefi_last_error(None)
        raise JefiError(f"jefi_config_init: {msg.decode() if msg else ''}")
    (cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, cfg.dt, cfg.c, cfg.eps0, cfg.H, cfg.hist_cap) = (nx, ny, nz, dx, dy, dz, dt, c, eps0, H, hist_cap)
    cfg.Eext, cfg.Bext = (C.c_double * 3)(*Eext), (C.c_double * 3)(*Bext)
    cfg.device, cfg.stream = device, C.c_void_p(stream)
    (cfg.field_impl, cfg.deposit_mode, cfg.delay_rule, cfg.shape_order, cfg.field_chunk, cfg.field_tile) = (
        field_impl, deposit_mode, delay_rule, shape_order, field_chunk, field_tile)
    h = C.c_void_p()
    rc = lib.jefi_create(C.byref(cfg), C.byref(h))
    if rc != JEFI_OK:
        msg = lib.jefi_last_error(None)
        raise JefiError(f"jefi_create failed with code {rc}: {msg.decode() if msg else ''}")
    return h.value


def jefi_destroy(handle: Optional[int]) -> None:
    if handle:
        load_library().jefi_destroy(handle)


def jefi_get_info(handle: int) -> dict:
    H, ndt, impl, step, rb = C.c_int(), C.c_int(), C.c_int(), C.c_long(), C.c_long()
    _check(handle, load_library().jefi_get_info(handle, C.byref(H), C.byref(ndt), C.byref(impl), C.byref(step),
                                                C.byref(rb)), "jefi_get_info")
    return dict(H=H.value, ndt=ndt.value, field_impl=impl.value, step=step.value, ring_bytes=rb.value)


def jefi_field_impl_reason(handle: int) -> str:
    msg = load_library().jefi_field_impl_reason(handle)
    return msg.decode() if msg else ""


def jefi_get_tile_info(handle: int) -> dict:
    ob, ts = (C.c_int * 3)(), (C.c_int * 3)()
    w, wp, ns = C.c_int(), C.c_int(), C.c_int()
    _check(handle, load_library().jefi_get_tile_info(handle, C.byref(ob), C.byref(ts), C.byref(w), C.byref(wp), C.byref(ns)),
           "jefi_get_tile_info")
    return dict(obs_tile=tuple(ob), src_tile=tuple(ts), window_slots=w.value, window_pitch=wp.value, source_split=ns.value)


def jefi_push_sources(handle: int, N: int, rho, jx, jy, jz) -> None:
    import torch

    f = torch.float32
    _check(handle, load_library().jefi_push_sources(handle, _dev(rho, f, N, "rho"), _dev(jx, f, N, "jx"),
                                                    _dev(jy, f, N, "jy"), _dev(jz, f, N, "jz")), "jefi_push_sources")


def jefi_field_step(handle: int, N: int, ex, ey, ez, bx, by, bz) -> None:
    import torch

    f = torch.float32
    ptrs = [_dev(t, f, N, n) for t, n in zip((ex, ey, ez, bx, by, bz), ("ex", "ey", "ez", "bx", "by", "bz"))]
    _check(handle, load_library().jefi_field_step(handle, *ptrs), "jefi_field_step")


def jefi_field_step_slab(handle: int, N: int, k0: int, k1: int, ex, ey, ez, bx, by, bz) -> None:
    import torch

    f = torch.float32
    ptrs = [_dev(t, f, N, n) for t, n in zip((ex, ey, ez, bx, by, bz), ("ex", "ey", "ez", "bx", "by", "bz"))]
    _check(handle, load_library().jefi_field_step_slab(handle, int(k0), int(k1), *ptrs), "jefi_field_step_slab")


def jefi_field_step_packed(handle: int, N: int, ex, ey, ez, bx, by, bz, eb_packed) -> None:
    import torch

    f = torch.float32
    ptrs = [_dev(t, f, N, n) for t, n in zip((ex, ey, ez, bx, by, bz), ("ex", "ey", "ez", "bx", "by", "bz"))]
    _check(handle, load_library().jefi_field_step_packed(handle, *ptrs, _dev(eb_packed, f, 8 * N, "eb_packed")),
           "jefi_field_step_packed")


def slab_range(nz: int, rank: int, world: int, edge: int = 8):
    """Observation z-planes [k0, k1) of `rank` out of `world`: whole layers of observation tiles (`edge` =
    jefi_get_tile_info()["obs_tile"][2]: 8, or 32 on nx <= 3 grids), spread as evenly as the layer count allows; ranks beyond
    the layer count get an empty range."""
    layers = (nz + edge - 1) // edge
    lo = (layers * rank) // world
    hi = (layers * (rank + 1)) // world
    return min(lo * edge, nz), min(hi * edge, nz)


def jefi_deposit(handle: int, N: int, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy, jz) -> None:
    import torch

    f = torch.float32
    np_ = x.numel()
    pin = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, qw), ("x", "y", "z", "ux", "uy", "uz", "qw"))]
    pal = _dev(alive, torch.uint8, np_, "alive") if alive is not None else 0
    pout = [_dev(t, f, N, n) for t, n in zip((rho, jx, jy, jz), ("rho", "jx", "jy", "jz"))]
    _check(handle, load_library().jefi_deposit(handle, np_, *pin, pal, *pout), "jefi_deposit")


def jefi_deposit_static(nx: int, ny: int, nz: int, dx: float, dy: float, dz: float, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy,
                        jz, c: float = 0.0, stream: Optional[int] = None) -> None:
    """Cell-sorted CIC deposit that allocates no device memory and needs no context (include/jefi.h, jefi_deposit_static).

    For programs that may not call cudaMalloc when they deposit: all device memory belongs to their own pool after start-up, or
    the step loop cannot afford the device-wide synchronisation an allocation can cause.  The sort scratch is a fixed 16 MiB
    array inside libjefi's CUDA module, so the list is limited to JEFI_STATIC_MAX_PARTICLES particles and the grid to
    (nx+1)(ny+1)(nz+1)+1 <= JEFI_STATIC_MAX_BINS; larger inputs raise JefiError (nothing is computed).  The output tensors
    are the caller's (this binding allocates nothing either).  Every call on a device shares that one array: keep calls on one
    stream, or order them with events; calls that overlap on the GPU corrupt each other.  Enqueues on `stream` (a
    cudaStream_t handle; default: torch's current stream of the tensors' device) and does not synchronise.  The first call on a
    device also looks up the array's device address; make it before starting any stream capture."""
    import torch

    f = torch.float32
    np_ = x.numel()
    N = nx * ny * nz
    pin = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, qw), ("x", "y", "z", "ux", "uy", "uz", "qw"))]
    pal = _dev(alive, torch.uint8, np_, "alive") if alive is not None else 0
    pout = [_dev(t, f, N, n) for t, n in zip((rho, jx, jy, jz), ("rho", "jx", "jy", "jz"))]
    dev = rho.device.index or 0
    if stream is None:
        stream = torch.cuda.current_stream(rho.device).cuda_stream
    err = C.create_string_buffer(512)
    rc = load_library().jefi_deposit_static(dev, C.c_void_p(stream), nx, ny, nz, dx, dy, dz, c, np_, *pin, pal, *pout, err, len(err))
    if rc != JEFI_OK:
        raise JefiError(f"jefi_deposit_static failed with code {rc}: {err.value.decode()}")


def jefi_push_particles(handle: int, N: int, x, y, z, ux, uy, uz, q_over_m, alive, ex, ey, ez, bx, by, bz) -> None:
    import torch

    f = torch.float32
    np_ = x.numel()
    pp = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, q_over_m), ("x", "y", "z", "ux", "uy", "uz", "q_over_m"))]
    pal = _dev(alive, torch.uint8, np_, "alive")
    pf = [_dev(t, f, N, n) for t, n in zip((ex, ey, ez, bx, by, bz), ("ex", "ey", "ez", "bx", "by", "bz"))]
    _check(handle, load_library().jefi_push_particles(handle, np_, *pp, pal, *pf), "jefi_push_particles")


def jefi_push_particles_packed(handle: int, N: int, x, y, z, ux, uy, uz, q_over_m, alive, eb_packed) -> None:
    import torch

    f = torch.float32
    np_ = x.numel()
    pp = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, q_over_m), ("x", "y", "z", "ux", "uy", "uz", "q_over_m"))]
    _check(handle, load_library().jefi_push_particles_packed(handle, np_, *pp, _dev(alive, torch.uint8, np_, "alive"),
                                                             _dev(eb_packed, f, 8 * N, "eb_packed")),
           "jefi_push_particles_packed")


def jefi_pic_step(handle: int, N: int, x, y, z, ux, uy, uz, qw, q_over_m, alive, rho, jx, jy, jz, ex, ey, ez, bx, by, bz,
                  eb_packed) -> None:
    import torch

    f = torch.float32
    np_ = x.numel()
    pp = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, qw, q_over_m), ("x", "y", "z", "ux", "uy", "uz", "qw", "q_over_m"))]
    pg = [_dev(t, f, N, n) for t, n in zip((rho, jx, jy, jz, ex, ey, ez, bx, by, bz), ("rho", "jx", "jy", "jz", "ex", "ey", "ez", "bx", "by", "bz"))]
    rc = load_library().jefi_pic_step(handle, np_, *pp, _dev(alive, torch.uint8, np_, "alive"), *pg, _dev(eb_packed, f, 8 * N, "eb_packed"))
    _check(handle, rc, "jefi_pic_step")


def jefi_sort_particles(handle: int, x, y, z, ux, uy, uz, qw, q_over_m, alive, tag=None) -> None:
    import torch

    f = torch.float32
    np_ = x.numel()
    pp = [_dev(t, f, np_, n) for t, n in zip((x, y, z, ux, uy, uz, qw, q_over_m), ("x", "y", "z", "ux", "uy", "uz", "qw", "q_over_m"))]
    rc = load_library().jefi_sort_particles(handle, np_, *pp, _dev(alive, torch.uint8, np_, "alive"),
                                            _dev(tag, torch.int32, np_, "tag"))
    _check(handle, rc, "jefi_sort_particles")


def jefi_field_step_host(handle: int, N: int, src_host, eb_host) -> None:
    """src_host: CPU float32 tensor [4*N] (pinned recommended); eb_host: CPU float32 tensor [6*N]."""
    import torch

    for t, n, name in ((src_host, 4 * N, "src_host"), (eb_host, 6 * N, "eb_host")):
        if t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.numel() != n:
            raise JefiError(f"{name}: expected a contiguous CPU float32 tensor of {n} elements")
    _check(handle, load_library().jefi_field_step_host(handle, src_host.data_ptr(), eb_host.data_ptr()),
           "jefi_field_step_host")


def jefi_launch_count(handle: int) -> int:
    return int(load_library().jefi_launch_count(handle))


def jefi_last_field_kernel_ms(handle: int) -> float:
    return float(load_library().jefi_last_field_kernel_ms(handle))


def jefi_field_kernel_ms(handle: int, calls_back: int) -> float:
    return float(load_library().jefi_field_kernel_ms(handle, int(calls_back)))


def jefi_debug_check_errors(handle: int):
    """(checked_build, [4 counters]) of the library's own device-side memory checks (include/jefi.h)."""
    e = (C.c_long * 4)()
    rc = load_library().jefi_debug_check_errors(handle, C.byref(e))
    if rc < 0:
        _check(handle, rc, "jefi_debug_check_errors")
    return rc == 1, list(e)


def jefi_debug_fp32_peak(handle: int, mode: int = 0) -> dict:
    """Measured FP32 FMA throughput of the device (TFLOP/s) and its SM count.  mode 0 / 1: scalar / packed FMA chains with
    shared multiplier and addend; 2 / 3: scalar / packed chains reading three registers of their own per FMA (include/jefi.h)."""
    tf, nsm = C.c_double(), C.c_int()
    _check(handle, load_library().jefi_debug_fp32_peak(handle, int(mode), C.byref(tf), C.byref(nsm)), "jefi_debug_fp32_peak")
    return dict(tflops=tf.value, sm_count=nsm.value, mode=int(mode))


def jefi_debug_lds128_cycles(handle: int, pattern: int) -> float:
    """SM cycles per warp-wide LDS.128 for an address pattern (include/jefi.h)."""
    cyc = C.c_double()
    _check(handle, load_library().jefi_debug_lds128_cycles(handle, int(pattern), C.byref(cyc)), "jefi_debug_lds128_cycles")
    return cyc.value


def jefi_debug_delay_table(handle: int, nx: int, ny: int, nz: int):
    import numpy as np

    out = np.empty((nz, ny, nx), dtype=np.int32)
    _check(handle, load_library().jefi_debug_delay_table(handle, out.ctypes.data), "jefi_debug_delay_table")
    return out


def jefi_debug_cell_order(handle: int, x, y, z, alive=None):
    """(order, n_alive): int32 CUDA tensor of the depositing particles in the internal cell order."""
    import torch

    np_ = x.numel()
    order = torch.empty(max(np_, 1), dtype=torch.int32, device=x.device)[:np_]
    na = C.c_long(0)
    f = torch.float32
    rc = load_library().jefi_debug_cell_order(handle, np_, _dev(x, f, np_, "x"), _dev(y, f, np_, "y"), _dev(z, f, np_, "z"),
                                              _dev(alive, torch.uint8, np_, "alive"), order.data_ptr(), C.byref(na))
    _check(handle, rc, "jefi_debug_cell_order")
    return order, na.value


def jefi_debug_cell_index(handle: int, x, y, z):
    import torch

    np_ = x.numel()
    out = torch.empty((np_, 3), dtype=torch.int32, device=x.device)
    f = torch.float32
    _check(handle, load_library().jefi_debug_cell_index(handle, np_, _dev(x, f, np_, "x"), _dev(y, f, np_, "y"),
                                                        _dev(z, f, np_, "z"), out.data_ptr()), "jefi_debug_cell_index")
    return out


def jefi_debug_history_slot(handle: int, N: int, steps_back: int, device):
    import torch

    out = torch.empty((4, N), dtype=torch.float32, device=device)
    _check(handle, load_library().jefi_debug_history_slot(handle, steps_back, out.data_ptr()), "jefi_debug_history_slot")
    return out


# ------------------------------------------------------------------------------------------------ convenience
@dataclass
class GridSpec:
    nx: int
    ny: int
    nz: int
    dx: float
    dy: float
    dz: float
    dt: float
    c: float = 0.0
    eps0: float = 0.0
    H: int = 0
    hist_cap: int = 0
    Eext: Sequence[float] = (0.0, 0.0, 0.0)
    Bext: Sequence[float] = (0.0, 0.0, 0.0)

    @property
    def N(self) -> int:
        return self.nx * self.ny * self.nz


class JefiContext:
    """Owns one jefi_ctx and the E/B/rho/J device tensors of a run; every method is one C-ABI call.

    The context enqueues on the torch stream that is current when it is created.  Created inside
    ``with torch.cuda.stream(torch.cuda.Stream())`` (any stream but the legacy default one) ``pic_step`` is one CUDA-graph
    launch per step (jefi_pic_step); the caller then keeps its own tensor work on that stream too."""

    def __init__(self, grid: GridSpec, device=None, field_impl: int = JEFI_FIELD_AUTO,
                 deposit_mode: int = JEFI_DEPOSIT_AUTO, sort_every: int = 0, delay_rule: int = JEFI_DELAY_NEAREST,
                 shape_order: int = 1, field_chunk: int = 0, packed_fields: bool = True, field_tile: int = 0):
        import torch

        if not torch.cuda.is_available():
            raise JefiError("no CUDA device: libjefi has no CPU fallback")
        self.device = torch.device(device if device is not None else "cuda:0")
        self.grid = grid
        self.N = grid.N
        torch.cuda.set_device(self.device)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        self.stream_handle = stream
        self.handle = jefi_create(grid.nx, grid.ny, grid.nz, grid.dx, grid.dy, grid.dz, grid.dt, grid.c, grid.eps0,
                                  grid.H, grid.hist_cap, grid.Eext, grid.Bext, self.device.index or 0, stream,
                                  field_impl, deposit_mode, delay_rule, shape_order, field_chunk, field_tile)
        self.info = jefi_get_info(self.handle)
        self.info["field_impl_reason"] = jefi_field_impl_reason(self.handle)
        self.tile_info = jefi_get_tile_info(self.handle)
        self.H = self.info["H"]
        # pic_step calls jefi_sort_particles every sort_every steps.  Default 0 = never: sorting permutes the caller's particle
        # arrays in place, so it is something a caller asks for, not something that happens to it.  PIC loops that want the
        # speed pass sort_every=8 (particles move at most c dt = dx/2 per step, and the deposit / push run 4-6x faster on a
        # cell-sorted list) and, if they identify particles by array position, a "tag" array in the
        # particle dict, which is permuted along.
        self.sort_every = int(sort_every)
        self._pic_steps = 0
        z = lambda k: torch.zeros((k, self.N), dtype=torch.float32, device=self.device)
        self.EB = z(6)   # ex ey ez bx by bz
        self.src = z(4)  # rho jx jy jz
        # interleaved copy of E, B written by the field kernel's epilogue and gathered by the push (pic_step only)
        self.EBp = torch.zeros(8 * self.N, dtype=torch.float32, device=self.device) if packed_fields else None

    def close(self) -> None:
        if getattr(self, "handle", None):
            checked, errs = jefi_debug_check_errors(self.handle) if _lib is not None else (False, [0])
            jefi_destroy(self.handle)
            self.handle = None
            if checked and any(errs):
                raise JefiError(f"libjefi (checked build): device-side memory checks fired: {errs}")

    __del__ = close

    def push_sources(self, src=None) -> None:
        s = self.src if src is None else src
        jefi_push_sources(self.handle, self.N, s[0], s[1], s[2], s[3])

    def field_step(self, out=None):
        o = self.EB if out is None else out
        jefi_field_step(self.handle, self.N, o[0], o[1], o[2], o[3], o[4], o[5])
        return o

    def field_step_slab(self, k0: int, k1: int, out=None):
        """E, B on the observation planes k0 <= k < k1 only (the other entries of `out` are left as they are)."""
        o = self.EB if out is None else out
        jefi_field_step_slab(self.handle, self.N, k0, k1, o[0], o[1], o[2], o[3], o[4], o[5])
        return o

    def field_step_packed(self):
        o = self.EB
        jefi_field_step_packed(self.handle, self.N, o[0], o[1], o[2], o[3], o[4], o[5], self.EBp)
        return o

    def push_particles_packed(self, part: dict) -> None:
        jefi_push_particles_packed(self.handle, self.N, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"],
                                   part["qm"], part["alive"], self.EBp)

    def slab_range(self, rank: int, world: int):
        return slab_range(self.grid.nz, rank, world, self.tile_info["obs_tile"][2])

    def deposit(self, part: dict, out=None):
        o = self.src if out is None else out
        jefi_deposit(self.handle, self.N, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"],
                     part["qw"], part.get("alive"), o[0], o[1], o[2], o[3])
        return o

    def push_particles(self, part: dict, EB=None) -> None:
        f = self.EB if EB is None else EB
        jefi_push_particles(self.handle, self.N, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"],
                            part["qm"], part["alive"], f[0], f[1], f[2], f[3], f[4], f[5])

    def sort_particles(self, part: dict) -> None:
        """Cell-sort the particle arrays in place (part["tag"], if present, is permuted along)."""
        jefi_sort_particles(self.handle, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"],
                            part["qm"], part["alive"], part.get("tag"))

    def pic_step(self, part: dict) -> None:
        """deposit -> push_sources -> field_step -> push_particles, all on one stream; with
        sort_every > 0 the particle arrays are first put in cell order every sort_every steps (jefi_sort_particles)."""
        if self.sort_every > 0 and self._pic_steps % self.sort_every == 0:
            self.sort_particles(part)
        self._pic_steps += 1
        if self.EBp is not None:
            s, o = self.src, self.EB
            jefi_pic_step(self.handle, self.N, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["qm"],
                          part["alive"], s[0], s[1], s[2], s[3], o[0], o[1], o[2], o[3], o[4], o[5], self.EBp)
        else:
            self.deposit(part)
            self.push_sources()
            self.field_step()
            self.push_particles(part)

    def launch_count(self) -> int:
        return jefi_launch_count(self.handle)

    def last_field_kernel_ms(self) -> float:
        return jefi_last_field_kernel_ms(self.handle)

    def field_kernel_ms(self, calls_back: int) -> float:
        return jefi_field_kernel_ms(self.handle, calls_back)
