"""Thin ctypes binding of include/jpet.h - argument marshalling only; every step runs in the CUDA kernels.

PyTorch appears here only as the owner of device memory and streams (tensor.data_ptr(), the current stream's
handle).  There is no CPU fallback: if libjpet.so is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os

from . import build as _build

JPET_OK, JPET_E_INVAL, JPET_E_CUDA, JPET_E_INTERNAL = 0, -1, -2, -3
JPET_MAX_PEERS = 16

EXPORTS = (
    "jpet_sensitivity", "jpet_mlem_iterate", "jpet_mlem_iterate_noalloc", "jpet_reconstruct", "jpet_mlem_begin", "jpet_mlem_accumulate",
    "jpet_mlem_end", "jpet_mlem_iterate_host", "jpet_reconstruct_host", "jpet_get_counters", "jpet_count_evals",
    "jpet_set_a3_coef", "jpet_get_a3_coef", "jpet_set_gamma", "jpet_get_gamma", "jpet_set_sigma_z_edge", "jpet_get_sigma_z_edge",
    "jpet_direct_histogram", "jpet_generate_events", "jpet_mlem_accumulator", "jpet_mlem_end_peers", "jpet_ipc_export",
    "jpet_ipc_open", "jpet_ipc_close", "jpet_plan_describe", "jpet_set_option", "jpet_get_option", "jpet_launch_count",
    "jpet_shape_name", "jpet_release", "jpet_last_error", "jpet_abi_version",
)


class Geometry(ctypes.Structure):
    _fields_ = [("R", ctypes.c_float), ("L", ctypes.c_float)]


class Sigmas(ctypes.Structure):
    _fields_ = [("sigma_z", ctypes.c_float), ("sigma_dl", ctypes.c_float)]


class Grid(ctypes.Structure):
    _fields_ = [("n_y", ctypes.c_int32), ("n_z", ctypes.c_int32), ("pixel", ctypes.c_float)]


class Primitive(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int32), ("cy", ctypes.c_float), ("cz", ctypes.c_float), ("hy", ctypes.c_float),
                ("hz", ctypes.c_float), ("phi_deg", ctypes.c_float), ("intensity", ctypes.c_float)]


class JpetError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"jpet error {code}: {text}")
        self.code = code


_lib = None


def library_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True) -> ctypes.CDLL:
    """Loads libjpet.so (building it in-tree with nvcc if it is missing and nvcc is there). Raises loudly otherwise."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        if not build_if_missing:
            raise FileNotFoundError(f"{path} is missing: run python -m paper_1502_07478_b200.build")
        path = _build.build()
    lib = ctypes.CDLL(path)
    p, i32, i64, u64p = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.POINTER(ctypes.c_uint64)
    G, S, Gr = ctypes.POINTER(Geometry), ctypes.POINTER(Sigmas), ctypes.POINTER(Grid)
    sigs = {
        "jpet_sensitivity": (ctypes.c_int, [G, Gr, p, p]),
        "jpet_mlem_iterate": (ctypes.c_int, [p, i64, G, S, Gr, p, p, p]),
        "jpet_mlem_iterate_noalloc": (ctypes.c_int, [p, i64, G, S, Gr, p, p, p]),
        "jpet_reconstruct": (ctypes.c_int, [p, i64, G, S, Gr, p, p, i32, p]),
        "jpet_mlem_begin": (ctypes.c_int, [G, S, Gr, p, p]),
        "jpet_mlem_accumulate": (ctypes.c_int, [p, i64, p]),
        "jpet_mlem_end": (ctypes.c_int, [p, p, p]),
        "jpet_mlem_iterate_host": (ctypes.c_int, [p, i64, G, S, Gr, p, p, i64]),
        "jpet_reconstruct_host": (ctypes.c_int, [p, i64, G, S, Gr, p, p, i32, i64]),
        "jpet_get_counters": (ctypes.c_int, [u64p, u64p, p]),
        "jpet_count_evals": (ctypes.c_int, [p, i64, G, S, Gr, u64p, u64p, p]),
        "jpet_set_a3_coef": (ctypes.c_int, [ctypes.c_float]),
        "jpet_get_a3_coef": (ctypes.c_float, []),
        "jpet_set_gamma": (ctypes.c_int, [ctypes.c_float]),
        "jpet_get_gamma": (ctypes.c_float, []),
        "jpet_set_sigma_z_edge": (ctypes.c_int, [ctypes.c_float]),
        "jpet_get_sigma_z_edge": (ctypes.c_float, []),
        "jpet_direct_histogram": (ctypes.c_int, [p, i64, G, Gr, p, u64p, p]),
        "jpet_generate_events": (ctypes.c_int, [ctypes.POINTER(Primitive), i32, i64, i64, G, S, ctypes.c_uint64, p, p]),
        "jpet_mlem_accumulator": (ctypes.c_int, [ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(i64)]),
        "jpet_mlem_end_peers": (ctypes.c_int, [p, p, ctypes.POINTER(ctypes.c_void_p), i32, p]),
        "jpet_ipc_export": (ctypes.c_int, [p, p]),
        "jpet_ipc_open": (ctypes.c_int, [p, ctypes.POINTER(ctypes.c_void_p)]),
        "jpet_ipc_close": (ctypes.c_int, [p]),
        "jpet_shape_name": (ctypes.c_char_p, [i32]),
        "jpet_plan_describe": (i64, [G, S, Gr, p, i32, p, i64]),
        "jpet_set_option": (ctypes.c_int, [ctypes.c_char_p, i64]),
        "jpet_get_option": (i64, [ctypes.c_char_p]),
        "jpet_launch_count": (ctypes.c_uint64, []),
        "jpet_release": (None, []),
        "jpet_last_error": (ctypes.c_char_p, []),
        "jpet_abi_version": (ctypes.c_int, []),
    }
    for name, (res, args) in sigs.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    _lib = lib
    return lib


def _check(rc: int) -> None:
    if rc != JPET_OK:
        raise JpetError(rc, load().jpet_last_error().decode())


def _stream_handle(stream) -> int:
    if stream is None:
        import torch

        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


def _dev_f32(t, numel: int | None, what: str) -> int:
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{what} must be a contiguous float32 CUDA tensor")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} must hold {numel} elements, has {t.numel()}")
    return t.data_ptr()


def _host_f32(t, numel: int | None, what: str) -> int:
    import torch

    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous():
        raise TypeError(f"{what} must be a contiguous float32 CPU tensor (pinned for asynchronous copies)")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{what} must hold {numel} elements, has {t.numel()}")
    return t.data_ptr()


def _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel):
    return Geometry(R, L), Sigmas(sigma_z, sigma_dl), Grid(n_y, n_z, pixel)


def _events_ptr(events, dev: bool):
    if events.dim() != 2 or events.shape[1] != 3:
        raise ValueError("events must be [n, 3]")
    return (_dev_f32 if dev else _host_f32)(events, None, "events"), int(events.shape[0])


# ---- the calls, same names as include/jpet.h ---------------------------------------------------------------
def jpet_sensitivity(R, L, n_y, n_z, pixel, s_dev, stream=None):
    g, _, gr = _structs(R, L, 1.0, 1.0, n_y, n_z, pixel)
    _check(load().jpet_sensitivity(g, gr, _dev_f32(s_dev, n_y * n_z, "s_dev"), _stream_handle(stream)))
    return s_dev


def jpet_mlem_iterate(events_dev, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_in_dev, rho_out_dev, stream=None):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_dev, True)
    _check(load().jpet_mlem_iterate(ev, n, g, s, gr, _dev_f32(rho_in_dev, n_y * n_z, "rho_in_dev"),
                                    _dev_f32(rho_out_dev, n_y * n_z, "rho_out_dev"), _stream_handle(stream)))
    return rho_out_dev


NOALLOC_MAX_PIXELS = 512 * 512      # JPET_NOALLOC_MAX_PIXELS of include/jpet.h


def jpet_mlem_iterate_noalloc(events_dev, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_in_dev, rho_out_dev, stream=None):
    """jpet_mlem_iterate for callers that cannot allocate device memory when the iteration is due (a loop with a latency
    budget, a host program whose pool owns all of HBM, a no-allocation-after-start-up rule): the library's scratch is a
    fixed array compiled into it, so the call never reaches cudaMalloc. Images of up to NOALLOC_MAX_PIXELS pixels; the
    slow direct kernel; calls share the scratch, so do not let two of them overlap on the GPU. See include/jpet.h."""
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_dev, True)
    _check(load().jpet_mlem_iterate_noalloc(ev, n, g, s, gr, _dev_f32(rho_in_dev, n_y * n_z, "rho_in_dev"),
                                            _dev_f32(rho_out_dev, n_y * n_z, "rho_out_dev"), _stream_handle(stream)))
    return rho_out_dev


def jpet_reconstruct(events_dev, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_init_dev, rho_out_dev, n_iter, stream=None):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_dev, True)
    init = None if rho_init_dev is None else _dev_f32(rho_init_dev, n_y * n_z, "rho_init_dev")
    _check(load().jpet_reconstruct(ev, n, g, s, gr, init, _dev_f32(rho_out_dev, n_y * n_z, "rho_out_dev"),
                                   int(n_iter), _stream_handle(stream)))
    return rho_out_dev


def jpet_mlem_begin(R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_in_dev, stream=None):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    _check(load().jpet_mlem_begin(g, s, gr, _dev_f32(rho_in_dev, n_y * n_z, "rho_in_dev"), _stream_handle(stream)))


def jpet_mlem_accumulate(events_dev, stream=None):
    ev, n = _events_ptr(events_dev, True)
    _check(load().jpet_mlem_accumulate(ev, n, _stream_handle(stream)))


def jpet_mlem_end(rho_in_dev, rho_out_dev, stream=None):
    _check(load().jpet_mlem_end(_dev_f32(rho_in_dev, None, "rho_in_dev"), _dev_f32(rho_out_dev, None, "rho_out_dev"),
                                _stream_handle(stream)))
    return rho_out_dev


def jpet_mlem_iterate_host(events_host, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_in_host, rho_out_host, chunk_events=0):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_host, False)
    _check(load().jpet_mlem_iterate_host(ev, n, g, s, gr, _host_f32(rho_in_host, n_y * n_z, "rho_in_host"),
                                         _host_f32(rho_out_host, n_y * n_z, "rho_out_host"), int(chunk_events)))
    return rho_out_host


def jpet_reconstruct_host(events_host, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_init_host, rho_out_host, n_iter,
                          chunk_events=0):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_host, False)
    init = None if rho_init_host is None else _host_f32(rho_init_host, n_y * n_z, "rho_init_host")
    _check(load().jpet_reconstruct_host(ev, n, g, s, gr, init, _host_f32(rho_out_host, n_y * n_z, "rho_out_host"),
                                        int(n_iter), int(chunk_events)))
    return rho_out_host


def jpet_get_counters(stream=None):
    """(n_evals, n_skipped) of the most recent iteration; synchronises the stream."""
    a, b = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(load().jpet_get_counters(ctypes.byref(a), ctypes.byref(b), _stream_handle(stream)))
    return int(a.value), int(b.value)


def jpet_count_evals(events_dev, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, stream=None):
    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    ev, n = _events_ptr(events_dev, True)
    a, b = ctypes.c_uint64(0), ctypes.c_uint64(0)
    _check(load().jpet_count_evals(ev, n, g, s, gr, ctypes.byref(a), ctypes.byref(b), _stream_handle(stream)))
    return int(a.value), int(b.value)


def jpet_set_a3_coef(k: float) -> None:
    _check(load().jpet_set_a3_coef(float(k)))


def jpet_get_a3_coef() -> float:
    return float(load().jpet_get_a3_coef())


PLAN_FIELDS = ("variant", "degree", "warps_per_event", "groups_per_cta", "cap_a", "cap_b", "HS", "WZ", "Sy", "Sz", "Hy", "Hz",
               "chunk", "smem_bytes", "tiled", "nr_min", "nr_max")


def jpet_plan_describe(R, L, sigma_z, sigma_dl, n_y, n_z, pixel):
    """Host-side plan of the event kernel (no GPU needed): dict of PLAN_FIELDS plus "table", the task table as a
    numpy uint32 array [row count - nr_min][32 * warps_per_event] (empty when the plan has none)."""
    import numpy as np

    g, s, gr = _structs(R, L, sigma_z, sigma_dl, n_y, n_z, pixel)
    out = (ctypes.c_int64 * 18)()
    n = load().jpet_plan_describe(g, s, gr, out, 18, None, 0)
    if n < 0:
        _check(int(n))
    tab = np.zeros(int(n), dtype=np.uint32)
    if n:
        load().jpet_plan_describe(g, s, gr, out, 18, tab.ctypes.data, int(n))
    plan = dict(zip(PLAN_FIELDS, [int(v) for v in out]))
    plan["variant_low"] = int(out[17])     # degree-3 instance for the events of degree class 1 (-1: one class)
    lanes = 32 * max(plan["warps_per_event"], 1)
    plan["table"] = tab.reshape(-1, lanes) if n else tab
    return plan


def jpet_set_gamma(gamma: float) -> None:
    _check(load().jpet_set_gamma(float(gamma)))


def jpet_get_gamma() -> float:
    return float(load().jpet_get_gamma())


def jpet_set_sigma_z_edge(eta: float) -> None:
    _check(load().jpet_set_sigma_z_edge(float(eta)))


def jpet_get_sigma_z_edge() -> float:
    return float(load().jpet_get_sigma_z_edge())


def jpet_direct_histogram(events_dev, R, L, n_y, n_z, pixel, hist_dev, count_outside=True, stream=None):
    """Eq. 2 + binning (Fig. 4b): increments hist_dev (int32 CUDA tensor [n_y*n_z], read as uint32); returns the number of
    events outside the grid (synchronises) or None when count_outside is False (asynchronous)."""
    import torch

    if not isinstance(hist_dev, torch.Tensor) or not hist_dev.is_cuda or hist_dev.dtype != torch.int32 or not hist_dev.is_contiguous() \
            or hist_dev.numel() != n_y * n_z:
        raise TypeError(f"hist_dev must be a contiguous int32 CUDA tensor of {n_y * n_z} elements")
    g, _, gr = _structs(R, L, 1.0, 1.0, n_y, n_z, pixel)
    ev, n = _events_ptr(events_dev, True)
    out = ctypes.c_uint64(0)
    _check(load().jpet_direct_histogram(ev, n, g, gr, hist_dev.data_ptr(), ctypes.byref(out) if count_outside else None,
                                        _stream_handle(stream)))
    return int(out.value) if count_outside else None


def jpet_generate_events(phantom, n, R, L, sigma_z, sigma_dl, seed, events_dev, first=0, stream=None):
    """Event simulation on the device. phantom: sequence of objects with kind ('E' / 'B' or 0 / 1), cy, cz, hy, hz, phi_deg,
    intensity (synth.Primitive fits); events_dev: float32 CUDA tensor [n, 3], written."""
    prims = (Primitive * len(phantom))()
    for k, q in enumerate(phantom):
        kind = {"E": 0, "B": 1}.get(q.kind, q.kind)
        prims[k] = Primitive(int(kind), q.cy, q.cz, q.hy, q.hz, q.phi_deg, q.intensity)
    g, s, _ = _structs(R, L, sigma_z, sigma_dl, 1, 1, 1.0)
    ev, n_ev = _events_ptr(events_dev, True)
    if n_ev != n:
        raise ValueError(f"events_dev must be [{n}, 3]")
    _check(load().jpet_generate_events(prims, len(phantom), int(n), int(first), g, s, int(seed), ev, _stream_handle(stream)))
    return events_dev


class _DeviceArray:
    """A raw device pointer seen through __cuda_array_interface__ (so that torch can wrap it without a copy)."""

    def __init__(self, ptr: int, n: int):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<f4", "data": (ptr, False), "version": 2}


def device_view(ptr: int, n: int):
    """float32 CUDA tensor over n floats at device pointer ptr (no copy, no ownership)."""
    import torch

    return torch.as_tensor(_DeviceArray(int(ptr), int(n)), device="cuda")


def jpet_mlem_accumulator():
    """The accumulator of the open iteration (between begin and end) as a float32 CUDA tensor view [n_z * n_y]."""
    ptr, n = ctypes.c_void_p(0), ctypes.c_int64(0)
    _check(load().jpet_mlem_accumulator(ctypes.byref(ptr), ctypes.byref(n)))
    return device_view(ptr.value, n.value)


def jpet_mlem_end_peers(rho_in_dev, rho_out_dev, peers, stream=None):
    """Step 4 with the accumulator read as the sum of `peers`: CUDA tensors or raw device pointers (IPC mappings)."""
    arr = (ctypes.c_void_p * len(peers))()
    for k, q in enumerate(peers):
        arr[k] = q if isinstance(q, int) else _dev_f32(q, None, "peer accumulator")
    _check(load().jpet_mlem_end_peers(_dev_f32(rho_in_dev, None, "rho_in_dev"), _dev_f32(rho_out_dev, None, "rho_out_dev"), arr,
                                      len(peers), _stream_handle(stream)))
    return rho_out_dev


def jpet_ipc_export(dev_ptr: int) -> bytes:
    buf = ctypes.create_string_buffer(64)
    _check(load().jpet_ipc_export(ctypes.c_void_p(int(dev_ptr)), buf))
    return buf.raw


def jpet_ipc_open(handle: bytes) -> int:
    out = ctypes.c_void_p(0)
    _check(load().jpet_ipc_open(ctypes.create_string_buffer(handle, 64), ctypes.byref(out)))
    return int(out.value)


def jpet_ipc_close(dev_ptr: int) -> None:
    _check(load().jpet_ipc_close(ctypes.c_void_p(int(dev_ptr))))


def jpet_shape_name(shape: int) -> str:
    return load().jpet_shape_name(int(shape)).decode()


def jpet_set_option(name: str, value: int) -> None:
    _check(load().jpet_set_option(name.encode(), int(value)))


def jpet_get_option(name: str) -> int:
    return int(load().jpet_get_option(name.encode()))


def jpet_launch_count() -> int:
    return int(load().jpet_launch_count())


def jpet_release() -> None:
    load().jpet_release()


def jpet_last_error() -> str:
    return load().jpet_last_error().decode()


def jpet_abi_version() -> int:
    return int(load().jpet_abi_version())
