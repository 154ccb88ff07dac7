"""ctypes front end of the fp64 CPU oracle (oracle/jpet_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this package.  It imports nothing from paper_1502_07478_b200 and the
CUDA path imports nothing from here.  Argument marshalling only - all arithmetic is in the C file, which
cites the paper passage each function follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "jpet_oracle.c")
_LIB = os.path.join(_HERE, "libjpet_oracle.so")
_lib = None

DEFAULT_A3_COEF = 2.0  # reading R5: a = d e / d theta; 1.0 = Eq. 9 as printed


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, -O2, OpenMP); returns the path of the shared library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-fno-fast-math", "-ffp-contract=off", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    d, i, i64, p = ctypes.c_double, ctypes.c_int, ctypes.c_int64, ctypes.c_void_p
    lib.jo_eq1_delta_l.restype = d
    lib.jo_eq1_delta_l.argtypes = [d] * 5
    lib.jo_eq2.restype = None
    lib.jo_eq2.argtypes = [d, d, d, d, p]
    lib.jo_sensitivity.restype = d
    lib.jo_sensitivity.argtypes = [d] * 4
    lib.jo_sensitivity_image.restype = None
    lib.jo_sensitivity_image.argtypes = [d, d, i, i, d, p]
    lib.jo_bCb.restype = d
    lib.jo_bCb.argtypes = [d] * 5
    lib.jo_kernel.restype = d
    lib.jo_kernel.argtypes = [d] * 9
    lib.jo_kernel_events.restype = None
    lib.jo_kernel_events.argtypes = [p, i64, d, d, d, d, d, d, p, p]
    lib.jo_bbox_half_extents.restype = None
    lib.jo_bbox_half_extents.argtypes = [d, d, d, p]
    lib.jo_mlem_iterate.restype = i
    lib.jo_mlem_iterate.argtypes = [p, i64, d, d, d, d, i, i, d, d, p, p, i, i, p, p]
    lib.jo_reconstruct.restype = i
    lib.jo_reconstruct.argtypes = [p, i64, d, d, d, d, i, i, d, d, p, p, i, i, p, p]
    lib.jo_num_threads.restype = i
    lib.jo_num_threads.argtypes = []
    lib.jo_set_gamma.restype = None
    lib.jo_set_gamma.argtypes = [d]
    lib.jo_get_gamma.restype = d
    lib.jo_get_gamma.argtypes = []
    lib.jo_set_sigma_z_edge.restype = None
    lib.jo_set_sigma_z_edge.argtypes = [d]
    lib.jo_get_sigma_z_edge.restype = d
    lib.jo_get_sigma_z_edge.argtypes = []
    lib.jo_sigma_z_at.restype = d
    lib.jo_sigma_z_at.argtypes = [d, d, d]
    lib.jo_cinv.restype = None
    lib.jo_cinv.argtypes = [d, d, d, d, d, p]
    lib.jo_bCb_c.restype = d
    lib.jo_bCb_c.argtypes = [d, d, d, p]
    lib.jo_kernel_c.restype = d
    lib.jo_kernel_c.argtypes = [d, d, d, d, d, d, p, d]
    lib.jo_kernel_exact.restype = d
    lib.jo_kernel_exact.argtypes = [d, d, p, d, p, i]
    lib.jo_bbox_half_extents_c.restype = None
    lib.jo_bbox_half_extents_c.argtypes = [d, p, p]
    lib.jo_set_exact_kernel.restype = None
    lib.jo_set_exact_kernel.argtypes = [i]
    lib.jo_get_exact_kernel.restype = i
    lib.jo_get_exact_kernel.argtypes = []
    lib.jo_direct_histogram.restype = ctypes.c_uint64
    lib.jo_direct_histogram.argtypes = [p, i64, d, i, i, d, p]
    lib.jo_direct_pixel_coords.restype = None
    lib.jo_direct_pixel_coords.argtypes = [p, i64, d, i, i, d, p]
    lib.jo_generate_events.restype = i
    lib.jo_generate_events.argtypes = [p, i, i64, i64, d, d, d, d, ctypes.c_uint64, p]
    lib.jo_kernel_exact_events.restype = None
    lib.jo_kernel_exact_events.argtypes = [p, i64, d, d, d, d, d, d, i, p]
    lib.jo_philox4x32_10_block.restype = None
    lib.jo_philox4x32_10_block.argtypes = [p, p, p]
    _lib = lib
    return lib


def set_gamma(gamma: float) -> None:
    """Off-diagonal coefficient gamma of C^-1 (Eq. 12); 0 = the paper's diagonal case (default).
    Process-wide: set it back to 0 after use."""
    _load().jo_set_gamma(float(gamma))


def get_gamma() -> float:
    return float(_load().jo_get_gamma())


def set_sigma_z_edge(eta: float) -> None:
    """Coefficient eta of sigma_z(z) = sigma_z (1 + eta min(1, (2z/L)^2)) (reading R22); 0 = constant
    (default).  Process-wide: set it back to 0 after use."""
    _load().jo_set_sigma_z_edge(float(eta))


def get_sigma_z_edge() -> float:
    return float(_load().jo_get_sigma_z_edge())


def sigma_z_at(z_hit, L, sigma_z) -> float:
    return float(_load().jo_sigma_z_at(z_hit, L, sigma_z))


def cinv(z_u_t, z_d_t, L, sigma_z, sigma_dl) -> np.ndarray:
    """Eq. 12 for one event: 3x3 inverse covariance at the event's hit positions (current gamma, eta)."""
    C = np.empty((3, 3), dtype=np.float64)
    _load().jo_cinv(z_u_t, z_d_t, L, sigma_z, sigma_dl, C.ctypes.data)
    return C


def bCb_c(dy, dz, tan_t, Cinv) -> float:
    C = np.ascontiguousarray(Cinv, dtype=np.float64)
    return float(_load().jo_bCb_c(dy, dz, tan_t, C.ctypes.data))


def kernel_c(y, z, tan_t, y_t, z_t, R, Cinv, a3_coef=DEFAULT_A3_COEF) -> float:
    """Eq. 7-11 with a given inverse covariance matrix."""
    C = np.ascontiguousarray(Cinv, dtype=np.float64)
    return float(_load().jo_kernel_c(y, z, tan_t, y_t, z_t, R, C.ctypes.data, a3_coef))


def kernel_exact(y, z, event, R, Cinv, n_theta=20001) -> float:
    """The integral Eq. 7 approximates: int dtheta/pi N(e~; e(y, z, theta), C), trapezoid rule."""
    C = np.ascontiguousarray(Cinv, dtype=np.float64)
    e = np.ascontiguousarray(event, dtype=np.float64)
    return float(_load().jo_kernel_exact(y, z, e.ctypes.data, R, C.ctypes.data, int(n_theta)))


def kernel_exact_events(events, y, z, R, L, sigma_z, sigma_dl, n_theta=2001) -> np.ndarray:
    """kernel_exact for events float64 [n, 3] at one pixel, each event with its own matrix (cinv)."""
    ev = np.ascontiguousarray(events, dtype=np.float64)
    P = np.empty(ev.shape[0], dtype=np.float64)
    _load().jo_kernel_exact_events(ev.ctypes.data, ev.shape[0], y, z, R, L, sigma_z, sigma_dl, int(n_theta), P.ctypes.data)
    return P


def philox4x32_10(counter, key):
    c, k, o = (np.ascontiguousarray(v, dtype=np.uint32) for v in (counter, key, np.zeros(4)))
    _load().jo_philox4x32_10_block(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return [int(v) for v in o]


def bbox_half_extents_c(tan_t, Cinv):
    C = np.ascontiguousarray(Cinv, dtype=np.float64)
    out = (ctypes.c_double * 2)()
    _load().jo_bbox_half_extents_c(tan_t, C.ctypes.data, out)
    return float(out[0]), float(out[1])


def set_exact_kernel(n_theta: int) -> None:
    """> 0: mlem_iterate / reconstruct use kernel_exact with that many nodes instead of Eq. 7.  Process-wide."""
    _load().jo_set_exact_kernel(int(n_theta))


def direct_histogram(events, R, n_y, n_z, pixel, hist=None):
    """Eq. 2 + binning (Fig. 4b). Returns (hist uint32 [n_y, n_z], n_outside); `hist` is incremented when given."""
    ev = _events_f32(events)
    h = np.zeros((n_y, n_z), dtype=np.uint32) if hist is None else hist
    assert h.dtype == np.uint32 and h.flags.c_contiguous and h.size == n_y * n_z
    out = _load().jo_direct_histogram(ev.ctypes.data, ev.shape[0], R, n_y, n_z, pixel, h.ctypes.data)
    return h, int(out)


def direct_pixel_coords(events, R, n_y, n_z, pixel) -> np.ndarray:
    """Eq. 2 in fp64: (c_y, c_z) of every event in pixels from the lower edge of the grid, float64 [n, 2]; the event lies in
    pixel (floor c_y, floor c_z). NaN for events with a non-finite component."""
    ev = _events_f32(events)
    out = np.empty((ev.shape[0], 2), dtype=np.float64)
    _load().jo_direct_pixel_coords(ev.ctypes.data, ev.shape[0], R, n_y, n_z, pixel, out.ctypes.data)
    return out


def generate_events(phantom, n, R, L, sigma_z, sigma_dl, seed, first=0) -> np.ndarray:
    """Counter-based event simulation (same generator as the CUDA path, fp64). phantom: objects with kind ('E'/'B'),
    cy, cz, hy, hz, phi_deg, intensity. Returns float32 [n, 3]."""
    kinds = {"E": 0.0, "B": 1.0, 0: 0.0, 1: 1.0}
    prims = np.array([[kinds[q.kind], q.cy, q.cz, q.hy, q.hz, q.phi_deg, q.intensity] for q in phantom], dtype=np.float64)
    out = np.empty((n, 3), dtype=np.float32)
    rc = _load().jo_generate_events(prims.ctypes.data, len(phantom), int(n), int(first), R, L, sigma_z, sigma_dl,
                                    int(seed), out.ctypes.data)
    if rc != 0:
        raise RuntimeError("jo_generate_events failed")
    return out


def num_threads() -> int:
    return int(_load().jo_num_threads())


def eq1_delta_l(e_y, e_z, z_u, z_d, R) -> float:
    """Eq. 1."""
    return float(_load().jo_eq1_delta_l(e_y, e_z, z_u, z_d, R))


def eq2(z_u_t, z_d_t, dl_t, R):
    """Eq. 2: returns (tan theta~, y~, z~)."""
    out = (ctypes.c_double * 3)()
    _load().jo_eq2(z_u_t, z_d_t, dl_t, R, out)
    return float(out[0]), float(out[1]), float(out[2])


def sensitivity(y, z, R, L) -> float:
    """Eq. 4 clamped at 0."""
    return float(_load().jo_sensitivity(y, z, R, L))


def sensitivity_image(R, L, n_y, n_z, pixel) -> np.ndarray:
    s = np.empty((n_y, n_z), dtype=np.float64)
    _load().jo_sensitivity_image(R, L, n_y, n_z, pixel, s.ctypes.data)
    return s


def bCb(dy, dz, tan_t, sigma_z, sigma_dl) -> float:
    """b C^-1 b, first line of B.3."""
    return float(_load().jo_bCb(dy, dz, tan_t, sigma_z, sigma_dl))


def kernel(y, z, tan_t, y_t, z_t, R, sigma_z, sigma_dl, a3_coef=DEFAULT_A3_COEF) -> float:
    """Eq. 7-12, no truncation."""
    return float(_load().jo_kernel(y, z, tan_t, y_t, z_t, R, sigma_z, sigma_dl, a3_coef))


def kernel_events(events, y, z, R, sigma_z, sigma_dl, a3_coef=DEFAULT_A3_COEF):
    """P(e~_j | pixel (y, z)) for events float64 [n, 3]; returns (P [n], inside-3-sigma mask [n])."""
    ev = np.ascontiguousarray(events, dtype=np.float64)
    P = np.empty(ev.shape[0], dtype=np.float64)
    inside = np.empty(ev.shape[0], dtype=np.uint8)
    _load().jo_kernel_events(ev.ctypes.data, ev.shape[0], y, z, R, sigma_z, sigma_dl, a3_coef,
                             P.ctypes.data, inside.ctypes.data)
    return P, inside.astype(bool)


def bbox_half_extents(tan_t, sigma_z, sigma_dl):
    """Appendix B.2: (h_y, h_z) of the 3-sigma ellipse's bounding box."""
    out = (ctypes.c_double * 2)()
    _load().jo_bbox_half_extents(tan_t, sigma_z, sigma_dl, out)
    return float(out[0]), float(out[1])


def _events_f32(events) -> np.ndarray:
    ev = np.ascontiguousarray(events, dtype=np.float32)
    if ev.ndim != 2 or ev.shape[1] != 3:
        raise ValueError("events must be [n, 3]")
    return ev


def mlem_iterate(events, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, rho_in, a3_coef=DEFAULT_A3_COEF,
                 brute=False, n_threads=0):
    """One MLEM iteration (Eq. 3 / Listing 1). Returns (rho_out float64 [n_y, n_z], n_evals, n_skipped)."""
    ev = _events_f32(events)
    rin = np.ascontiguousarray(rho_in, dtype=np.float64).reshape(n_y, n_z)
    rout = np.empty((n_y, n_z), dtype=np.float64)
    ne, ns = ctypes.c_uint64(0), ctypes.c_uint64(0)
    rc = _load().jo_mlem_iterate(ev.ctypes.data, ev.shape[0], R, L, sigma_z, sigma_dl, n_y, n_z, pixel, a3_coef,
                                 rin.ctypes.data, rout.ctypes.data, int(bool(brute)), int(n_threads),
                                 ctypes.addressof(ne), ctypes.addressof(ns))
    if rc != 0:
        raise RuntimeError("jo_mlem_iterate failed")
    return rout, int(ne.value), int(ns.value)


def reconstruct(events, R, L, sigma_z, sigma_dl, n_y, n_z, pixel, n_iter, rho_init=None,
                a3_coef=DEFAULT_A3_COEF, n_threads=0):
    """n_iter MLEM iterations from rho_init (None => ones). Returns (rho float64, n_evals, n_skipped) of the last."""
    ev = _events_f32(events)
    rinit = None if rho_init is None else np.ascontiguousarray(rho_init, dtype=np.float64).reshape(n_y, n_z)
    rout = np.empty((n_y, n_z), dtype=np.float64)
    ne, ns = ctypes.c_uint64(0), ctypes.c_uint64(0)
    rc = _load().jo_reconstruct(ev.ctypes.data, ev.shape[0], R, L, sigma_z, sigma_dl, n_y, n_z, pixel, a3_coef,
                                None if rinit is None else rinit.ctypes.data, rout.ctypes.data, int(n_iter),
                                int(n_threads), ctypes.addressof(ne), ctypes.addressof(ns))
    if rc != 0:
        raise RuntimeError("jo_reconstruct failed")
    return rout, int(ne.value), int(ns.value)
