"""ctypes front end of the CPU oracle (oracle/velo_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs. The product package never imports this module, and this
module never imports the product's CUDA path. See the header of velo_oracle.c for what the
oracle computes and which passages it follows (§5).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "velo_oracle.c")
_LIB = os.path.join(_HERE, "libvelo_oracle.so")
CFLAGS = ["-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared"]

STATE_NAMES = ("x", "y", "tx", "ty", "z", "cxx", "cxtx", "ctxtx", "cyy", "cyty", "ctyty", "chi2", "n_hits")


class Params(ctypes.Structure):
    """SURVEY.md §8(b)/(c) parameter block with the default reading (A5, A6, A7, A10, A12, A13)."""
    _fields_ = [
        ("phi_window_seed", ctypes.c_int32), ("phi_window_fwd", ctypes.c_int32),
        ("max_scatter_seed", ctypes.c_float), ("max_scatter_fwd", ctypes.c_float),
        ("max_scatter_weak", ctypes.c_float),
        ("max_skipped", ctypes.c_uint32),
        ("sigma_hit", ctypes.c_float),
        ("max_chi2_ndof", ctypes.c_float),
        ("clone_num", ctypes.c_uint32), ("clone_den", ctypes.c_uint32),
    ]


def default_params(pitch: float = 0.055) -> Params:
    return Params(phi_window_seed=300, phi_window_fwd=300, max_scatter_seed=0.1, max_scatter_fwd=0.1,
                  max_scatter_weak=0.05, max_skipped=1,
                  sigma_hit=float(np.float32(pitch / np.sqrt(12.0))), max_chi2_ndof=100.0,
                  clone_num=1, clone_den=3)


def _compile(src: str, lib: str) -> None:
    """gcc into a temporary file, then an atomic rename: forked test workers may all find the library
    stale at the same moment."""
    tmp = f"{lib}.{os.getpid()}.tmp"
    subprocess.run(["gcc", *CFLAGS, "-o", tmp, src, "-lm"], check=True)
    os.replace(tmp, lib)


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        _compile(_SRC, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        vp = ctypes.c_void_p
        L.vo_phi16.argtypes = [ctypes.c_float, ctypes.c_float]
        L.vo_phi16.restype = ctypes.c_int16
        L.vo_scatter.argtypes = [ctypes.c_float] * 9
        L.vo_scatter.restype = ctypes.c_float
        L.vo_in_window.argtypes = [ctypes.c_int16, ctypes.c_int16, ctypes.c_int32]
        L.vo_in_window.restype = ctypes.c_int
        L.vo_sort_event.argtypes = [ctypes.c_uint32, vp, vp, vp, ctypes.c_uint32, vp, vp, vp]
        L.vo_sort_event.restype = ctypes.c_int
        L.vo_fit.argtypes = [ctypes.c_uint32, vp, vp, vp, ctypes.c_float, vp]
        L.vo_fit.restype = None
        L.vo_reconstruct.argtypes = [ctypes.c_uint32, vp, vp, vp, vp, vp, ctypes.c_uint32,
                                     ctypes.POINTER(Params)]
        L.vo_reconstruct.restype = vp
        L.vo_result_sizes.argtypes = [vp, vp]
        L.vo_result_copy.argtypes = [vp, vp, vp, vp, vp]
        L.vo_result_free.argtypes = [vp]
        L.vo_event_candidates.argtypes = [ctypes.c_uint32, vp, vp, vp, vp, ctypes.c_uint32,
                                          ctypes.POINTER(Params), ctypes.c_uint32] + [vp] * 7
        L.vo_event_candidates.restype = ctypes.c_int
        _lib = L
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def phi16(x, y) -> np.ndarray:
    L = lib()
    x = np.atleast_1d(_f32(x)); y = np.atleast_1d(_f32(y))
    return np.array([L.vo_phi16(float(a), float(b)) for a, b in zip(x, y)], dtype=np.int16)


def scatter(h0, h1, h2) -> float:
    a = [float(np.float32(v)) for v in (*h0, *h1, *h2)]
    return float(lib().vo_scatter(*a))


def in_window(phi, c, W) -> bool:
    return bool(lib().vo_in_window(int(phi), int(c), int(W)))


def sort_event(x, y, module, n_modules):
    x = _f32(x); y = _f32(y); module = np.ascontiguousarray(module, dtype=np.uint8)
    n = x.shape[0]
    perm = np.zeros(max(n, 1), np.uint32); phi = np.zeros(max(n, 1), np.int16)
    mod_off = np.zeros(n_modules + 1, np.uint32)
    rc = lib().vo_sort_event(n, _p(x), _p(y), _p(module), n_modules, _p(perm), _p(phi), _p(mod_off))
    if rc != 0:
        raise ValueError("module id out of range")
    return perm[:n], phi[:n], mod_off


def fit(hx, hy, hz, sigma_hit) -> np.ndarray:
    hx = _f32(hx); hy = _f32(hy); hz = _f32(hz)
    out = np.zeros(13, np.float32)
    lib().vo_fit(hx.shape[0], _p(hx), _p(hy), _p(hz), float(np.float32(sigma_hit)), _p(out))
    return out


def reconstruct(x, y, z, module, event_offsets, n_modules: int, params: Params | None = None) -> dict:
    """Run the oracle on a batch (host numpy arrays). Returns a dict with event_track_offsets,
    track_hit_offsets, track_hits (global original hit indices), states (13 x n_tracks f32; the
    last plane holds n_hits as u32 bits), n_tracks, n_track_hits, status, n_candidates."""
    L = lib()
    P = params if params is not None else default_params()
    x = _f32(x); y = _f32(y); z = _f32(z)
    module = np.ascontiguousarray(module, dtype=np.uint8)
    off = np.ascontiguousarray(event_offsets, dtype=np.uint32)
    n_events = off.shape[0] - 1
    h = L.vo_reconstruct(n_modules, _p(x), _p(y), _p(z), _p(module), _p(off), n_events, ctypes.byref(P))
    try:
        sz = np.zeros(4, np.uint32)
        L.vo_result_sizes(h, _p(sz))
        nt, nth = int(sz[0]), int(sz[1])
        status = int(np.int32(sz[2]))
        eto = np.zeros(n_events + 1, np.uint32); tho = np.zeros(nt + 1, np.uint32)
        th = np.zeros(max(nth, 1), np.uint32); st = np.zeros((13, max(nt, 1)), np.float32)
        L.vo_result_copy(h, _p(eto), _p(tho), _p(th), _p(st))
    finally:
        L.vo_result_free(h)
    return {"event_track_offsets": eto, "track_hit_offsets": tho, "track_hits": th[:nth],
            "states": st[:, :nt], "n_tracks": nt, "n_track_hits": nth, "status": status,
            "n_candidates": int(sz[3])}


def event_candidates(x, y, z, module, n_modules: int, params: Params | None = None, cap: int = 0) -> dict:
    """Single-event dump of every candidate track (before and after filtering) and of the sort,
    for the brute-force pins."""
    P = params if params is not None else default_params()
    x = _f32(x); y = _f32(y); z = _f32(z); module = np.ascontiguousarray(module, dtype=np.uint8)
    n = x.shape[0]
    cap = cap or max(n, 1)
    hits = np.zeros((cap, 32), np.uint32); meta = np.zeros((cap, 8), np.uint32)
    states = np.zeros((cap, 13), np.float32)
    perm = np.zeros(max(n, 1), np.uint32); phi = np.zeros(max(n, 1), np.int16)
    mod_off = np.zeros(n_modules + 1, np.uint32); flags = np.zeros(max(n, 1), np.uint8)
    nc = lib().vo_event_candidates(n, _p(x), _p(y), _p(z), _p(module), n_modules, ctypes.byref(P), cap,
                                   _p(hits), _p(meta), _p(states), _p(perm), _p(phi), _p(mod_off), _p(flags))
    if nc < 0:
        raise ValueError("bad input")
    nc = min(nc, cap)
    key = meta[:nc, 5].astype(np.uint64) | (meta[:nc, 6].astype(np.uint64) << np.uint64(32))
    return {"n_cand": nc, "hits": hits[:nc], "n": meta[:nc, 0], "centre": meta[:nc, 1],
            "pass": meta[:nc, 2].astype(bool), "survive": meta[:nc, 3].astype(bool), "lost": meta[:nc, 4],
            "key": key, "seed_scatter": meta[:nc, 7].copy().view(np.float32), "states": states[:nc],
            "perm": perm[:n], "phi": phi[:n], "mod_off": mod_off, "flags": flags[:n].astype(bool)}


# ---- the steps after the hot path: oracle/velo_next_oracle.c ------------------
_SRC_NEXT = os.path.join(_HERE, "velo_next_oracle.c")
_LIB_NEXT = os.path.join(_HERE, "libvelo_next_oracle.so")
MS_THETA2_DEFAULT = float(np.float32(9.0e-8))      # K-1: (0.3 mrad)^2


class PvParams(ctypes.Structure):
    """DESIGN.md §2 readings P-1 ... P-6 (paper silent)."""
    _fields_ = [("z_min", ctypes.c_float), ("bin_width", ctypes.c_float), ("n_bins", ctypes.c_uint32),
                ("seed_min_sum", ctypes.c_uint32), ("seed_half_window", ctypes.c_uint32),
                ("chi2_max", ctypes.c_float), ("n_iterations", ctypes.c_uint32), ("min_tracks", ctypes.c_uint32),
                ("max_pv_per_event", ctypes.c_uint32)]


def default_pv_params() -> PvParams:
    return PvParams(z_min=-300.0, bin_width=0.25, n_bins=2400, seed_min_sum=5, seed_half_window=6,
                    chi2_max=16.0, n_iterations=4, min_tracks=4, max_pv_per_event=32)


def build_next(force: bool = False) -> str:
    if force or not os.path.exists(_LIB_NEXT) or os.path.getmtime(_LIB_NEXT) < os.path.getmtime(_SRC_NEXT):
        _compile(_SRC_NEXT, _LIB_NEXT)
    return _LIB_NEXT


_lib_next = None


def lib_next():
    global _lib_next
    if _lib_next is None:
        L = ctypes.CDLL(build_next())
        vp = ctypes.c_void_p
        L.vn_pixel_decode.argtypes = [ctypes.c_uint32, vp, ctypes.c_double, ctypes.c_double, vp, ctypes.c_uint32,
                                      vp, vp, vp, vp]
        L.vn_pixel_decode.restype = ctypes.c_int
        L.vn_kalman.argtypes = [ctypes.c_uint32, vp, vp, vp, ctypes.c_float, ctypes.c_float, vp]
        L.vn_kalman.restype = None
        L.vn_kalman_tracks.argtypes = [ctypes.c_uint32, vp, vp, vp, vp, vp, ctypes.c_float, ctypes.c_float, vp]
        L.vn_kalman_tracks.restype = None
        L.vn_pv_bin.argtypes = [ctypes.c_float, ctypes.c_float, ctypes.c_float, ctypes.c_uint32]
        L.vn_pv_bin.restype = ctypes.c_int32
        L.vn_pv_seeds.argtypes = [vp, ctypes.c_uint32, ctypes.POINTER(PvParams), vp]
        L.vn_pv_seeds.restype = ctypes.c_uint32
        L.vn_pv_event.argtypes = [vp, ctypes.c_size_t, ctypes.c_uint32, ctypes.c_uint32, ctypes.POINTER(PvParams), vp]
        L.vn_pv_event.restype = ctypes.c_uint32
        L.vn_pv_find.argtypes = [ctypes.c_uint32, vp, vp, ctypes.c_size_t, ctypes.POINTER(PvParams), vp, vp,
                                 ctypes.c_uint32]
        L.vn_pv_find.restype = ctypes.c_uint32
        _lib_next = L
    return _lib_next


def kalman(hx, hy, hz, sigma_hit, ms_theta2=MS_THETA2_DEFAULT) -> np.ndarray:
    """K-1 ... K-5 on one track's hits (discovery order). 13 state words (O-11 layout)."""
    hx = _f32(hx); hy = _f32(hy); hz = _f32(hz)
    out = np.zeros(13, np.float32)
    lib_next().vn_kalman(hx.shape[0], _p(hx), _p(hy), _p(hz), float(np.float32(sigma_hit)),
                         float(np.float32(ms_theta2)), _p(out))
    return out


def kalman_tracks(res: dict, x, y, z, sigma_hit, ms_theta2=MS_THETA2_DEFAULT) -> np.ndarray:
    """The filter on every track of a reconstruct() result. Returns 13 x n_tracks f32."""
    x = _f32(x); y = _f32(y); z = _f32(z)
    nt = int(res["n_tracks"])
    tho = np.ascontiguousarray(res["track_hit_offsets"], dtype=np.uint32)
    th = np.ascontiguousarray(res["track_hits"], dtype=np.uint32)
    if th.shape[0] == 0:
        th = np.zeros(1, np.uint32)
    out = np.zeros((13, max(nt, 1)), np.float32)
    if nt:
        lib_next().vn_kalman_tracks(nt, _p(tho), _p(th), _p(x), _p(y), _p(z), float(np.float32(sigma_hit)),
                                    float(np.float32(ms_theta2)), _p(out))
    return out[:, :nt]


def pv_bin(z, params: PvParams | None = None) -> int:
    P = params if params is not None else default_pv_params()
    inv_w = float(np.float32(1.0) / np.float32(P.bin_width))
    return int(lib_next().vn_pv_bin(float(np.float32(z)), P.z_min, inv_w, P.n_bins))


def pv_seeds(hist, params: PvParams | None = None) -> np.ndarray:
    P = params if params is not None else default_pv_params()
    h = np.ascontiguousarray(hist, dtype=np.uint32)
    out = np.zeros(32, np.uint32)
    n = lib_next().vn_pv_seeds(_p(h), h.shape[0], ctypes.byref(P), _p(out))
    return out[:n].copy()


def pv_find(event_track_offsets, states, params: PvParams | None = None) -> dict:
    """P-1 ... P-6 on a batch of reconstructed tracks (states: 13 x n_tracks). Returns
    event_pv_offsets (u32[n_events+1]), pvs (5 x n_pvs f32: x, y, z, sum of weights, n_tracks bits)."""
    P = params if params is not None else default_pv_params()
    eto = np.ascontiguousarray(event_track_offsets, dtype=np.uint32)
    st = np.ascontiguousarray(states, dtype=np.float32)
    ne = eto.shape[0] - 1
    cap = max(32 * ne, 1)
    epo = np.zeros(ne + 1, np.uint32)
    pvs = np.zeros((5, cap), np.float32)
    stride = st.shape[1] if st.ndim == 2 and st.shape[1] > 0 else 1
    if st.size == 0:
        st = np.zeros((13, 1), np.float32)
    n = lib_next().vn_pv_find(ne, _p(eto), _p(st), stride, ctypes.byref(P), _p(epo), _p(pvs), cap)
    return {"event_pv_offsets": epo, "pvs": pvs[:, :n].copy(), "n_pvs": int(n)}


def pixel_decode(pixel, module_z, pitch: float = 0.055, half_shift_x: float = 0.0) -> dict:
    """F-1, F-2: packed pixel addresses -> x, y, z (f32), module (u8)."""
    px = np.ascontiguousarray(pixel, dtype=np.uint32)
    mz = _f32(module_z)
    n = px.shape[0]
    x = np.zeros(max(n, 1), np.float32); y = np.zeros(max(n, 1), np.float32); z = np.zeros(max(n, 1), np.float32)
    m = np.zeros(max(n, 1), np.uint8)
    if n:
        rc = lib_next().vn_pixel_decode(n, _p(px), float(pitch), float(half_shift_x), _p(mz), mz.shape[0],
                                        _p(x), _p(y), _p(z), _p(m))
        if rc != 0:
            raise ValueError("module id out of range")
    return {"x": x[:n], "y": y[:n], "z": z[:n], "module": m[:n]}
