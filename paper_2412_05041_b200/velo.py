"""Thin ctypes binding of libvelo (include/velo.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C-ABI; PyTorch supplies device
memory and streams. There is no CPU fallback: if libvelo.so is missing or no CUDA device is
present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_float, c_int, c_int32, c_size_t, c_uint32, c_void_p

import numpy as np

from . import build as _build

VELO_OK, VELO_ERR_ARG, VELO_ERR_GEOMETRY, VELO_ERR_WORKSPACE = 0, -1, -2, -3
VELO_ERR_CUDA, VELO_ERR_CAPACITY, VELO_ERR_INPUT = -4, -5, -6
VELO_ERR_STATIC_LIMIT = -7
VELO_PV_STATIC_MAX_EVENTS, VELO_PV_STATIC_MAX_TRACKS = 4096, 2097152
VELO_MAX_MODULES, VELO_MAX_EVENT_HITS, VELO_N_STATE = 32, 65535, 13
VELO_PATH_DEFAULT, VELO_PATH_SLAB_ONLY = 0, 1
VELO_N_STAGE_EVENTS = 6
VELO_N_SUMMARY = 8
STATE_NAMES = ("x", "y", "tx", "ty", "z", "cxx", "cxtx", "ctxtx", "cyy", "cyty", "ctyty", "chi2", "n_hits")
ERROR_NAMES = {0: "VELO_OK", -1: "VELO_ERR_ARG", -2: "VELO_ERR_GEOMETRY", -3: "VELO_ERR_WORKSPACE",
               -4: "VELO_ERR_CUDA", -5: "VELO_ERR_CAPACITY", -6: "VELO_ERR_INPUT",
               -7: "VELO_ERR_STATIC_LIMIT"}

# every symbol include/velo.h declares
EXPORTS = ("velo_version", "velo_geometry_load", "velo_geometry_free", "velo_geometry_n_modules",
           "velo_params_default", "velo_workspace_bytes", "velo_workspace_bytes_opts", "velo_reconstruct",
           "velo_reconstruct_opts", "velo_scheduler_create",
           "velo_scheduler_free", "velo_scheduler_run_host",
           "velo_kalman_fit", "velo_pv_params_default", "velo_pv_workspace_bytes", "velo_pv_find",
           "velo_reconstruct_pixels", "velo_scheduler_run_host_pixels", "velo_kalman_fit_pixels", "velo_pv_find_static")


class VeloError(RuntimeError):
    def __init__(self, code: int, where: str):
        super().__init__(f"{where}: {ERROR_NAMES.get(code, code)}")
        self.code = code


class GeometryDesc(ctypes.Structure):
    _fields_ = [("n_modules", c_uint32), ("module_z", POINTER(c_float)), ("r_in", c_float),
                ("r_out", c_float), ("pitch", c_float), ("half_shift_x", c_float), ("module_z_b", POINTER(c_float))]


class Params(ctypes.Structure):
    _fields_ = [("phi_window_seed", c_int32), ("phi_window_fwd", c_int32),
                ("max_scatter_seed", c_float), ("max_scatter_fwd", c_float), ("max_scatter_weak", c_float),
                ("max_skipped", c_uint32), ("sigma_hit", c_float), ("max_chi2_ndof", c_float),
                ("clone_num", c_uint32), ("clone_den", c_uint32)]


class Hits(ctypes.Structure):
    _fields_ = [("x", c_void_p), ("y", c_void_p), ("z", c_void_p), ("module", c_void_p),
                ("event_offsets", c_void_p), ("n_events", c_uint32), ("n_hits", c_uint32)]


class PixelHits(ctypes.Structure):
    _fields_ = [("pixel", c_void_p), ("event_offsets", c_void_p), ("n_events", c_uint32), ("n_hits", c_uint32)]


class PixelFormat(ctypes.Structure):
    _fields_ = [("pitch", ctypes.c_double), ("half_shift_x", ctypes.c_double)]


class Tracks(ctypes.Structure):
    _fields_ = [("event_track_offsets", c_void_p), ("track_hit_offsets", c_void_p), ("track_hits", c_void_p),
                ("states", c_void_p), ("cap_tracks", c_uint32), ("cap_track_hits", c_uint32),
                ("summary", c_void_p)]


class LaunchOptions(ctypes.Structure):
    _fields_ = [("stage_events", c_void_p * VELO_N_STAGE_EVENTS), ("ctas_per_sm", c_uint32),
                ("path", c_uint32), ("track_group", c_uint32),
                ("track_teams", c_uint32), ("fit_teams", c_uint32), ("sort_teams", c_uint32),
                ("pool_units", c_uint32)]


class PvParams(ctypes.Structure):
    _fields_ = [("z_min", c_float), ("bin_width", c_float), ("n_bins", c_uint32), ("seed_min_sum", c_uint32),
                ("seed_half_window", c_uint32), ("chi2_max", c_float), ("n_iterations", c_uint32),
                ("min_tracks", c_uint32), ("max_pv_per_event", c_uint32)]


class Pvs(ctypes.Structure):
    _fields_ = [("event_pv_offsets", c_void_p), ("pvs", c_void_p), ("cap_pvs", c_uint32), ("summary", c_void_p)]


VELO_N_PV_WORDS = 5
MS_THETA2_DEFAULT = 9.0e-8      # K-1: (0.3 mrad)^2

_lib = None


def lib():
    """Loads libvelo.so (built in-tree by paper_2412_05041_b200.build). Fails loudly if absent."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if os.environ.get("VELO_TIMELINE_BUILD"):          # bench.py --timeline: the instrumented build
            path = _build.build_timeline()
        if not os.path.exists(path):
            raise RuntimeError(f"{path} is missing: run `python -m paper_2412_05041_b200.build` "
                               "(there is no fallback path)")
        L = ctypes.CDLL(path)
        L.velo_version.restype = ctypes.c_char_p
        L.velo_geometry_load.argtypes = [POINTER(GeometryDesc), POINTER(c_void_p)]
        L.velo_geometry_load.restype = c_int
        L.velo_geometry_free.argtypes = [c_void_p]
        L.velo_geometry_free.restype = None
        L.velo_geometry_n_modules.argtypes = [c_void_p]
        L.velo_geometry_n_modules.restype = c_uint32
        L.velo_params_default.argtypes = [c_void_p, POINTER(Params)]
        L.velo_params_default.restype = None
        L.velo_workspace_bytes.argtypes = [c_uint32, c_uint32, c_uint32, c_uint32]
        L.velo_workspace_bytes.restype = c_size_t
        L.velo_reconstruct.argtypes = [c_void_p, POINTER(Hits), POINTER(Params), POINTER(Tracks), c_void_p,
                                       c_size_t, c_void_p]
        L.velo_reconstruct.restype = c_int
        L.velo_workspace_bytes_opts.argtypes = [c_uint32, c_uint32, c_uint32, c_uint32, POINTER(LaunchOptions)]
        L.velo_workspace_bytes_opts.restype = c_size_t
        L.velo_reconstruct_opts.argtypes = [c_void_p, POINTER(Hits), POINTER(Params), POINTER(Tracks), c_void_p,
                                            c_size_t, c_void_p, POINTER(LaunchOptions)]
        L.velo_reconstruct_opts.restype = c_int
        L.velo_scheduler_create.argtypes = [c_void_p, c_uint32, c_uint32, c_uint32, POINTER(c_void_p)]
        L.velo_scheduler_create.restype = c_int
        L.velo_scheduler_free.argtypes = [c_void_p]
        L.velo_scheduler_free.restype = None
        L.velo_scheduler_run_host.argtypes = [c_void_p, POINTER(Params), POINTER(Hits), c_void_p, c_uint32,
                                              POINTER(Tracks)]
        L.velo_scheduler_run_host.restype = c_int
        L.velo_reconstruct_pixels.argtypes = [c_void_p, POINTER(PixelHits), POINTER(PixelFormat), POINTER(Params),
                                              POINTER(Tracks), c_void_p, c_size_t, c_void_p, POINTER(LaunchOptions)]
        L.velo_reconstruct_pixels.restype = c_int
        L.velo_scheduler_run_host_pixels.argtypes = [c_void_p, POINTER(Params), POINTER(PixelHits), POINTER(PixelFormat),
                                                     c_void_p, c_uint32, POINTER(Tracks)]
        L.velo_scheduler_run_host_pixels.restype = c_int
        L.velo_kalman_fit_pixels.argtypes = [c_void_p, POINTER(PixelHits), POINTER(PixelFormat), POINTER(Tracks), c_float,
                                             c_float, c_void_p, c_void_p]
        L.velo_kalman_fit_pixels.restype = c_int
        L.velo_kalman_fit.argtypes = [POINTER(Hits), POINTER(Tracks), c_float, c_float, c_void_p, c_void_p]
        L.velo_kalman_fit.restype = c_int
        L.velo_pv_params_default.argtypes = [POINTER(PvParams)]
        L.velo_pv_params_default.restype = None
        L.velo_pv_workspace_bytes.argtypes = [c_uint32, c_uint32]
        L.velo_pv_workspace_bytes.restype = c_size_t
        L.velo_pv_find.argtypes = [POINTER(Tracks), c_uint32, POINTER(PvParams), POINTER(Pvs), c_void_p, c_size_t,
                                   c_void_p]
        L.velo_pv_find.restype = c_int
        L.velo_pv_find_static.argtypes = [POINTER(Tracks), c_uint32, POINTER(PvParams), POINTER(Pvs), c_void_p]
        L.velo_pv_find_static.restype = c_int
        _lib = L
    return _lib


def velo_version() -> str:
    return lib().velo_version().decode()


class Geometry:
    """Owns a velo_geometry_t handle."""

    def __init__(self, module_z, r_in=5.1, r_out=42.0, pitch=0.055, half_shift_x=0.0, module_z_b=None):
        z = np.ascontiguousarray(module_z, dtype=np.float32)
        zb = None if module_z_b is None else np.ascontiguousarray(module_z_b, dtype=np.float32)
        if zb is not None and zb.shape != z.shape:
            raise ValueError("module_z_b: one plane per module")
        desc = GeometryDesc(n_modules=z.shape[0], module_z=z.ctypes.data_as(POINTER(c_float)),
                            r_in=r_in, r_out=r_out, pitch=pitch, half_shift_x=half_shift_x,
                            module_z_b=None if zb is None else zb.ctypes.data_as(POINTER(c_float)))
        h = c_void_p()
        rc = lib().velo_geometry_load(byref(desc), byref(h))
        if rc != VELO_OK:
            raise VeloError(rc, "velo_geometry_load")
        self.handle = h
        self.n_modules = int(lib().velo_geometry_n_modules(h))

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:
            _lib.velo_geometry_free(h)


def velo_geometry_load(module_z, **kw) -> Geometry:
    return Geometry(module_z, **kw)


def velo_params_default(geometry: Geometry | None = None) -> Params:
    p = Params()
    lib().velo_params_default(geometry.handle if geometry is not None else None, byref(p))
    return p


def velo_workspace_bytes(n_events: int, n_hits: int, cap_tracks: int, cap_track_hits: int) -> int:
    return int(lib().velo_workspace_bytes(n_events, n_hits, cap_tracks, cap_track_hits))


def velo_workspace_bytes_opts(n_events: int, n_hits: int, cap_tracks: int, cap_track_hits: int,
                              opts: LaunchOptions | None) -> int:
    return int(lib().velo_workspace_bytes_opts(n_events, n_hits, cap_tracks, cap_track_hits,
                                               byref(opts) if opts is not None else None))


# ---- device-side helpers (PyTorch = device memory and streams only) -----------------------------
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libvelo needs a CUDA device (there is no CPU path)")
    return torch


def default_capacities(n_events: int, n_hits: int) -> tuple[int, int]:
    """Practical output sizing of include/velo.h: cap_tracks = n_hits/4 + n_events,
    cap_track_hits = 2*n_hits (+1 so that an empty batch still has non-zero capacities)."""
    return n_hits // 4 + n_events + 1, 2 * n_hits + 1


class DeviceHits:
    """Hits of a batch resident in HBM: x, y, z (f32), module (u8), event_offsets (u32 stored in an
    int32 tensor: torch has no unsigned 32-bit arithmetic, the bits are what the library reads)."""

    def __init__(self, x, y, z, module, event_offsets, device="cuda"):
        torch = _torch()
        f = lambda a, dt: torch.as_tensor(np.ascontiguousarray(a, dtype=dt)).to(device, non_blocking=False)
        self.x, self.y, self.z = f(x, np.float32), f(y, np.float32), f(z, np.float32)
        self.module = f(module, np.uint8)
        off = np.ascontiguousarray(event_offsets, dtype=np.uint32)
        self.event_offsets = torch.as_tensor(off.view(np.int32)).to(device)
        self.n_events = off.shape[0] - 1
        self.n_hits = int(off[-1]) - int(off[0]) if off.shape[0] else 0
        self.first_hit = int(off[0]) if off.shape[0] else 0

    def slice_struct(self, e0: int = 0, e1: int | None = None, n_hits: int | None = None) -> Hits:
        """velo_hits_t for events [e0, e1): same hit arrays, a slice of the offsets."""
        e1 = self.n_events if e1 is None else e1
        return Hits(x=self.x.data_ptr(), y=self.y.data_ptr(), z=self.z.data_ptr(), module=self.module.data_ptr(),
                    event_offsets=self.event_offsets.data_ptr() + 4 * e0, n_events=e1 - e0,
                    n_hits=self.n_hits if n_hits is None else n_hits)


class DeviceTracks:
    """Caller-allocated output buffers of one batch (velo_tracks_t) plus its workspace."""

    def __init__(self, n_events: int, n_hits: int, cap_tracks: int | None = None, cap_track_hits: int | None = None,
                 device="cuda", opts: LaunchOptions | None = None):
        torch = _torch()
        ct, ch = default_capacities(n_events, n_hits)
        self.cap_tracks = int(cap_tracks if cap_tracks is not None else ct)
        self.cap_track_hits = int(cap_track_hits if cap_track_hits is not None else ch)
        self.n_events = n_events
        i32 = dict(dtype=torch.int32, device=device)
        self.event_track_offsets = torch.empty(n_events + 1, **i32)
        self.track_hit_offsets = torch.empty(self.cap_tracks + 1, **i32)
        self.track_hits = torch.empty(self.cap_track_hits, **i32)
        self.states = torch.empty((VELO_N_STATE, self.cap_tracks), dtype=torch.float32, device=device)
        self.summary = torch.zeros(VELO_N_SUMMARY, **i32)
        self.workspace_bytes = velo_workspace_bytes_opts(n_events, n_hits, self.cap_tracks, self.cap_track_hits, opts)
        self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=device)
        self.workspace_ptr = (self.workspace.data_ptr() + 255) // 256 * 256

    def struct(self) -> Tracks:
        return Tracks(event_track_offsets=self.event_track_offsets.data_ptr(),
                      track_hit_offsets=self.track_hit_offsets.data_ptr(), track_hits=self.track_hits.data_ptr(),
                      states=self.states.data_ptr(), cap_tracks=self.cap_tracks, cap_track_hits=self.cap_track_hits,
                      summary=self.summary.data_ptr())

    def to_host(self) -> dict:
        """Synchronises and returns the result as numpy arrays (same keys as the test oracle's
        result dict). Raises VeloError on a device-side status."""
        s = self.summary.cpu().numpy().view(np.uint32)
        nt, nh, status = int(s[0]), int(s[1]), int(np.int32(s[2]))
        if status != VELO_OK:
            raise VeloError(status, f"velo_reconstruct (device status; required tracks={nt}, track_hits={nh})")
        u = lambda t: t.cpu().numpy().view(np.uint32)
        return {"event_track_offsets": u(self.event_track_offsets), "track_hit_offsets": u(self.track_hit_offsets[:nt + 1]),
                "track_hits": u(self.track_hits[:nh]), "states": self.states[:, :nt].cpu().numpy(),
                "n_tracks": nt, "n_track_hits": nh, "status": status, "n_candidates": int(s[3]), "n_deferred": int(s[4]),
                "n_big": int(s[5])}


def velo_reconstruct(geometry: Geometry, hits: Hits, params: Params, out: DeviceTracks, stream=None,
                     opts: LaunchOptions | None = None) -> None:
    """Enqueues one batch on `stream` (a torch.cuda.Stream; default: the current stream). With
    `opts` the call goes through velo_reconstruct_opts."""
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    tr = out.struct()
    rc = lib().velo_reconstruct_opts(geometry.handle, byref(hits), byref(params), byref(tr),
                                     c_void_p(out.workspace_ptr), c_size_t(out.workspace_bytes),
                                     c_void_p(st.cuda_stream), byref(opts) if opts is not None else None)
    if rc != VELO_OK:
        raise VeloError(rc, "velo_reconstruct")


velo_reconstruct_opts = velo_reconstruct


# ---- packed pixel input: the decode is fused into stage 1 ------------------------
class DevicePixelHits:
    """Packed pixel addresses of a batch resident in HBM (velo_pixel_hits_t): 4 bytes per hit."""

    def __init__(self, pixel, event_offsets, device="cuda"):
        torch = _torch()
        px = np.ascontiguousarray(pixel, dtype=np.uint32)
        self.pixel = torch.as_tensor(px.view(np.int32)).to(device)
        off = np.ascontiguousarray(event_offsets, dtype=np.uint32)
        self.event_offsets = torch.as_tensor(off.view(np.int32)).to(device)
        self.n_events = off.shape[0] - 1
        self.n_hits = int(off[-1]) - int(off[0]) if off.shape[0] else 0

    def slice_struct(self, e0: int = 0, e1: int | None = None, n_hits: int | None = None) -> PixelHits:
        e1 = self.n_events if e1 is None else e1
        return PixelHits(pixel=self.pixel.data_ptr(), event_offsets=self.event_offsets.data_ptr() + 4 * e0,
                         n_events=e1 - e0, n_hits=self.n_hits if n_hits is None else n_hits)


def velo_reconstruct_pixels(geometry: Geometry, hits: PixelHits, fmt: PixelFormat, params: Params, out: DeviceTracks,
                            stream=None, opts: LaunchOptions | None = None) -> None:
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    tr = out.struct()
    rc = lib().velo_reconstruct_pixels(geometry.handle, byref(hits), byref(fmt), byref(params), byref(tr),
                                       c_void_p(out.workspace_ptr), c_size_t(out.workspace_bytes),
                                       c_void_p(st.cuda_stream), byref(opts) if opts is not None else None)
    if rc != VELO_OK:
        raise VeloError(rc, "velo_reconstruct_pixels")


def reconstruct_pixels(pixel, event_offsets, module_z, pitch: float = 0.055, half_shift_x: float = 0.0,
                       params: Params | None = None, n_batches: int = 1, opts: LaunchOptions | None = None) -> dict:
    """Convenience for tests: as reconstruct(), from packed pixel addresses."""
    torch = _torch()
    g = Geometry(module_z, pitch=pitch, half_shift_x=half_shift_x)
    P = params if params is not None else velo_params_default(g)
    fmt = PixelFormat(pitch=pitch, half_shift_x=half_shift_x)
    dh = DevicePixelHits(pixel, event_offsets)
    off = np.ascontiguousarray(event_offsets, dtype=np.uint32).astype(np.int64)
    cuts = [dh.n_events * b // n_batches for b in range(n_batches + 1)]
    streams = [torch.cuda.Stream() for _ in range(n_batches)]
    sizes = [(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]] - off[cuts[b]])) for b in range(n_batches)]
    outs = [DeviceTracks(ne, nh, opts=opts) for ne, nh in sizes]
    torch.cuda.synchronize()
    for b in range(n_batches):
        velo_reconstruct_pixels(g, dh.slice_struct(cuts[b], cuts[b + 1], sizes[b][1]), fmt, P, outs[b], streams[b], opts)
    torch.cuda.synchronize()
    return stitch([o.to_host() for o in outs])


# ---- after the hot path: Kalman filter on the VELO segment, primary vertices ----
def velo_kalman_fit(hits: Hits, tracks: DeviceTracks, sigma_hit: float, ms_theta2: float = MS_THETA2_DEFAULT,
                    stream=None, out=None):
    """Enqueues the filter for every track of `tracks` (the outputs of velo_reconstruct for `hits`).
    Returns a device tensor whose first 13 x cap_tracks words are the state planes (`out`, if given,
    must hold at least that many)."""
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    if out is None:
        out = torch.empty((VELO_N_STATE, tracks.cap_tracks), dtype=torch.float32, device=tracks.states.device)
    assert out.numel() >= VELO_N_STATE * tracks.cap_tracks
    tr = tracks.struct()
    rc = lib().velo_kalman_fit(byref(hits), byref(tr), c_float(sigma_hit), c_float(ms_theta2), c_void_p(out.data_ptr()),
                               c_void_p(st.cuda_stream))
    if rc != VELO_OK:
        raise VeloError(rc, "velo_kalman_fit")
    return out


def velo_kalman_fit_pixels(geometry: Geometry, hits: PixelHits, fmt: PixelFormat, tracks: DeviceTracks, sigma_hit: float,
                           ms_theta2: float = MS_THETA2_DEFAULT, stream=None):
    """velo_kalman_fit for the packed-pixel path. Returns a device tensor of 13 planes x cap_tracks."""
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    out = torch.empty((VELO_N_STATE, tracks.cap_tracks), dtype=torch.float32, device=tracks.states.device)
    tr = tracks.struct()
    rc = lib().velo_kalman_fit_pixels(geometry.handle, byref(hits), byref(fmt), byref(tr), c_float(sigma_hit), c_float(ms_theta2),
                                      c_void_p(out.data_ptr()), c_void_p(st.cuda_stream))
    if rc != VELO_OK:
        raise VeloError(rc, "velo_kalman_fit_pixels")
    return out


def velo_pv_params_default() -> PvParams:
    p = PvParams()
    lib().velo_pv_params_default(byref(p))
    return p


def velo_pv_workspace_bytes(n_events: int, cap_tracks: int) -> int:
    return int(lib().velo_pv_workspace_bytes(n_events, cap_tracks))


class DevicePvs:
    """Caller-allocated output buffers of velo_pv_find (velo_pvs_t) plus its workspace."""

    def __init__(self, n_events: int, cap_tracks: int, cap_pvs: int | None = None, device="cuda",
                 with_workspace: bool = True):
        """with_workspace=False: output buffers only, for velo_pv_find_static (the library's own scratch)."""
        torch = _torch()
        self.n_events = n_events
        self.cap_pvs = int(cap_pvs if cap_pvs is not None else 32 * n_events + 1)
        i32 = dict(dtype=torch.int32, device=device)
        self.event_pv_offsets = torch.empty(n_events + 1, **i32)
        self.pvs = torch.empty((VELO_N_PV_WORDS, self.cap_pvs), dtype=torch.float32, device=device)
        self.summary = torch.zeros(4, **i32)
        if not with_workspace:
            self.workspace_bytes, self.workspace, self.workspace_ptr = 0, None, 0
            return
        self.workspace_bytes = velo_pv_workspace_bytes(n_events, cap_tracks)
        self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=device)
        self.workspace_ptr = (self.workspace.data_ptr() + 255) // 256 * 256

    def struct(self) -> Pvs:
        return Pvs(event_pv_offsets=self.event_pv_offsets.data_ptr(), pvs=self.pvs.data_ptr(), cap_pvs=self.cap_pvs,
                   summary=self.summary.data_ptr())

    def to_host(self) -> dict:
        s = self.summary.cpu().numpy().view(np.uint32)
        n, status = int(s[0]), int(np.int32(s[1]))
        if status != VELO_OK:
            raise VeloError(status, f"velo_pv_find (device status; required cap_pvs={n})")
        return {"event_pv_offsets": self.event_pv_offsets.cpu().numpy().view(np.uint32),
                "pvs": self.pvs[:, :n].cpu().numpy(), "n_pvs": n}


def velo_pv_find(tracks: DeviceTracks, out: DevicePvs, params: PvParams | None = None, stream=None) -> None:
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    P = params if params is not None else velo_pv_params_default()
    tr = tracks.struct(); pv = out.struct()
    rc = lib().velo_pv_find(byref(tr), tracks.n_events, byref(P), byref(pv), c_void_p(out.workspace_ptr),
                            c_size_t(out.workspace_bytes), c_void_p(st.cuda_stream))
    if rc != VELO_OK:
        raise VeloError(rc, "velo_pv_find")


def velo_pv_find_static(tracks: DeviceTracks, out: DevicePvs, params: PvParams | None = None, stream=None) -> None:
    """velo_pv_find over the library's fixed scratch array: the call allocates nothing (include/velo.h). At most
    VELO_PV_STATIC_MAX_EVENTS events and VELO_PV_STATIC_MAX_TRACKS of track capacity; calls that overlap on the
    GPU race on the shared array."""
    torch = _torch()
    st = stream if stream is not None else torch.cuda.current_stream()
    P = params if params is not None else velo_pv_params_default()
    tr = tracks.struct(); pv = out.struct()
    rc = lib().velo_pv_find_static(byref(tr), tracks.n_events, byref(P), byref(pv), c_void_p(st.cuda_stream))
    if rc != VELO_OK:
        raise VeloError(rc, "velo_pv_find_static")


def reconstruct(x, y, z, module, event_offsets, module_z, params: Params | None = None, n_batches: int = 1,
                cap_tracks: int | None = None, cap_track_hits: int | None = None,
                opts: LaunchOptions | None = None, **geom_kw) -> dict:
    """Convenience for tests and examples: upload host arrays, run n_batches streamed batches,
    download, and stitch the batch results into one result dict (offsets made global)."""
    torch = _torch()
    g = Geometry(module_z, **geom_kw)
    P = params if params is not None else velo_params_default(g)
    dh = DeviceHits(x, y, z, module, event_offsets)
    off = np.ascontiguousarray(event_offsets, dtype=np.uint32).astype(np.int64)
    cuts = [dh.n_events * b // n_batches for b in range(n_batches + 1)]
    streams = [torch.cuda.Stream() for _ in range(n_batches)]
    sizes = [(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]] - off[cuts[b]])) for b in range(n_batches)]
    # every buffer exists (and its zero-fill on the current stream is done) before the side streams start
    outs = [DeviceTracks(ne, nh, cap_tracks, cap_track_hits, opts=opts) for ne, nh in sizes]
    torch.cuda.synchronize()
    for b in range(n_batches):
        velo_reconstruct(g, dh.slice_struct(cuts[b], cuts[b + 1], sizes[b][1]), P, outs[b], streams[b], opts)
    torch.cuda.synchronize()
    return stitch([o.to_host() for o in outs])


def stitch(parts: list[dict]) -> dict:
    """Concatenates per-batch results (batch-local offsets) into one result."""
    eto, tho, th, st = [np.zeros(1, np.uint32)], [np.zeros(1, np.uint32)], [], []
    nt = nh = nc = nd = nbig = 0
    for p in parts:
        nd += p.get("n_deferred", 0); nbig += p.get("n_big", 0)
        eto.append(p["event_track_offsets"][1:] + np.uint32(nt))
        tho.append(p["track_hit_offsets"][1:] + np.uint32(nh))
        th.append(p["track_hits"]); st.append(p["states"])
        nt += p["n_tracks"]; nh += p["n_track_hits"]; nc += p["n_candidates"]
    return {"event_track_offsets": np.concatenate(eto), "track_hit_offsets": np.concatenate(tho),
            "track_hits": np.concatenate(th) if th else np.zeros(0, np.uint32),
            "states": np.concatenate(st, axis=1) if st else np.zeros((VELO_N_STATE, 0), np.float32),
            "n_tracks": nt, "n_track_hits": nh, "status": 0, "n_candidates": nc, "n_deferred": nd, "n_big": nbig}


# ---- end-to-end path over host buffers: the event-batch scheduler -------------------------------
class HostTracks:
    """Host output buffers of one batch (pinned when torch can pin), velo_tracks_t with HOST pointers."""

    def __init__(self, n_events: int, n_hits: int, pinned: bool = True):
        import torch
        self.cap_tracks, self.cap_track_hits = default_capacities(n_events, n_hits)
        pin = pinned and torch.cuda.is_available()
        mk = lambda n, dt: torch.empty(n, dtype=dt, pin_memory=pin)
        self.event_track_offsets = mk(n_events + 1, torch.int32)
        self.track_hit_offsets = mk(self.cap_tracks + 1, torch.int32)
        self.track_hits = mk(self.cap_track_hits, torch.int32)
        self.states = mk(VELO_N_STATE * self.cap_tracks, torch.float32).view(VELO_N_STATE, self.cap_tracks)
        self.summary = torch.zeros(VELO_N_SUMMARY, dtype=torch.int32)

    def struct(self) -> Tracks:
        return Tracks(event_track_offsets=self.event_track_offsets.data_ptr(),
                      track_hit_offsets=self.track_hit_offsets.data_ptr(), track_hits=self.track_hits.data_ptr(),
                      states=self.states.data_ptr(), cap_tracks=self.cap_tracks, cap_track_hits=self.cap_track_hits,
                      summary=self.summary.data_ptr())

    def result(self) -> dict:
        s = self.summary.numpy().view(np.uint32)
        nt, nh, status = int(s[0]), int(s[1]), int(np.int32(s[2]))
        if status != VELO_OK:
            raise VeloError(status, f"velo_scheduler_run_host (batch status; tracks={nt}, track_hits={nh})")
        u = lambda t: t.numpy().view(np.uint32)
        return {"event_track_offsets": u(self.event_track_offsets), "track_hit_offsets": u(self.track_hit_offsets)[:nt + 1],
                "track_hits": u(self.track_hits)[:nh], "states": self.states.numpy()[:, :nt], "n_tracks": nt,
                "n_track_hits": nh, "status": status, "n_candidates": int(s[3]), "n_deferred": int(s[4])}


class Scheduler:
    """velo_scheduler_t: n_streams streams with device buffers for batches of the given size."""

    def __init__(self, geometry: Geometry, n_streams: int, max_batch_events: int, max_batch_hits: int):
        _torch()
        self.geometry = geometry
        h = c_void_p()
        rc = lib().velo_scheduler_create(geometry.handle, n_streams, max_batch_events, max_batch_hits, byref(h))
        if rc != VELO_OK:
            raise VeloError(rc, "velo_scheduler_create")
        self.handle = h

    def run_host(self, params: Params, x, y, z, module, event_offsets, batch_begin, outs: list) -> None:
        """x, y, z, module, event_offsets: HOST numpy arrays or CPU torch tensors (pinned memory makes
        the copies asynchronous); outs: one HostTracks per batch. Returns when all copies are done."""
        ptr = lambda a: a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        n_events = int(event_offsets.shape[0]) - 1
        bb = np.ascontiguousarray(batch_begin, dtype=np.uint32)
        first, last = int(event_offsets[0]), int(event_offsets[n_events])
        hits = Hits(x=ptr(x), y=ptr(y), z=ptr(z), module=ptr(module), event_offsets=ptr(event_offsets),
                    n_events=n_events, n_hits=(last - first) & 0xffffffff)
        arr = (Tracks * len(outs))(*[o.struct() for o in outs])
        rc = lib().velo_scheduler_run_host(self.handle, byref(params), byref(hits), c_void_p(bb.ctypes.data),
                                           len(outs), arr)
        if rc != VELO_OK:
            raise VeloError(rc, "velo_scheduler_run_host")

    def run_host_pixels(self, params: Params, pixel, event_offsets, fmt: PixelFormat, batch_begin, outs: list) -> None:
        """As run_host, from packed pixel addresses (HOST u32 array or CPU tensor): 4 bytes per hit cross the bus."""
        ptr = lambda a: a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        n_events = int(event_offsets.shape[0]) - 1
        bb = np.ascontiguousarray(batch_begin, dtype=np.uint32)
        first, last = int(event_offsets[0]), int(event_offsets[n_events])
        hits = PixelHits(pixel=ptr(pixel), event_offsets=ptr(event_offsets), n_events=n_events,
                         n_hits=(last - first) & 0xffffffff)
        arr = (Tracks * len(outs))(*[o.struct() for o in outs])
        rc = lib().velo_scheduler_run_host_pixels(self.handle, byref(params), byref(hits), byref(fmt),
                                                  c_void_p(bb.ctypes.data), len(outs), arr)
        if rc != VELO_OK:
            raise VeloError(rc, "velo_scheduler_run_host_pixels")

    def close(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:
            _lib.velo_scheduler_free(h)

    __del__ = close
