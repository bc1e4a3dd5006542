"""Seeded synthetic VELO event generator (inputs only; none of the method's arithmetic).

Recipe: BASELINE.json:configs[0..4] as restated in SURVEY.md §8(d) and DESIGN.md §4. These
inputs stand in for the LHCb collision data of the paper, which are not
available. Both the CPU oracle (tests only) and the CUDA path consume the arrays written here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, replace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "velo_gen.cpp")
_LIB = os.path.join(_HERE, "libvelogen.so")

# 26 modules from -289 to +751 mm (BASELINE.json:configs[0]); 25 mm pitch
# around the luminous region, sparse ends. Any table works: it is loaded through
# velo_geometry_load.
MODULE_Z = np.array(
    [-289, -264, -239, -214, -144, -74, -49, -24, 1, 26, 51, 76, 101, 126, 151, 176, 201, 226,
     251, 313, 390, 485, 604, 649, 694, 751], dtype=np.float64)
R_IN, R_OUT, PITCH = 5.1, 42.0, 0.055
OPEN_HALF_SHIFT = 24.5  # PAPER.md:24 §2: 49 mm opening in 2023


class _CConfig(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64), ("n_modules", ctypes.c_uint32), ("ion_mode", ctypes.c_int32),
        ("r_in", ctypes.c_double), ("r_out", ctypes.c_double), ("pitch", ctypes.c_double),
        ("half_shift_x", ctypes.c_double),
        ("mu", ctypes.c_double), ("trk_mean", ctypes.c_double), ("mult_lo", ctypes.c_double),
        ("mult_hi", ctypes.c_double),
        ("eta_lo", ctypes.c_double), ("eta_hi", ctypes.c_double),
        ("sigma_vxy", ctypes.c_double), ("sigma_vz", ctypes.c_double),
        ("hit_eff", ctypes.c_double), ("noise_frac", ctypes.c_double), ("ms_sigma", ctypes.c_double),
        ("quantise", ctypes.c_int32), ("shuffle", ctypes.c_int32),
        ("backward_frac", ctypes.c_double), ("stagger_z", ctypes.c_double), ("overlap_x", ctypes.c_double),
    ]


@dataclass(frozen=True)
class GenConfig:
    """One workload recipe. Defaults = BASELINE.json:configs[0..2] (pp, mu=5, closed VELO)."""
    seed: int = 1
    ion_mode: bool = False
    half_shift_x: float = 0.0
    mu: float = 5.0              # PAPER.md:18 §1
    trk_mean: float = 40.0
    mult_lo: float = 50.0
    mult_hi: float = 5000.0
    eta_lo: float = 2.0          # PAPER.md:22 §2
    eta_hi: float = 5.0
    sigma_vxy: float = 0.015
    sigma_vz: float = 45.0
    hit_eff: float = 0.98
    noise_frac: float = 0.005
    ms_sigma: float = 0.3e-3
    quantise: bool = True
    shuffle: bool = True
    backward_frac: float = 0.0   # tracks towards -z (none in BASELINE's configs)
    stagger_z: float = 0.0       # §8(f) f4, 52-sensor layout: the two sensors of a station at z -+ stagger_z/2 ...
    overlap_x: float = 0.0       # ... both reaching this far over x = 0 (0, 0 in BASELINE's configs)
    r_in: float = R_IN
    r_out: float = R_OUT
    pitch: float = PITCH
    module_z: tuple = tuple(MODULE_Z.tolist())


# (recipe, n_events, n_batches) for BASELINE.json:configs[i]
CONFIGS = {
    0: (GenConfig(), 100, 1),
    1: (GenConfig(), 10_000, 1),
    2: (GenConfig(), 100_000, 4),
    3: (GenConfig(half_shift_x=OPEN_HALF_SHIFT), 100_000, 4),
    4: (GenConfig(ion_mode=True, noise_frac=0.01), 2_000, 1),
}


def build(force: bool = False) -> str:
    """Compile the generator with g++ (host only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = f"{_LIB}.{os.getpid()}.tmp"      # atomic: several ranks or test workers may build at once
        cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-pthread", "-o", tmp, _SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        u32p = ctypes.POINTER(ctypes.c_uint32)
        lib.velogen_count.argtypes = [ctypes.POINTER(_CConfig), ctypes.c_void_p, ctypes.c_uint64,
                                      ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.velogen_count.restype = ctypes.c_int
        lib.velogen_fill.argtypes = [ctypes.POINTER(_CConfig), ctypes.c_void_p, ctypes.c_uint64,
                                     ctypes.c_uint32] + [ctypes.c_void_p] * 8 + [ctypes.c_int]
        lib.velogen_fill.restype = ctypes.c_int
        lib.velogen_pixels.argtypes = [ctypes.POINTER(_CConfig), ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32,
                                       ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
        lib.velogen_pixels.restype = ctypes.c_int
        del u32p
        _lib = lib
    return _lib


def _cconfig(cfg: GenConfig) -> _CConfig:
    return _CConfig(
        seed=cfg.seed, n_modules=len(cfg.module_z), ion_mode=int(cfg.ion_mode),
        r_in=cfg.r_in, r_out=cfg.r_out, pitch=cfg.pitch, half_shift_x=cfg.half_shift_x,
        mu=cfg.mu, trk_mean=cfg.trk_mean, mult_lo=cfg.mult_lo, mult_hi=cfg.mult_hi,
        eta_lo=cfg.eta_lo, eta_hi=cfg.eta_hi, sigma_vxy=cfg.sigma_vxy, sigma_vz=cfg.sigma_vz,
        hit_eff=cfg.hit_eff, noise_frac=cfg.noise_frac, ms_sigma=cfg.ms_sigma,
        quantise=int(cfg.quantise), shuffle=int(cfg.shuffle), backward_frac=cfg.backward_frac,
        stagger_z=cfg.stagger_z, overlap_x=cfg.overlap_x)


def _ptr(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else None


def generate(cfg: GenConfig, e0: int, n_events: int, truth: bool = False, nthreads: int | None = None,
             alloc=None, pixels: bool = False) -> dict:
    """Generate events [e0, e0+n_events). Returns numpy arrays:
    x, y, z (f32[n_hits]), module (u8[n_hits]), event_offsets (u32[n_events+1]); with truth=True
    also hit_track (i32[n_hits], -1 = noise), trk_offsets (u32[n_events+1]), trk_truth
    (f64[n_trk, 5] = xv, yv, zv, tx, ty); with pixels=True (quantised recipes only) also pixel
    (u32[n_hits], the packed pixel address of every hit: include/velo.h velo_pixel_hits_t).
    `alloc(shape, dtype)` may supply the hit buffers (e.g. views of pinned host memory)."""
    lib = _load()
    if nthreads is None:
        nthreads = os.cpu_count() or 1
    cc = _cconfig(cfg)
    mz = np.ascontiguousarray(np.asarray(cfg.module_z, dtype=np.float64))
    nh = np.zeros(n_events, dtype=np.uint32)
    nt = np.zeros(n_events, dtype=np.uint32)
    rc = lib.velogen_count(ctypes.byref(cc), _ptr(mz), e0, n_events, _ptr(nh), _ptr(nt), nthreads)
    if rc != 0:
        raise RuntimeError(f"velogen_count failed: {rc}")
    tot_h = int(nh.sum(dtype=np.uint64))
    tot_t = int(nt.sum(dtype=np.uint64))
    if tot_h >= 2**32 or tot_t >= 2**31:
        raise ValueError("batch too large for u32 offsets")
    hoff = np.zeros(n_events + 1, dtype=np.uint32)
    toff = np.zeros(n_events + 1, dtype=np.uint32)
    np.cumsum(nh, out=hoff[1:])
    np.cumsum(nt, out=toff[1:])
    mk = alloc if alloc is not None else (lambda shape, dtype: np.empty(shape, dtype=dtype))
    x = mk(tot_h, np.float32)
    y = mk(tot_h, np.float32)
    z = mk(tot_h, np.float32)
    mod = mk(tot_h, np.uint8)
    ht = np.empty(tot_h, dtype=np.int32) if truth else None
    tt = np.empty((tot_t, 5), dtype=np.float64) if truth else None
    rc = lib.velogen_fill(ctypes.byref(cc), _ptr(mz), e0, n_events, _ptr(hoff), _ptr(toff),
                          _ptr(x), _ptr(y), _ptr(z), _ptr(mod), _ptr(ht), _ptr(tt), nthreads)
    if rc != 0:
        raise RuntimeError(f"velogen_fill failed: {rc}")
    out = {"x": x, "y": y, "z": z, "module": mod, "event_offsets": hoff, "n_events": n_events,
           "n_hits": tot_h, "module_z": mz.astype(np.float32), "cfg": cfg}
    if truth:
        out.update(hit_track=ht, trk_offsets=toff, trk_truth=tt)
    if pixels:
        px = mk(tot_h, np.uint32)
        rc = lib.velogen_pixels(ctypes.byref(cc), _ptr(mz), e0, n_events, _ptr(hoff), _ptr(px), nthreads)
        if rc != 0:
            raise RuntimeError(f"velogen_pixels failed: {rc} (-3: the recipe is not quantised to pixels)")
        out["pixel"] = px
    return out


def generate_config(i: int, n_events: int | None = None, e0: int = 0, **kw) -> dict:
    cfg, n, _ = CONFIGS[i]
    return generate(cfg, e0, n if n_events is None else n_events, **kw)


def sensor_planes(cfg: GenConfig) -> tuple[np.ndarray, np.ndarray]:
    """z of the two sensor planes of every station in the 52-sensor layout (stagger_z): the -x sensor's and
    the +x sensor's, as the fp32 values the generated hits carry (include/velo.h: module_z, module_z_b)."""
    z = np.asarray(cfg.module_z, dtype=np.float64)
    return (z - 0.5 * cfg.stagger_z).astype(np.float32), (z + 0.5 * cfg.stagger_z).astype(np.float32)


def ideal_config(**kw) -> GenConfig:
    """Noise-free, 100 % efficient, unquantised, unscattered straight tracks (SURVEY.md §8(c)
    whole-path pin (ii))."""
    return replace(GenConfig(), hit_eff=1.0, noise_frac=0.0, ms_sigma=0.0, quantise=False, **kw)
