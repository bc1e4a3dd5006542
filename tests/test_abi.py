"""The C-ABI boundary without a GPU: libvelo.so builds for sm_100a, loads, exports every symbol
include/velo.h declares, and its host-only entry points behave as documented. No compute call."""
import ctypes
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2412_05041_b200 import build as vbuild
from paper_2412_05041_b200 import datagen, velo

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    vbuild.build()
    return velo.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "velo.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(velo_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(lib):
    names = _declared_functions()
    assert set(names) == set(velo.EXPORTS)
    for n in names:
        assert hasattr(lib, n), n


def test_header_compiles_as_plain_c(tmp_path):
    c = tmp_path / "t.c"
    c.write_text('#include "velo.h"\nint main(void){velo_params_t p; (void)p; return VELO_OK;}\n')
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(c),
                    "-o", str(tmp_path / "t.o")], check=True)


def test_library_is_sm100a_only(lib):
    out = subprocess.run(["cuobjdump", "-lelf", vbuild.LIB], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_geometry_and_params(lib):
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    assert g.n_modules == 26
    p = velo.velo_params_default(g)
    assert (p.phi_window_seed, p.phi_window_fwd, p.max_skipped, p.clone_num, p.clone_den) == (300, 300, 1, 1, 3)
    assert np.float32(p.sigma_hit) == np.float32(float.fromhex("0x1.042186p-6"))
    assert np.float32(p.max_scatter_seed) == np.float32(0.1) and np.float32(p.max_scatter_weak) == np.float32(0.05)
    assert np.float32(p.max_chi2_ndof) == np.float32(100.0)
    # the oracle's defaults are written independently; they must describe the same reading
    import oracle
    q = oracle.default_params()
    for name, _ in velo.Params._fields_:
        assert getattr(p, name) == getattr(q, name), name
    with pytest.raises(velo.VeloError) as e:
        velo.velo_geometry_load([0.0, 1.0])                            # fewer than 3 modules
    assert e.value.code == velo.VELO_ERR_GEOMETRY
    with pytest.raises(velo.VeloError):
        velo.velo_geometry_load([0.0, 2.0, 1.0])                       # not increasing
    with pytest.raises(velo.VeloError):
        velo.velo_geometry_load(np.arange(33, dtype=np.float32))       # more than VELO_MAX_MODULES


def test_workspace_bytes_and_argument_checks(lib):
    w0 = velo.velo_workspace_bytes(100, 200_000, 50_100, 400_001)
    w1 = velo.velo_workspace_bytes(25_000, 48_000_000, 12_025_001, 96_000_001)
    assert 0 < w0 < w1 < 8 << 30
    assert w0 % 256 == 0
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    p = velo.velo_params_default(g)
    # null structs are rejected before anything touches CUDA
    rc = lib.velo_reconstruct(g.handle, None, ctypes.byref(p), None, None, 0, None)
    assert rc == velo.VELO_ERR_ARG
    assert velo.velo_version().startswith("velo-b200")


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2412_05041_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "velo_oracle" not in text, f


def test_entry_points_around_the_path_check_their_arguments(lib):
    """velo_pv_params_default holds the readings P-1 ... P-6 (and equals the oracle's own defaults, which
    are written independently); null or inconsistent arguments come back as VELO_ERR_ARG before any CUDA
    call (so this runs without a GPU)."""
    import oracle
    p = velo.velo_pv_params_default()
    q = oracle.default_pv_params()
    for name, _ in velo.PvParams._fields_:
        assert getattr(p, name) == getattr(q, name), name
    assert (p.n_bins, p.seed_min_sum, p.seed_half_window, p.n_iterations, p.min_tracks, p.max_pv_per_event) == (2400, 5, 6, 4, 4, 32)
    assert velo.velo_pv_workspace_bytes(1000, 50000) > 1000 * 32 * 5 * 4
    assert np.float32(velo.MS_THETA2_DEFAULT) == np.float32(oracle.MS_THETA2_DEFAULT)
    L = lib
    assert L.velo_kalman_fit(None, None, 0.016, 9e-8, None, None) == velo.VELO_ERR_ARG
    assert L.velo_pv_find(None, 0, None, None, None, 0, None) == velo.VELO_ERR_ARG
    assert L.velo_reconstruct_pixels(None, None, None, None, None, None, 0, None, None) == velo.VELO_ERR_ARG
    assert L.velo_scheduler_run_host_pixels(None, None, None, None, None, 0, None) == velo.VELO_ERR_ARG
    # a histogram larger than the kernel's shared memory is refused
    tr = velo.Tracks(event_track_offsets=8, track_hit_offsets=8, track_hits=8, states=8, cap_tracks=4, cap_track_hits=4, summary=8)
    pv = velo.Pvs(event_pv_offsets=8, pvs=8, cap_pvs=4, summary=8)
    bad = velo.velo_pv_params_default(); bad.n_bins = 5000
    assert L.velo_pv_find(ctypes.byref(tr), 1, ctypes.byref(bad), ctypes.byref(pv), ctypes.c_void_p(256), 1 << 20, None) == velo.VELO_ERR_ARG
