"""velo_pv_find_static (include/velo.h): the vertex finder over the library's own fixed scratch array, for
callers that cannot allocate device memory. Its output must equal velo_pv_find's (the existing path with a
caller-allocated workspace) bit for bit, on two calls in a row that share the array: the second call runs on
another, smaller batch, so that anything it wrongly kept from the first one would show.

This file is named so that pytest collects it last (the suite runs with pytest -x)."""
import ctypes

import numpy as np
import pytest

from paper_2412_05041_b200 import datagen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def velo():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2412_05041_b200 import build as vbuild
    from paper_2412_05041_b200 import velo as v
    vbuild.build()
    v.lib()
    return v


def reconstructed(velo, config, n_events, e0=0):
    """Device outputs of velo_reconstruct for a seeded batch."""
    d = datagen.generate_config(config, n_events=n_events, e0=e0)
    g = velo.velo_geometry_load(datagen.MODULE_Z, half_shift_x=d["cfg"].half_shift_x)
    dh = velo.DeviceHits(d["x"], d["y"], d["z"], d["module"], d["event_offsets"])
    out = velo.DeviceTracks(dh.n_events, dh.n_hits)
    velo.velo_reconstruct(g, dh.slice_struct(), velo.velo_params_default(g), out)
    return out, (g, dh)        # keep the inputs alive until the caller has synchronised


def same_vertices(a: dict, b: dict):
    assert a["n_pvs"] == b["n_pvs"] > 0
    np.testing.assert_array_equal(a["event_pv_offsets"], b["event_pv_offsets"])
    np.testing.assert_array_equal(a["pvs"].view(np.uint32), b["pvs"].view(np.uint32))     # bit for bit


def test_two_calls_in_a_row_equal_the_existing_path(velo):
    import torch
    big, keep1 = reconstructed(velo, 1, 2500)            # mu = 5, closed VELO
    small, keep2 = reconstructed(velo, 3, 900, e0=50)    # open VELO: fewer events, fewer tracks per event
    assert big.cap_tracks <= velo.VELO_PV_STATIC_MAX_TRACKS
    want = []
    for tr in (big, small):                              # the existing path, a workspace per call
        pv = velo.DevicePvs(tr.n_events, tr.cap_tracks)
        velo.velo_pv_find(tr, pv)
        want.append(pv.to_host())
    outs = [velo.DevicePvs(tr.n_events, tr.cap_tracks, with_workspace=False) for tr in (big, small)]
    velo.velo_pv_find_static(big, outs[0])               # warm: the array's address is looked up here
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # two calls in a row on one stream (calls that overlap on the GPU would race on the shared array)
    velo.velo_pv_find_static(big, outs[0])
    velo.velo_pv_find_static(small, outs[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0         # no device memory was taken by the calls
    same_vertices(outs[0].to_host(), want[0])
    same_vertices(outs[1].to_host(), want[1])
    # and once more in the other order, with other parameters for one of them
    P = velo.velo_pv_params_default()
    P.bin_width = 1.0; P.n_bins = 600; P.n_iterations = 2; P.min_tracks = 2
    pv = velo.DevicePvs(big.n_events, big.cap_tracks)
    velo.velo_pv_find(big, pv, P)
    velo.velo_pv_find_static(small, outs[1])
    velo.velo_pv_find_static(big, outs[0], P)
    torch.cuda.synchronize()
    same_vertices(outs[1].to_host(), want[1])
    same_vertices(outs[0].to_host(), pv.to_host())
    del keep1, keep2


def test_sizes_beyond_the_fixed_maximum_are_refused(velo):
    import torch
    tr, keep = reconstructed(velo, 3, 64)
    out = velo.DevicePvs(tr.n_events, tr.cap_tracks, with_workspace=False)
    L, P = velo.lib(), velo.velo_pv_params_default()
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    call = lambda t, ne: L.velo_pv_find_static(ctypes.byref(t), ne, ctypes.byref(P), ctypes.byref(out.struct()), st)
    t = tr.struct()
    assert call(t, tr.n_events) == velo.VELO_OK
    assert call(t, velo.VELO_PV_STATIC_MAX_EVENTS + 1) == velo.VELO_ERR_STATIC_LIMIT
    t.cap_tracks = velo.VELO_PV_STATIC_MAX_TRACKS + 1
    assert call(t, tr.n_events) == velo.VELO_ERR_STATIC_LIMIT
    assert L.velo_pv_find_static(None, 0, None, None, None) == velo.VELO_ERR_ARG
    torch.cuda.synchronize()
    with pytest.raises(velo.VeloError) as ei:
        big = velo.DeviceTracks(velo.VELO_PV_STATIC_MAX_EVENTS + 1, 1000)
        velo.velo_pv_find_static(big, velo.DevicePvs(big.n_events, big.cap_tracks, with_workspace=False))
    assert ei.value.code == velo.VELO_ERR_STATIC_LIMIT and "VELO_ERR_STATIC_LIMIT" in str(ei.value)
    del keep
