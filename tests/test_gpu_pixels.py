"""GPU parity of the packed-pixel path: velo_reconstruct_pixels decodes F-1/F-2
addresses inside stage 1. Its tracks must equal, bit for bit, (a) the oracle run on the oracle's own
decode of the same words and (b) the fp32-SoA path on the generator's coordinates."""
import numpy as np
import pytest

import oracle
from paper_2412_05041_b200 import datagen
from tests import velo_testlib as T

pytestmark = pytest.mark.gpu
M = 26


@pytest.fixture(scope="module")
def velo():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2412_05041_b200 import build as vbuild
    from paper_2412_05041_b200 import velo as v
    vbuild.build()
    v.lib()
    return v


def same(got, want):
    info = T.assert_same_result(got, want)
    assert info["bit_identical_states"]
    np.testing.assert_array_equal(got["track_hits"], want["track_hits"])
    assert got["n_tracks"] == want["n_tracks"] > 0


@pytest.mark.parametrize("config,n_events,kw", [
    (0, 100, {}), (1, 4000, {"n_batches": 3}), (3, 4000, {}), (4, 60, {}),           # ion-like: large events are deferred
    (0, 100, {"opts": {"path": 1}}), (0, 100, {"opts": {"pool_units": 24}}),          # slab only; tiny pool: deferrals
])
def test_pixels_equal_oracle_and_fp32_path(velo, config, n_events, kw):
    d = datagen.generate_config(config, n_events=n_events, pixels=True)
    shift = d["cfg"].half_shift_x
    kw = dict(kw)
    opts = velo.LaunchOptions(**kw.pop("opts")) if "opts" in kw else None
    got = velo.reconstruct_pixels(d["pixel"], d["event_offsets"], datagen.MODULE_Z, half_shift_x=shift, opts=opts, **kw)
    dec = oracle.pixel_decode(d["pixel"], datagen.MODULE_Z, half_shift_x=shift)
    dd = dict(d); dd.update(dec)
    want = T.oracle_parallel(dd, M, None, None)
    same(got, want)
    soa = velo.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], datagen.MODULE_Z, half_shift_x=shift)
    same(got, soa)
    if config == 4:
        assert got["n_deferred"] + got["n_big"] > 0


def test_bad_module_id_is_reported(velo):
    d = datagen.generate_config(0, n_events=10, pixels=True)
    px = d["pixel"].copy(); px[5] = (px[5] & ((1 << 23) - 1)) | (30 << 23)
    with pytest.raises(velo.VeloError) as ei:
        velo.reconstruct_pixels(px, d["event_offsets"], datagen.MODULE_Z)
    assert ei.value.code == velo.VELO_ERR_INPUT


def test_scheduler_with_packed_host_buffers(velo):
    import torch
    d = datagen.generate_config(0, n_events=100, pixels=True)
    off = d["event_offsets"]
    cuts = [0, 37, 37, 80, 100]                                   # ragged, one empty batch
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    P = velo.velo_params_default(g)
    nb = len(cuts) - 1
    sched = velo.Scheduler(g, 2, 50, int(max(off[cuts[b + 1]] - off[cuts[b]] for b in range(nb))))
    houts = [velo.HostTracks(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]])) for b in range(nb)]
    px = torch.from_numpy(d["pixel"].view(np.int32).copy()).pin_memory()
    sched.run_host_pixels(P, px, off, velo.PixelFormat(pitch=0.055, half_shift_x=0.0), cuts, houts)
    got = velo.stitch([h.result() for h in houts])
    want = T.oracle_parallel(d, M, None, None)
    same(got, want)
    sched.close()


def test_kalman_filter_on_the_packed_path(velo):
    """velo_reconstruct_pixels -> velo_kalman_fit_pixels: the states equal the oracle's filter on the oracle's decode."""
    import torch
    d = datagen.generate_config(3, n_events=1500, pixels=True)
    shift = d["cfg"].half_shift_x
    g = velo.velo_geometry_load(datagen.MODULE_Z, half_shift_x=shift)
    P = velo.velo_params_default(g)
    fmt = velo.PixelFormat(pitch=0.055, half_shift_x=shift)
    dh = velo.DevicePixelHits(d["pixel"], d["event_offsets"])
    out = velo.DeviceTracks(dh.n_events, dh.n_hits)
    hs = dh.slice_struct()
    velo.velo_reconstruct_pixels(g, hs, fmt, P, out)
    ks = velo.velo_kalman_fit_pixels(g, hs, fmt, out, P.sigma_hit)
    torch.cuda.synchronize()
    res = out.to_host()
    dec = oracle.pixel_decode(d["pixel"], datagen.MODULE_Z, half_shift_x=shift)
    want = oracle.kalman_tracks(res, dec["x"], dec["y"], dec["z"], P.sigma_hit)
    np.testing.assert_array_equal(ks[:, :res["n_tracks"]].cpu().numpy().view(np.uint32), want.view(np.uint32))
    assert res["n_tracks"] > 50000
