"""GPU-vs-oracle parity of the steps after the hot path: velo_kalman_fit and
velo_pv_find through the C-ABI against oracle/velo_next_oracle.c on the same seeded inputs. Both
follow DESIGN.md §2 (K-1 ... K-5, P-1 ... P-6) operator by operator without FMA contraction, so
every word is compared bit for bit."""
import numpy as np
import pytest

import oracle
from paper_2412_05041_b200 import datagen

pytestmark = pytest.mark.gpu
M = 26
SIG = oracle.default_params().sigma_hit


@pytest.fixture(scope="module")
def velo():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2412_05041_b200 import build as vbuild
    from paper_2412_05041_b200 import velo as v
    vbuild.build()
    v.lib()
    return v


def run_gpu(velo, d, ms_theta2=None, pv_params=None, cap_pvs=None):
    """velo_reconstruct, then velo_kalman_fit and velo_pv_find on its device outputs (one stream)."""
    import torch
    g = velo.velo_geometry_load(datagen.MODULE_Z, half_shift_x=d["cfg"].half_shift_x)
    P = velo.velo_params_default(g)
    dh = velo.DeviceHits(d["x"], d["y"], d["z"], d["module"], d["event_offsets"])
    out = velo.DeviceTracks(dh.n_events, dh.n_hits)
    hs = dh.slice_struct()
    velo.velo_reconstruct(g, hs, P, out)
    ks = velo.velo_kalman_fit(hs, out, P.sigma_hit, velo.MS_THETA2_DEFAULT if ms_theta2 is None else ms_theta2)
    pv = velo.DevicePvs(dh.n_events, out.cap_tracks, cap_pvs)
    velo.velo_pv_find(out, pv, pv_params)
    torch.cuda.synchronize()
    res = out.to_host()
    return res, ks[:, :res["n_tracks"]].cpu().numpy(), pv


def same_bits(a, b):
    np.testing.assert_array_equal(np.ascontiguousarray(a, np.float32).view(np.uint32),
                                  np.ascontiguousarray(b, np.float32).view(np.uint32))


@pytest.mark.parametrize("config,n_events", [(0, 100), (1, 3000), (3, 3000), (4, 40)])
def test_kalman_and_vertices_equal_the_oracle(velo, config, n_events):
    d = datagen.generate_config(config, n_events=n_events)
    res, ks, pv = run_gpu(velo, d)
    # the oracle takes the GPU's tracks as input (they equal the oracle's own: tests/test_gpu_parity.py),
    # so that this test isolates the two new steps
    want_k = oracle.kalman_tracks(res, d["x"], d["y"], d["z"], SIG)
    same_bits(ks, want_k)
    got = pv.to_host()
    want = oracle.pv_find(res["event_track_offsets"], res["states"])
    np.testing.assert_array_equal(got["event_pv_offsets"], want["event_pv_offsets"])
    assert got["n_pvs"] == want["n_pvs"] > 0
    same_bits(got["pvs"], want["pvs"])


def test_parameter_variants_and_edge_cases(velo):
    d = datagen.generate_config(0, n_events=60)
    # zero scattering noise; other vertex parameters (coarser bins, one iteration, every seed kept)
    P = velo.velo_pv_params_default()
    P.bin_width = 1.0; P.n_bins = 600; P.n_iterations = 1; P.min_tracks = 2; P.seed_min_sum = 3; P.seed_half_window = 2
    res, ks, pv = run_gpu(velo, d, ms_theta2=0.0, pv_params=P)
    same_bits(ks, oracle.kalman_tracks(res, d["x"], d["y"], d["z"], SIG, 0.0))
    Po = oracle.PvParams(z_min=P.z_min, bin_width=P.bin_width, n_bins=P.n_bins, seed_min_sum=P.seed_min_sum,
                         seed_half_window=P.seed_half_window, chi2_max=P.chi2_max, n_iterations=P.n_iterations,
                         min_tracks=P.min_tracks, max_pv_per_event=P.max_pv_per_event)
    got, want = pv.to_host(), oracle.pv_find(res["event_track_offsets"], res["states"], Po)
    np.testing.assert_array_equal(got["event_pv_offsets"], want["event_pv_offsets"])
    same_bits(got["pvs"], want["pvs"])
    # an odd number of bins that is no multiple of 32 (the last packed word holds one bin, the last block of the
    # seed scan is ragged), fine bins, a seed window wider than a block's halo
    for nb, bw, hw in ((2399, 0.25, 6), (4095, 0.15, 9), (33, 20.0, 1)):
        P3 = velo.velo_pv_params_default()
        P3.n_bins = nb; P3.bin_width = bw; P3.seed_half_window = hw; P3.seed_min_sum = 1
        _, _, pv3 = run_gpu(velo, d, pv_params=P3)
        Po3 = oracle.default_pv_params()
        Po3.n_bins = nb; Po3.bin_width = bw; Po3.seed_half_window = hw; Po3.seed_min_sum = 1
        got3, want3 = pv3.to_host(), oracle.pv_find(res["event_track_offsets"], res["states"], Po3)
        np.testing.assert_array_equal(got3["event_pv_offsets"], want3["event_pv_offsets"])
        same_bits(got3["pvs"], want3["pvs"])
        assert got3["n_pvs"] > 0
    # at most two vertices per event, lowest z first
    P2 = velo.velo_pv_params_default(); P2.max_pv_per_event = 2
    _, _, pv2 = run_gpu(velo, d, pv_params=P2)
    Po2 = oracle.default_pv_params(); Po2.max_pv_per_event = 2
    got2, want2 = pv2.to_host(), oracle.pv_find(res["event_track_offsets"], res["states"], Po2)
    np.testing.assert_array_equal(got2["event_pv_offsets"], want2["event_pv_offsets"])
    same_bits(got2["pvs"], want2["pvs"])
    assert np.all(np.diff(got2["event_pv_offsets"].astype(np.int64)) <= 2)
    # capacity overflow is reported with the required size, nothing is truncated silently
    _, _, pv3 = run_gpu(velo, d, cap_pvs=3)
    with pytest.raises(velo.VeloError) as ei:
        pv3.to_host()
    n_required = oracle.pv_find(res["event_track_offsets"], res["states"])["n_pvs"]
    assert ei.value.code == velo.VELO_ERR_CAPACITY and str(n_required) in str(ei.value)


def test_empty_batches(velo):
    import torch
    # events without hits: no tracks, no vertices, offsets all zero
    z = np.zeros(0, np.float32)
    d = {"x": z, "y": z, "z": z, "module": np.zeros(0, np.uint8), "event_offsets": np.zeros(6, np.uint32),
         "cfg": datagen.GenConfig()}
    res, ks, pv = run_gpu(velo, d)
    got = pv.to_host()
    assert res["n_tracks"] == 0 and ks.shape[1] == 0 and got["n_pvs"] == 0
    np.testing.assert_array_equal(got["event_pv_offsets"], np.zeros(6, np.uint32))
    torch.cuda.synchronize()


def test_vertices_match_the_generator(velo):
    """End to end on the GPU: >= 90 % of the generated vertices with >= 10 tracks are found within 0.5 mm."""
    ne = 300
    d = datagen.generate_config(1, n_events=ne, truth=True)
    res, _, pv = run_gpu(velo, d)
    got = pv.to_host()
    found = total = 0
    for e in range(ne):
        tr = d["trk_truth"][d["trk_offsets"][e]:d["trk_offsets"][e + 1]]
        zt, cnt = np.unique(tr[:, 2], return_counts=True)
        zp = got["pvs"][2, got["event_pv_offsets"][e]:got["event_pv_offsets"][e + 1]]
        for z0 in zt[cnt >= 10]:
            total += 1
            found += bool(len(zp) and np.min(np.abs(zp - z0)) < 0.5)
    assert found / total >= 0.90
