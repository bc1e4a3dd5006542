"""The seeded generator (inputs only): determinism, prefix property (A21), shapes of the
BASELINE.json workloads. CPU only."""
import numpy as np

from paper_2412_05041_b200 import datagen


def test_event_stream_independent_of_batch_and_threads():
    a = datagen.generate_config(1, n_events=150, nthreads=1)
    b = datagen.generate_config(1, n_events=400, nthreads=5)
    n = a["n_hits"]
    for k in ("x", "y", "z", "module"):
        assert (a[k] == b[k][:n]).all()
    c = datagen.generate_config(1, n_events=50, e0=100)
    o = int(b["event_offsets"][100])
    assert (c["x"] == b["x"][o:o + c["n_hits"]]).all()


def test_config_shapes(cfg0):
    d = cfg0
    nh = np.diff(d["event_offsets"].astype(np.int64))
    assert 1700 < nh.mean() < 2200                      # SURVEY.md §8 probe: 1924 hits/event at mu=5
    assert d["module"].max() <= 25 and (d["z"] == datagen.MODULE_Z.astype(np.float32)[d["module"]]).all()
    r = np.hypot(d["x"], d["y"])
    assert r.min() > 5.0 and r.max() < 42.1
    # hits sit on pixel centres: (k + 0.5) * 0.055
    k = d["y"].astype(np.float64) / 0.055 - 0.5
    assert np.abs(k - np.round(k)).max() < 1e-3
    d3 = datagen.generate_config(3, n_events=300)
    assert 250 < np.diff(d3["event_offsets"].astype(np.int64)).mean() < 400   # probe: 316
    assert np.abs(d3["x"]).min() > 24.5                 # halves displaced by +-24.5 mm
    d4 = datagen.generate_config(4, n_events=60)
    nh4 = np.diff(d4["event_offsets"].astype(np.int64))
    assert nh4.max() > 15000 and nh4.min() > 100


def test_truth_tables(cfg0):
    d = cfg0
    assert d["hit_track"].shape[0] == d["n_hits"] and d["trk_truth"].shape[1] == 5
    frac_noise = (d["hit_track"] < 0).mean()
    assert 0.002 < frac_noise < 0.01
    eta = -np.log(np.tan(0.5 * np.arctan(np.hypot(d["trk_truth"][:, 3], d["trk_truth"][:, 4]))))
    assert eta.min() >= 2.0 - 1e-9 and eta.max() <= 5.0 + 1e-9
