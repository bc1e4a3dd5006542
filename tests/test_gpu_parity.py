"""GPU-vs-oracle parity (BASELINE.json:north_star): the CUDA path,
called through the C-ABI, against the CPU oracle on the same seeded inputs. Hit lists, offsets and
n_hits bit-exact after canonical ordering; states within 1e-5 relative (in fact bit-identical,
because the kernels follow O-11 operator by operator without FMA contraction)."""
import numpy as np
import pytest

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
    v.lib()  # fails loudly if the extension is missing
    return v


def gpu(velo, d, **kw):
    return velo.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], datagen.MODULE_Z, **kw)


def cpu(d, params=None, workers=None):
    return T.oracle_parallel(d, M, params, workers)


def check(got, want):
    info = T.assert_same_result(got, want)
    assert got["n_tracks"] == want["n_tracks"] and got["n_track_hits"] == want["n_track_hits"]
    return info


# ---- BASELINE.json:configs[0]: everything, element by element -----------------------------------
def test_config0_full(velo):
    d = datagen.generate_config(0)
    got, want = gpu(velo, d), cpu(d)
    info = check(got, want)
    assert info["bit_identical_states"]
    assert got["n_candidates"] == want["n_candidates"]
    assert got["n_deferred"] == 0            # every event ran in the pipeline kernels
    assert want["n_tracks"] > 15000          # 100 events x ~190 tracks: the comparison is not vacuous


def test_config0_emits_oracle_order(velo):
    """Tracks come out in creation order (include/velo.h), which is also the oracle's order."""
    d = datagen.generate_config(0, n_events=20)
    got, want = gpu(velo, d), cpu(d, workers=1)
    np.testing.assert_array_equal(got["track_hit_offsets"], want["track_hit_offsets"])
    np.testing.assert_array_equal(got["track_hits"], want["track_hits"])
    np.testing.assert_array_equal(got["states"].view(np.uint32), want["states"].view(np.uint32))


def test_streamed_batches_equal_single_batch(velo):
    d = datagen.generate_config(1, n_events=403)     # ragged: 403 events in 4 batches
    a, b = gpu(velo, d), gpu(velo, d, n_batches=4)
    for k in ("event_track_offsets", "track_hit_offsets", "track_hits"):
        np.testing.assert_array_equal(a[k], b[k])
    np.testing.assert_array_equal(a["states"].view(np.uint32), b["states"].view(np.uint32))
    check(b, cpu(d))


def test_run_to_run_determinism(velo):
    d = datagen.generate_config(0, n_events=60)
    ref = gpu(velo, d)
    for _ in range(5):
        r = gpu(velo, d)
        for k in ("event_track_offsets", "track_hit_offsets", "track_hits"):
            np.testing.assert_array_equal(ref[k], r[k])
        np.testing.assert_array_equal(ref["states"].view(np.uint32), r["states"].view(np.uint32))


# ---- the event kernels: the three-stage pipeline (default) in several launch geometries, the general
# slab kernel on its own ------------------------------------------------------------------------------
@pytest.mark.parametrize("kw", [
    {"path": 1},                                                  # general slab kernel only
    {"track_group": 32, "track_teams": 8}, {"track_group": 32, "track_teams": 24},
    {"track_group": 64}, {"track_group": 64, "track_teams": 15}, {"track_group": 128},
    {"fit_teams": 4}, {"fit_teams": 12}, {"fit_teams": 254}, {"sort_teams": 4}, {"sort_teams": 7}, {"sort_teams": 252},
    {"pool_units": 48}, {"pool_units": 24, "track_group": 64}], ids=str)
def test_pipeline_geometries_and_other_paths_agree(velo, kw):
    d = datagen.generate_config(0)
    want = cpu(d)
    got = gpu(velo, d, opts=velo.LaunchOptions(**kw))
    info = check(got, want)
    assert info["bit_identical_states"], kw
    np.testing.assert_array_equal(got["track_hits"], want["track_hits"])    # emitted in the oracle's order
    if kw.get("path", 0) == 0 and "pool_units" not in kw:
        assert got["n_deferred"] == 0, kw


def test_hand_made_pin_events(velo):
    """The events of tests/test_oracle_hand_events.py (stated outcomes: forwarding tie, window centre,
    miss reset, flagged hits in seeding, same-step flags, chi2 cut, clone pairs) through the CUDA path."""
    import oracle
    built = [f() for f in T.PIN_EVENTS]
    events = [b[0] for b in built]
    x, y, z, m, off = T.batch_of(events)
    for kw in ({}, {"track_group": 64}, {"path": velo.VELO_PATH_SLAB_ONLY}):
        got = velo.reconstruct(x, y, z, m, off, datagen.MODULE_Z, opts=velo.LaunchOptions(**kw))
        for e, b in enumerate(built):
            o0 = int(off[e])
            assert sorted(tuple(h - o0 for h in hits) for hits, _ in T.split_tracks(got, e)) == b[1], (e, kw)
        check(got, oracle.reconstruct(x, y, z, m, off, M))
    # the chi2 cut on both sides of the threshold (O-12)
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    for n in (3, 5):
        ev, want, chi2 = T.pin_chi2_track(n)
        xe, ye, ze, me, offe = T.batch_of([ev])
        for factor, expect in ((1.04, want), (0.96, [])):
            p = velo.velo_params_default(g)
            p.max_chi2_ndof = float(np.float32(chi2 / (2 * n - 4) * factor))
            got = velo.reconstruct(xe, ye, ze, me, offe, datagen.MODULE_Z, params=p)
            assert sorted(hits for hits, _ in T.split_tracks(got, 0)) == expect


def test_hits_off_their_module_plane_are_deferred_to_the_general_kernel(velo):
    """The pipeline requires z == module_z[module]; events that break it take the slab kernel
    inside the same call, and the batch result is still the oracle's."""
    d = datagen.generate_config(0, n_events=40)
    z = d["z"].copy()
    off = d["event_offsets"].astype(np.int64)
    rng = np.random.default_rng(3)
    for e in (0, 3, 4, 17, 39):
        idx = rng.integers(off[e], off[e + 1], 25)
        z[idx] += rng.normal(0, 0.2, idx.shape[0]).astype(np.float32)
    d2 = dict(d); d2["z"] = z
    got = gpu(velo, d2)
    assert got["n_deferred"] == 5
    check(got, cpu(d2))
    z3 = d["z"].copy(); z3[z3 == 1.0] = np.float32(1.0) + np.float32(2.0 ** -20)   # every event, one module
    d3 = dict(d); d3["z"] = z3
    got = gpu(velo, d3)
    assert got["n_deferred"] >= 25      # every event with a hit on that module
    check(got, cpu(d3))


def test_events_the_team_kernel_gives_up_on_midway(velo):
    """Deferral after work has started: (a) more candidates than the team path's table (n/8 + 32)
    - an event made of short tracks only; (b) more than 2047 hits in one phi bucket; (c) a module
    holding every hit. All three continue in the general kernel and must still equal the oracle."""
    import oracle
    rng = np.random.default_rng(11)
    # (a) 120 three-hit tracks on modules 10, 11, 12, spread in phi: 360 hits, 120 candidates > 77
    xs, ys, zs, ms = [], [], [], []
    for k in range(120):
        phi = 2 * np.pi * (k + 0.37) / 120
        tx, ty = 0.08 * np.cos(phi), 0.08 * np.sin(phi)
        for m in (10, 11, 12):
            z = float(T.MODULE_Z[m])
            xs.append(tx * z); ys.append(ty * z); zs.append(z); ms.append(m)
    short = (np.array(xs, np.float32), np.array(ys, np.float32), np.array(zs, np.float32), np.array(ms, np.uint8))
    # (b) 2500 hits of module 7 inside one phi bucket (plus a track elsewhere)
    r = rng.uniform(6.0, 40.0, 2500); ph = rng.uniform(0.50, 0.52, 2500)
    line = T.line_event([10, 11, 12, 13], tx=-0.1, ty=0.02)
    dense = (np.concatenate([(r * np.cos(ph)).astype(np.float32), line[0]]),
             np.concatenate([(r * np.sin(ph)).astype(np.float32), line[1]]),
             np.concatenate([np.full(2500, T.MODULE_Z[7], np.float32), line[2]]),
             np.concatenate([np.full(2500, 7, np.uint8), line[3]]))
    # (c) 700 hits, all on module 3, all over phi
    r = rng.uniform(6.0, 40.0, 700); ph = rng.uniform(-np.pi, np.pi, 700)
    flat = ((r * np.cos(ph)).astype(np.float32), (r * np.sin(ph)).astype(np.float32),
            np.full(700, T.MODULE_Z[3], np.float32), np.full(700, 3, np.uint8))
    normal = T.line_event([10, 11, 12, 13, 14])
    x, y, z, m, off = T.batch_of([normal, short, normal, dense, flat, normal])
    got = velo.reconstruct(x, y, z, m, off, datagen.MODULE_Z)
    want = oracle.reconstruct(x, y, z, m, off, M)
    check(got, want)
    assert got["n_deferred"] >= 2 and want["n_tracks"] >= 120 + 3 + 1
    slab = velo.reconstruct(x, y, z, m, off, datagen.MODULE_Z, opts=velo.LaunchOptions(path=velo.VELO_PATH_SLAB_ONLY))
    check(slab, want)


@pytest.mark.parametrize("n_modules", [3, 4, 17, 32])
def test_other_module_counts(velo, n_modules):
    import oracle
    from dataclasses import replace
    mz = tuple(np.linspace(-50.0, 700.0, n_modules).round(0).tolist())
    cfg = replace(datagen.GenConfig(), module_z=mz)
    d = datagen.generate(cfg, 0, 24)
    got = velo.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], np.array(mz))
    want = oracle.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], n_modules)
    check(got, want)
    slab = velo.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], np.array(mz),
                            opts=velo.LaunchOptions(path=velo.VELO_PATH_SLAB_ONLY))
    check(slab, want)
    if n_modules >= 4:
        assert want["n_tracks"] > 0


# ---- the other workloads ------------------------------------------------------------------------
def test_config1_10k_events(velo):
    d = datagen.generate_config(1)
    got = gpu(velo, d)
    want = cpu(d)
    check(got, want)


def test_config3_open_velo(velo):
    d = datagen.generate_config(3, n_events=20000)
    check(gpu(velo, d, n_batches=4), cpu(d))


def test_config4_ion_like(velo):
    d = datagen.generate_config(4, n_events=160)
    nh = np.diff(d["event_offsets"].astype(np.int64))
    assert nh.max() > 20000                  # the large-event path is exercised
    got = gpu(velo, d)
    assert 0 < got["n_big"] + got["n_deferred"] < 160      # the per-SM pipeline and the one-event-per-CTA pipeline took part
    check(got, cpu(d))
    # the same batch through the general kernel alone, and with the large events in the general kernel (mu-like batch rule)
    check(gpu(velo, d, opts=velo.LaunchOptions(path=1)), cpu(d))


# ---- hand-made and degenerate inputs (SURVEY.md §8(c) whole-path pins, A14, A15) -----------------
def _run_events(velo, events, params=None):
    x, y, z, m, off = T.batch_of(events)
    d = {"x": x, "y": y, "z": z, "module": m, "event_offsets": off, "n_events": len(events)}
    got = velo.reconstruct(x, y, z, m, off, datagen.MODULE_Z, params=params)
    import oracle
    want = oracle.reconstruct(x, y, z, m, off, M, None if params is None else _oracle_params(params))
    return got, want, d


def _oracle_params(p):
    import oracle
    q = oracle.Params()
    for name, _ in q._fields_:
        setattr(q, name, getattr(p, name))
    return q


def test_hand_events_and_empty_events(velo):
    empty = (np.zeros(0, np.float32),) * 3 + (np.zeros(0, np.uint8),)
    events = [
        T.line_event([10, 11, 12, 13]),
        empty,
        T.line_event([10, 11, 12, 13, 14, 15]),
        T.line_event([10, 11, 13, 14, 15]),                      # one miss bridged
        T.line_event([13, 14, 15, 10]),                          # weak 3-hit track + lone hit
        T.line_event([9, 10, 11, 14, 15, 16]),                   # two consecutive misses: two tracks
        T.line_event([10, 12, 13]),                              # no three consecutive modules
        T.line_event([10, 11, 12, 13], extra=[(7.6 + 0.07, 0.05, 11), (10.1 + 0.07, 0.05, 12)]),
        empty,
        T.line_event(list(range(26)), tx=0.02, ty=-0.03),        # crosses every module
        T.line_event([3, 4, 5, 6], tx=0.05, ty=0.0),             # x < 0, y = 0: phi16 = -32768
        tuple(np.concatenate(p) for p in zip(T.line_event([3, 4, 5, 6], tx=0.05, ty=2e-4),     # two tracks on
                                             T.line_event([3, 4, 5, 6], tx=0.05, ty=-2e-4))),  # either side of the wrap
    ]
    got, want, d = _run_events(velo, events)
    check(got, want)
    assert [len(T.split_tracks(got, e)) for e in range(len(events))] == [1, 0, 1, 1, 1, 2, 0, 1, 0, 2, 1, 2]
    assert T.track_modules(got, d["module"], 3) == [(15, 14, 13, 11, 10)]


def test_zero_events_and_all_empty(velo):
    z = np.zeros(0, np.float32)
    r = velo.reconstruct(z, z, z, np.zeros(0, np.uint8), np.zeros(1, np.uint32), datagen.MODULE_Z)
    assert r["n_tracks"] == 0 and r["event_track_offsets"].tolist() == [0]
    r = velo.reconstruct(z, z, z, np.zeros(0, np.uint8), np.zeros(6, np.uint32), datagen.MODULE_Z)
    assert r["n_tracks"] == 0 and r["event_track_offsets"].tolist() == [0] * 6


def test_duplicate_hits_and_ties(velo):
    """A14: identical coordinates are legal; ties resolve by index on both sides alike."""
    e = T.line_event([10, 11, 12, 13, 14])
    dup = tuple(np.concatenate([a, a]) for a in e)
    got, want, _ = _run_events(velo, [dup, e, dup])
    check(got, want)


def test_parameter_variants(velo):
    d = datagen.generate_config(0, n_events=30)
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    for change in ({"phi_window_seed": 40000, "phi_window_fwd": 40000},      # whole-module windows
                   {"phi_window_seed": 0, "phi_window_fwd": 5},
                   {"max_skipped": 0}, {"max_skipped": 3},
                   {"clone_num": 0, "clone_den": 1}, {"clone_num": 1, "clone_den": 1},
                   {"max_chi2_ndof": 2.0}, {"max_scatter_seed": 0.5, "max_scatter_fwd": 0.02, "max_scatter_weak": 0.5},
                   # cuts at the edges of the single-comparison form of the scans: nothing passes (negative), only an exact
                   # match passes (zero), the largest finite cut, and cuts that are not finite (these take the general kernel)
                   {"max_scatter_seed": -1.0, "max_scatter_fwd": 0.1}, {"max_scatter_seed": 0.1, "max_scatter_fwd": 0.0},
                   {"max_scatter_seed": 3.4028234663852886e38, "max_scatter_fwd": 3.4028234663852886e38, "phi_window_seed": 60, "phi_window_fwd": 60},
                   {"max_scatter_seed": float("inf"), "max_scatter_fwd": 0.1, "phi_window_seed": 60},
                   {"max_scatter_seed": 0.1, "max_scatter_fwd": float("nan")}):
        p = velo.velo_params_default(g)
        for k, v in change.items():
            setattr(p, k, v)
        got = velo.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], datagen.MODULE_Z, params=p,
                               cap_tracks=d["n_hits"], cap_track_hits=4 * d["n_hits"])     # (wide cuts make many tracks)
        check(got, cpu(d, _oracle_params(p), workers=4))


def test_status_codes(velo):
    d = datagen.generate_config(0, n_events=10)
    # capacity overflow: required sizes are reported, nothing is silently truncated
    full = gpu(velo, d)
    with pytest.raises(velo.VeloError) as e:
        gpu(velo, d, cap_tracks=full["n_tracks"] - 1)
    assert e.value.code == velo.VELO_ERR_CAPACITY and f"tracks={full['n_tracks']}" in str(e.value)
    with pytest.raises(velo.VeloError) as e:
        gpu(velo, d, cap_track_hits=full["n_track_hits"] - 1)
    assert e.value.code == velo.VELO_ERR_CAPACITY
    exact = gpu(velo, d, cap_tracks=full["n_tracks"], cap_track_hits=full["n_track_hits"])
    np.testing.assert_array_equal(exact["track_hits"], full["track_hits"])
    # bad module id
    bad = dict(d); bad["module"] = d["module"].copy(); bad["module"][5] = 26
    with pytest.raises(velo.VeloError) as e:
        gpu(velo, bad)
    assert e.value.code == velo.VELO_ERR_INPUT
    # non-monotone offsets
    bad = dict(d); bad["event_offsets"] = d["event_offsets"].copy(); bad["event_offsets"][3] = bad["event_offsets"][5] + 7
    with pytest.raises(velo.VeloError) as e:
        gpu(velo, bad)
    assert e.value.code == velo.VELO_ERR_INPUT


# ---- full size, in the launch configuration bench.py times: EVERY event against the oracle ----------
def _compare_in_chunks(got, d, chunk):
    """All events, a chunk of events at a time (bounds the host memory of the comparison)."""
    identical = True
    for e0 in range(0, d["n_events"], chunk):
        ids = np.arange(e0, min(e0 + chunk, d["n_events"]))
        sub = T.gather_events(d, ids)
        info = check(T.select_events(got, d, ids), cpu(sub))
        identical &= info["bit_identical_states"]
    return identical


@pytest.mark.parametrize("config", [2, 3])
def test_full_size_every_event(velo, config):
    d = datagen.generate_config(config)
    got = gpu(velo, d, n_batches=4)
    assert got["n_deferred"] == 0
    assert _compare_in_chunks(got, d, 25000)
    # properties that hold at any size
    eto = got["event_track_offsets"].astype(np.int64); tho = got["track_hit_offsets"].astype(np.int64)
    assert (np.diff(eto) >= 0).all() and (np.diff(tho) >= 3).all() and tho[-1] == got["n_track_hits"]
    ev_of_track = np.repeat(np.arange(d["n_events"]), np.diff(eto))
    ev_of_hit = np.repeat(ev_of_track, np.diff(tho))
    off = d["event_offsets"].astype(np.int64)
    th = got["track_hits"].astype(np.int64)
    assert ((th >= off[ev_of_hit]) & (th < off[ev_of_hit + 1])).all()        # hits belong to their event
    mod = d["module"][th].astype(np.int64)
    same_track = np.ones(th.shape[0] - 1, bool); same_track[tho[1:-1] - 1] = False
    assert (np.diff(mod)[same_track] < 0).all()                              # decreasing module order


def test_one_launch_beyond_a_single_wave_of_the_scans(velo):
    """More than 148 x 256 events in ONE launch: a thread of velo_offsets_kernel then takes several events
    (its chunks no longer hold 256), velo_order_kernel runs a few hundred CTAs, and the offsets must still
    be the exclusive scan over all events. Every event against the oracle, and against four streamed batches."""
    d = datagen.generate_config(3, n_events=60000)
    got = gpu(velo, d, n_batches=1)
    assert got["n_deferred"] == 0
    assert _compare_in_chunks(got, d, 20000)
    four = gpu(velo, d, n_batches=4)
    for k in ("event_track_offsets", "track_hit_offsets"):
        np.testing.assert_array_equal(got[k], four[k])


# ---- the end-to-end call over host buffers: velo_scheduler_run_host (S8) --------------------------
def _run_scheduler(velo, d, cuts, n_streams, pinned=True):
    import torch
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    P = velo.velo_params_default(g)
    off = d["event_offsets"]
    sizes = [(cuts[b + 1] - cuts[b], int(off[cuts[b + 1]]) - int(off[cuts[b]])) for b in range(len(cuts) - 1)]
    sched = velo.Scheduler(g, n_streams, max(1, max(s[0] for s in sizes)), max(s[1] for s in sizes))
    outs = [velo.HostTracks(ne, nh, pinned=pinned) for ne, nh in sizes]
    sched.run_host(P, d["x"], d["y"], d["z"], d["module"], off, cuts, outs)
    torch.cuda.synchronize()
    res = velo.stitch([o.result() for o in outs])
    sched.close()
    return res


def test_scheduler_host_buffers_equal_oracle(velo):
    d = datagen.generate_config(1, n_events=611)
    want = cpu(d)
    # ragged batches, more batches than streams (every lane is reused), one empty batch
    cuts = [0, 100, 100, 333, 334, 500, 611]
    for n_streams, pinned in ((2, True), (4, False), (1, True)):
        got = _run_scheduler(velo, d, cuts, n_streams, pinned)
        info = check(got, want)
        assert info["bit_identical_states"]
        np.testing.assert_array_equal(got["track_hits"], want["track_hits"])


def test_scheduler_reports_an_oversized_batch(velo):
    import torch
    d = datagen.generate_config(0, n_events=20)
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    P = velo.velo_params_default(g)
    off = d["event_offsets"]
    sched = velo.Scheduler(g, 2, 10, int(off[10]))          # sized for the first ten events only
    outs = [velo.HostTracks(10, int(off[10])), velo.HostTracks(10, int(off[20]) - int(off[10]))]
    sched.run_host(P, d["x"], d["y"], d["z"], d["module"], off, [0, 10, 20], outs)
    torch.cuda.synchronize()
    first = outs[0].result()
    assert first["n_tracks"] > 0
    if int(off[20]) - int(off[10]) > int(off[10]):          # the second batch has more hits than the lanes hold
        with pytest.raises(velo.VeloError) as e:
            outs[1].result()
        assert e.value.code == velo.VELO_ERR_CAPACITY
    sched.close()


def test_config4_full_size_every_event(velo):
    """BASELINE.json:configs[4] at full size (2 000 ion-like events, one call): every event against the
    oracle; events above 12 000 hits run in the one-event-per-CTA pipeline, the others in the per-SM pipeline."""
    d = datagen.generate_config(4)
    got = gpu(velo, d)
    assert 0 < got["n_big"] < d["n_events"] and got["n_deferred"] < 20
    assert _compare_in_chunks(got, d, 500)


def test_scheduler_summary_is_eight_words(velo):
    """include/velo.h: out[b].summary is a HOST u32[VELO_N_SUMMARY]; nothing is written past it."""
    import ctypes
    import torch
    d = datagen.generate_config(0, n_events=16)
    g = velo.velo_geometry_load(datagen.MODULE_Z)
    P = velo.velo_params_default(g)
    off = d["event_offsets"]
    sched = velo.Scheduler(g, 2, 16, int(off[16]))
    out = velo.HostTracks(16, int(off[16]))
    guard = torch.full((velo.VELO_N_SUMMARY + 8,), 0x5A5A5A5A, dtype=torch.int32)
    out.summary = guard[:velo.VELO_N_SUMMARY]
    sched.run_host(P, d["x"], d["y"], d["z"], d["module"], off, [0, 16], [out])
    torch.cuda.synchronize()
    assert (guard[velo.VELO_N_SUMMARY:] == 0x5A5A5A5A).all()
    assert out.result()["n_tracks"] > 0
    sched.close()
