"""Whole-path pins of the oracle (SURVEY.md §8(c) "Whole-path pins" (i)...(vii), O-6 ... O-13):
exhaustive triplet enumeration, ideal straight tracks all found, hand examples with stated
outcomes, brute-force restatements of the ghost and clone rules, invariants. CPU only."""
import itertools
from dataclasses import replace

import numpy as np

import oracle
from paper_2412_05041_b200 import datagen
from tests.velo_testlib import MODULE_Z, batch_of, canonical, line_event, split_tracks, track_modules

F = np.float32


def run(ev, params=None, n_modules=26):
    x, y, z, m, off = batch_of([ev])
    return oracle.reconstruct(x, y, z, m, off, n_modules, params)


# ---------------------------------------------------------------- (i) exhaustive triplets
def _scatter32(h0, h1, h2):
    """Independent evaluation in float64 of the squared extrapolation miss (only used to RANK
    triplets whose float32 scatters differ by far more than rounding)."""
    (x0, y0, z0), (x1, y1, z1), (x2, y2, z2) = h0, h1, h2
    tz = (z2 - z1) / (z1 - z0)
    return ((x1 + (x1 - x0) * tz) - x2) ** 2 + ((y1 + (y1 - y0) * tz) - y2) ** 2


def test_seeding_equals_exhaustive_triplet_enumeration():
    rng = np.random.default_rng(123)
    P = oracle.default_params()
    P.phi_window_seed = 32768       # whole module
    P.max_scatter_seed = 4.0
    for trial in range(60):
        n = [int(rng.integers(1, 9)) for _ in range(3)]
        mod = np.repeat(np.arange(3), n).astype(np.uint8)
        x = rng.uniform(-3, 3, mod.size).astype(F)
        y = rng.uniform(-3, 3, mod.size).astype(F)
        z = np.array([0.0, 25.0, 50.0], F)[mod]
        c = oracle.event_candidates(x, y, z, mod, 3, P)
        perm = c["perm"]
        pos = np.empty_like(perm); pos[perm] = np.arange(perm.size)     # original -> sorted index
        want = {}
        for i1 in np.where(mod == 1)[0]:
            best = None
            for i0, i2 in itertools.product(np.where(mod == 2)[0], np.where(mod == 0)[0]):
                sc = _scatter32(*[(float(x[i]), float(y[i]), float(z[i])) for i in (i0, i1, i2)])
                if sc <= 4.0 * (1 - 1e-6):
                    key = (sc, int(pos[i0]), int(pos[i2]))
                    if best is None or key < best:
                        best = key
            if best is not None:
                want[int(pos[i1])] = (best[1], best[2])
        got = {int(c["hits"][t, 1]): (int(c["hits"][t, 0]), int(c["hits"][t, 2])) for t in range(c["n_cand"])}
        assert got == want, trial
        # candidates are appended in sorted-h1 order, one per centre hit
        assert list(c["centre"]) == sorted(got)


def test_seeding_tie_break_lowest_indices():
    # duplicate hits (A14): identical coordinates -> equal scatter -> lowest sorted index wins,
    # and sorted index ties resolve by original index (O-2)
    ev = line_event([12, 11, 10], extra=[(0.1 * 101, 0.0, 12), (0.1 * 51, 0.0, 10)])
    c = oracle.event_candidates(*ev, 26)
    assert c["n_cand"] == 1
    h0, h1, h2 = (int(c["perm"][i]) for i in c["hits"][0, :3])
    assert (h0, h1, h2) == (0, 1, 2)      # the duplicates (original indices 3, 4) lose the tie


# ---------------------------------------------------------------- (ii) ideal tracks all found
def test_ideal_straight_tracks_all_found_exactly():
    # north_star: "every noise-free straight-line track with >=3 hits found". In EVERY event each
    # such track is contained in exactly one output track; in events whose tracks are well separated
    # in phi (> 0.08 rad = 2.8 windows) the output is exactly the truth (SURVEY.md §8(c) pin (ii)).
    cfg = datagen.ideal_config(mu=1.0, trk_mean=6.0)
    d = datagen.generate(cfg, 0, 600, truth=True)
    r = oracle.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], 26)
    assert r["status"] == 0
    n_exact = n_all = 0
    for e in range(600):
        o0, o1 = int(d["event_offsets"][e]), int(d["event_offsets"][e + 1])
        truth = {}
        for h in range(o0, o1):
            truth.setdefault(int(d["hit_track"][h]), set()).add(h)
        want = sorted(tuple(sorted(s)) for s in truth.values() if len(s) >= 3)
        got = sorted(tuple(sorted(hits)) for hits, _ in split_tracks(r, e))
        for w in want:
            assert sum(set(w) <= set(g) for g in got) == 1, e
        n_all += len(want)
        ids = sorted(truth)
        phi = np.sort(np.arctan2(d["trk_truth"][ids, 4], d["trk_truth"][ids, 3]))
        gaps = np.diff(np.concatenate([phi, phi[:1] + 2 * np.pi])) if len(ids) > 1 else np.array([9.0])
        if gaps.min() > 0.08:
            assert got == want, e
            n_exact += len(want)
    assert n_all > 2000 and n_exact > 400


def test_ideal_tracks_fit_reproduces_generating_line():
    cfg = datagen.ideal_config(mu=1.0, trk_mean=12.0)
    d = datagen.generate(cfg, 0, 50, truth=True)
    r = oracle.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], 26)
    n = 0
    for e in range(50):
        for hits, st in split_tracks(r, e):
            xv, yv, zv, tx, ty = d["trk_truth"][int(d["hit_track"][hits[0]])]
            assert abs(st[2] - tx) < 2e-6 + 1e-5 * abs(tx) and abs(st[3] - ty) < 2e-6 + 1e-5 * abs(ty)
            # state at closest approach to the z axis lies on the generating line
            assert abs(st[0] - (xv + tx * (st[4] - zv))) < 2e-3 and abs(st[1] - (yv + ty * (st[4] - zv))) < 2e-3
            n += 1
    assert n > 200


# ---------------------------------------------------------------- (iii)-(v) hand examples
def test_hand_four_hit_line():
    ev = line_event([13, 12, 11, 10])
    r = run(ev)
    trk = split_tracks(r, 0)
    assert len(trk) == 1 and trk[0][0] == (0, 1, 2, 3)
    st = trk[0][1]
    assert abs(st[2] - 0.1) < 1e-6 and st[3] == 0 and abs(st[0]) < 1e-4 and st[1] == 0 and abs(st[4]) < 1e-3
    assert st[11] < 1e-3 and st[12:13].view(np.uint32)[0] == 4


def test_hand_three_hit_weak_track_survives_and_dies_when_flagged():
    assert track_modules(run(line_event([12, 11, 10])), line_event([12, 11, 10])[3]) == [(12, 11, 10)]
    # (iv) dies if a 4-hit track flags one of its hits: a second line through the same module-12 hit
    x12, z12 = 0.1 * 101.0, 101.0
    ev = line_event([12, 11, 10])
    extra = []
    for m in (13, 11, 10):     # line through (x12, 0.0) with ty = 0.004: distinct from the first
        z = float(MODULE_Z[m])
        extra.append((x12 + 0.1 * (z - z12), 0.004 * (z - z12), m))
    ev2 = line_event([12, 11, 10], extra=extra)
    r = run(ev2)
    mods = track_modules(r, ev2[3])
    assert (13, 12, 11, 10) in mods
    c = oracle.event_candidates(*ev2, 26)
    # every 3-hit candidate containing a flagged hit is removed by O-10
    for t in range(c["n_cand"]):
        if c["n"][t] == 3 and c["flags"][c["hits"][t, :3]].any():
            assert not c["pass"][t]


def test_hand_skip_behaviour():
    def mods(modules, **kw):
        ev = line_event(modules, **kw)
        return track_modules(run(ev), ev[3])
    assert mods([15, 14, 13, 12, 11, 10]) == [(15, 14, 13, 12, 11, 10)]
    assert mods([15, 14, 13, 11, 10]) == [(15, 14, 13, 11, 10)]            # one miss bridged
    assert mods([15, 14, 13, 10]) == [(15, 14, 13)]                        # two misses end the track
    assert mods([16, 15, 14, 11, 10, 9]) == [(11, 10, 9), (16, 15, 14)]    # two 3-hit tracks
    assert mods([13, 12, 10]) == []                                        # seeds need consecutive modules
    stray = [(0.1 * 76 + 0.07, 0.05, 11), (0.1 * 101 - 0.06, -0.08, 12)]
    assert mods([13, 12, 11, 10], extra=stray) == [(13, 12, 11, 10)]


def test_max_skipped_parameter():
    P = oracle.default_params(); P.max_skipped = 0
    ev = line_event([15, 14, 13, 11, 10, 9])
    assert track_modules(run(ev, P), ev[3]) == [(11, 10, 9), (15, 14, 13)]
    P.max_skipped = 2
    ev = line_event([15, 14, 13, 10, 9])
    assert track_modules(run(ev, P), ev[3]) == [(15, 14, 13, 10, 9)]


# ---------------------------------------------------------------- O-10, O-12, O-13 restated
def _check_filters(x, y, z, mod, P):
    c = oracle.event_candidates(x, y, z, mod, 26, P)
    nc = c["n_cand"]
    hits = [tuple(int(v) for v in c["hits"][t, :c["n"][t]]) for t in range(nc)]
    # flags: exactly the hits of candidates that reached 4 hits
    want_flags = np.zeros(x.size, bool)
    for t in range(nc):
        if c["n"][t] >= 4:
            want_flags[list(hits[t])] = True
    assert (c["flags"] == want_flags).all()
    chi2 = c["states"][:, 11]
    for t in range(nc):
        ok = True
        if c["n"][t] == 3:
            ok = (not want_flags[list(hits[t])].any()) and c["seed_scatter"][t] <= P.max_scatter_weak
        if ok:
            ok = not (chi2[t] > F(P.max_chi2_ndof) * F(2 * int(c["n"][t]) - 4))
        assert bool(c["pass"][t]) == ok, t
    # clone rule, O(T^2): a hit is lost if ANOTHER passing candidate containing it is better
    # under (more hits, lower chi2, lower centre index)
    rank = lambda t: (-int(c["n"][t]), float(chi2[t]), int(c["centre"][t]))
    for t in range(nc):
        if not c["pass"][t]:
            assert not c["survive"][t]
            continue
        lost = 0
        for h in hits[t]:
            if any(u != t and c["pass"][u] and h in hits[u] and rank(u) < rank(t) for u in range(nc)):
                lost += 1
        assert lost == c["lost"][t], t
        assert bool(c["survive"][t]) == (not (lost * P.clone_den > int(c["n"][t]) * P.clone_num)), t
    # key packs (255-n, chi2 bits, centre)
    for t in range(nc):
        if c["pass"][t]:
            k = int(c["key"][t])
            assert k >> 56 == 255 - int(c["n"][t]) and k & 0xFFFFFF == int(c["centre"][t])
            assert (k >> 24) & 0xFFFFFFFF == int(chi2[t:t + 1].view(np.uint32)[0])
    return c


def test_filters_bruteforce_on_generated_events(cfg0):
    d = cfg0
    P = oracle.default_params()
    tot_killed = 0
    for e in range(12):
        o0, o1 = int(d["event_offsets"][e]), int(d["event_offsets"][e + 1])
        c = _check_filters(d["x"][o0:o1], d["y"][o0:o1], d["z"][o0:o1], d["module"][o0:o1], P)
        tot_killed += int((c["pass"] & ~c["survive"]).sum())
    # a denser, noisier event sample so that clones and ghosts actually occur
    cfg = replace(datagen.GenConfig(), ion_mode=True, mult_lo=800, mult_hi=1500, noise_frac=0.05, seed=5)
    dd = datagen.generate(cfg, 0, 2)
    for e in range(2):
        o0, o1 = int(dd["event_offsets"][e]), int(dd["event_offsets"][e + 1])
        c = _check_filters(dd["x"][o0:o1], dd["y"][o0:o1], dd["z"][o0:o1], dd["module"][o0:o1], P)
        tot_killed += int((c["pass"] & ~c["survive"]).sum())
    assert tot_killed > 0


# (the clone rule on real candidate pairs with stated outcomes: tests/test_oracle_hand_events.py)


# ---------------------------------------------------------------- (vi), (vii), edge cases
def test_order_independence_under_input_permutation(cfg0):
    d = cfg0
    rng = np.random.default_rng(17)
    for e in range(6):
        o0, o1 = int(d["event_offsets"][e]), int(d["event_offsets"][e + 1])
        ev = tuple(d[k][o0:o1] for k in ("x", "y", "z", "module"))
        p = rng.permutation(o1 - o0)
        evp = tuple(a[p] for a in ev)
        ra, rb = run(ev), run(evp)
        coords = lambda r, E: sorted(tuple((float(E[0][h]), float(E[1][h]), float(E[2][h])) for h in hits)
                                     for hits, _ in split_tracks(r, 0))
        assert coords(ra, ev) == coords(rb, evp)


def test_physics_sanity_config0(cfg0):
    # indicative only (SURVEY.md §8 probe: 99.5 % / 0.05 % / 0.13 % with another RNG)
    d = cfg0
    r = oracle.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], 26)
    ht = d["hit_track"]
    n_reco = {}
    ghosts = clones = 0
    matched = set()
    tho, th = r["track_hit_offsets"], r["track_hits"]
    for t in range(r["n_tracks"]):
        ids = ht[th[tho[t]:tho[t + 1]]]
        vals, cnt = np.unique(ids, return_counts=True)
        k = int(np.argmax(cnt))
        if vals[k] < 0 or cnt[k] < 0.7 * ids.size:
            ghosts += 1
        elif int(vals[k]) in matched:
            clones += 1
        else:
            matched.add(int(vals[k]))
    ids, cnt = np.unique(ht[ht >= 0], return_counts=True)
    reconstructible = set(int(i) for i in ids[cnt >= 3])
    eff = len(matched & reconstructible) / len(reconstructible)
    assert eff > 0.985 and ghosts / r["n_tracks"] < 0.01 and clones / r["n_tracks"] < 0.01
    assert 150 < r["n_tracks"] / 100 < 260


def test_edge_cases_empty_inputs():
    z = np.zeros(0, F)
    r = oracle.reconstruct(z, z, z, np.zeros(0, np.uint8), np.zeros(1, np.uint32), 26)
    assert r["n_tracks"] == 0 and r["status"] == 0 and r["event_track_offsets"].tolist() == [0]
    r = oracle.reconstruct(z, z, z, np.zeros(0, np.uint8), np.zeros(4, np.uint32), 26)
    assert r["n_tracks"] == 0 and r["event_track_offsets"].tolist() == [0, 0, 0, 0]
    # an empty event between two non-empty ones; global hit indices carry the event offset
    e = line_event([13, 12, 11, 10])
    x, y, zz, m, off = batch_of([e, (z, z, z, np.zeros(0, np.uint8)), e])
    r = oracle.reconstruct(x, y, zz, m, off, 26)
    assert r["event_track_offsets"].tolist() == [0, 1, 1, 2]
    assert r["track_hits"].tolist() == [0, 1, 2, 3, 4, 5, 6, 7]
    cz = canonical(r)
    assert cz["n"].tolist() == [4, 4]


def test_bad_input_status():
    e = line_event([13, 12, 11, 10])
    x, y, z, m, off = batch_of([e])
    m2 = m.copy(); m2[0] = 26
    assert oracle.reconstruct(x, y, z, m2, off, 26)["status"] == -6
    assert oracle.reconstruct(x, y, z, m, np.array([0, 4, 2], np.uint32), 26)["status"] == -6
