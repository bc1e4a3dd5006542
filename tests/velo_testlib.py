"""Shared helpers for the tests: canonical ordering, comparison rule
(O-17), hand-made events. Holds no method arithmetic of either side."""
from __future__ import annotations

import numpy as np

from paper_2412_05041_b200 import datagen

MODULE_Z = datagen.MODULE_Z.astype(np.float32)
M = MODULE_Z.shape[0]


def split_tracks(res: dict, event: int):
    """List of (hit-index tuple, state vector[13]) of one event."""
    eto, tho, th, st = res["event_track_offsets"], res["track_hit_offsets"], res["track_hits"], res["states"]
    out = []
    for t in range(int(eto[event]), int(eto[event + 1])):
        hits = tuple(int(v) for v in th[int(tho[t]):int(tho[t + 1])])
        out.append((hits, np.array(st[:, t], dtype=np.float32)))
    return out


def canonical_order(res: dict) -> np.ndarray:
    """Permutation of track ids putting every event's tracks in canonical order (O-16): by hit list,
    lexicographic. The first two hits (h0, centre h1) are unique per candidate (O-8: one seed per
    centre hit), so (event, hits[0], hits[1]) is a total order equal to the lexicographic one."""
    eto = np.asarray(res["event_track_offsets"], dtype=np.int64)
    tho = np.asarray(res["track_hit_offsets"], dtype=np.int64)
    th = np.asarray(res["track_hits"], dtype=np.int64)
    nt = int(eto[-1])
    if nt == 0:
        return np.zeros(0, dtype=np.int64)
    ev = np.repeat(np.arange(eto.shape[0] - 1), np.diff(eto))
    h0 = th[tho[:nt]]
    h1 = th[tho[:nt] + 1]
    return np.lexsort((h1, h0, ev))


def canonical(res: dict) -> dict:
    """Canonically ordered copy: event_track_offsets, per-track n, flattened hits, states."""
    eto = np.asarray(res["event_track_offsets"], dtype=np.int64)
    tho = np.asarray(res["track_hit_offsets"], dtype=np.int64)
    th = np.asarray(res["track_hits"])
    nt = int(eto[-1])
    order = canonical_order(res)
    n = (tho[1:nt + 1] - tho[:nt])[order]
    starts = tho[:nt][order]
    new_off = np.zeros(nt + 1, dtype=np.int64)
    np.cumsum(n, out=new_off[1:])
    idx = np.repeat(starts - new_off[:-1], n) + np.arange(int(new_off[-1]))
    hits = th[idx] if nt else th[:0]
    st = np.asarray(res["states"])[:, :nt][:, order]
    return {"event_track_offsets": eto, "n": n, "track_hit_offsets": new_off, "track_hits": hits, "states": st}


def assert_same_result(got: dict, want: dict, rel: float = 1e-5):
    """O-17: hit lists, offsets, n_hits bit-exact; states |g-o| <= rel*|o| with 0 == 0 passing."""
    a, b = canonical(got), canonical(want)
    np.testing.assert_array_equal(a["event_track_offsets"], b["event_track_offsets"])
    np.testing.assert_array_equal(a["n"], b["n"])
    np.testing.assert_array_equal(a["track_hits"], b["track_hits"])
    ga, wa = a["states"], b["states"]
    # last plane: n_hits as u32 bits, exact
    np.testing.assert_array_equal(ga[12].view(np.uint32), wa[12].view(np.uint32))
    np.testing.assert_array_equal(ga[12].view(np.uint32).astype(np.int64), a["n"])
    g = ga[:12].astype(np.float64)
    w = wa[:12].astype(np.float64)
    bad = np.abs(g - w) > rel * np.abs(w)
    assert not bad.any(), f"{int(bad.sum())} state words beyond {rel} relative; first at {np.argwhere(bad)[:5]}"
    return {"bit_identical_states": bool(np.array_equal(ga.view(np.uint32), wa.view(np.uint32)))}


def line_event(modules, tx=0.1, ty=0.0, x0=0.0, y0=0.0, extra=()):
    """Hits of the line x = x0 + tx z, y = y0 + ty z on the given modules (fp32-rounded), plus
    extra (x, y, module) hits. Returns x, y, z, module arrays."""
    xs, ys, zs, ms = [], [], [], []
    for m in modules:
        z = float(MODULE_Z[m])
        xs.append(x0 + tx * z); ys.append(y0 + ty * z); zs.append(z); ms.append(m)
    for (x, y, m) in extra:
        xs.append(x); ys.append(y); zs.append(float(MODULE_Z[m])); ms.append(m)
    return (np.array(xs, np.float32), np.array(ys, np.float32), np.array(zs, np.float32),
            np.array(ms, np.uint8))


def batch_of(events):
    """Concatenate per-event (x, y, z, module) tuples into batch arrays + offsets."""
    off = np.zeros(len(events) + 1, np.uint32)
    for i, e in enumerate(events):
        off[i + 1] = off[i] + e[0].shape[0]
    cat = lambda k, dt: (np.concatenate([e[k] for e in events]).astype(dt) if events else np.zeros(0, dt))
    return cat(0, np.float32), cat(1, np.float32), cat(2, np.float32), cat(3, np.uint8), off


def track_modules(res, module, event=0):
    """Sorted tuple of module-id tuples of the event's tracks."""
    return sorted(tuple(int(module[h]) for h in hits) for hits, _ in split_tracks(res, event))


def gather_events(d: dict, ids) -> dict:
    """Sub-batch made of the selected events of a generated batch (inputs only)."""
    off = d["event_offsets"].astype(np.int64)
    ids = np.asarray(ids, dtype=np.int64)
    n = off[ids + 1] - off[ids]
    new_off = np.zeros(ids.shape[0] + 1, np.int64)
    np.cumsum(n, out=new_off[1:])
    idx = np.repeat(off[ids] - new_off[:-1], n) + np.arange(int(new_off[-1]))
    return {"x": d["x"][idx], "y": d["y"][idx], "z": d["z"][idx], "module": d["module"][idx],
            "event_offsets": new_off.astype(np.uint32), "n_events": ids.shape[0], "n_hits": int(new_off[-1])}


def select_events(res: dict, d: dict, ids) -> dict:
    """The part of a full-batch result that belongs to the selected events, re-indexed as if the
    sub-batch of gather_events(d, ids) had been reconstructed on its own."""
    off = d["event_offsets"].astype(np.int64)
    ids = np.asarray(ids, dtype=np.int64)
    eto = np.asarray(res["event_track_offsets"]).astype(np.int64)
    tho = np.asarray(res["track_hit_offsets"]).astype(np.int64)
    th = np.asarray(res["track_hits"]).astype(np.int64)
    new_hoff = np.concatenate([[0], np.cumsum(off[ids + 1] - off[ids])])
    nt = eto[ids + 1] - eto[ids]
    new_eto = np.concatenate([[0], np.cumsum(nt)])
    tids = np.repeat(eto[ids] - new_eto[:-1], nt) + np.arange(int(new_eto[-1]))
    shift = np.repeat(new_hoff[:-1] - off[ids], nt)          # per selected track: hit index shift
    n = tho[tids + 1] - tho[tids]
    new_tho = np.concatenate([[0], np.cumsum(n)])
    hidx = np.repeat(tho[tids] - new_tho[:-1], n) + np.arange(int(new_tho[-1]))
    hits = th[hidx] + np.repeat(shift, n)
    return {"event_track_offsets": new_eto.astype(np.uint32), "track_hit_offsets": new_tho.astype(np.uint32),
            "track_hits": hits.astype(np.uint32), "states": np.asarray(res["states"])[:, tids],
            "n_tracks": int(new_eto[-1]), "n_track_hits": int(new_tho[-1])}


def oracle_parallel(d: dict, n_modules: int, params=None, workers: int | None = None) -> dict:
    """The oracle over a batch, forked over contiguous event ranges (events are independent), and
    the per-range results stitched. Each worker is the single-threaded oracle as it stands."""
    import multiprocessing as mp
    import os
    ne = int(d["n_events"])
    workers = workers or min(os.cpu_count() or 1, 32)
    workers = max(1, min(workers, ne // 8 or 1))
    off = d["event_offsets"].astype(np.int64)
    tot = int(off[-1] - off[0])
    # cut so that every range holds about the same number of hits
    cuts = [0] + [int(np.searchsorted(off - off[0], tot * k / workers)) for k in range(1, workers)] + [ne]
    cuts = sorted(set(min(max(c, 0), ne) for c in cuts))
    jobs = [(d, n_modules, params, cuts[i], cuts[i + 1]) for i in range(len(cuts) - 1)]
    if len(jobs) == 1:
        parts = [_oracle_range(jobs[0])]
    else:
        with mp.get_context("fork").Pool(len(jobs)) as pool:
            parts = pool.map(_oracle_range, jobs)
    eto, tho, th, st = [np.zeros(1, np.int64)], [np.zeros(1, np.int64)], [], []
    nt = nh = nc = 0
    for p in parts:
        eto.append(p["event_track_offsets"][1:].astype(np.int64) + nt)
        tho.append(p["track_hit_offsets"][1:].astype(np.int64) + nh)
        th.append(p["track_hits"]); st.append(p["states"])
        nt += p["n_tracks"]; nh += p["n_track_hits"]; nc += p["n_candidates"]
    return {"event_track_offsets": np.concatenate(eto).astype(np.uint32),
            "track_hit_offsets": np.concatenate(tho).astype(np.uint32),
            "track_hits": np.concatenate(th), "states": np.concatenate(st, axis=1), "n_tracks": nt,
            "n_track_hits": nh, "status": max((p["status"] for p in parts), key=abs), "n_candidates": nc}


def _oracle_range(job):
    import oracle
    d, n_modules, params, e0, e1 = job
    off = d["event_offsets"]
    h0, h1 = int(off[e0]), int(off[e1])
    r = oracle.reconstruct(d["x"][h0:h1], d["y"][h0:h1], d["z"][h0:h1], d["module"][h0:h1],
                           (off[e0:e1 + 1].astype(np.int64) - h0).astype(np.uint32), n_modules, params)
    r["track_hits"] = r["track_hits"] + np.uint32(h0)
    return r


# ---- hand-made events with STATED outcomes (round 2 pins of O-7, O-8, O-6(B), O-12, A11) ----------
# Each builder returns (event, expected): event = (x, y, z, module) arrays, expected = the list of
# output tracks as tuples of ORIGINAL hit indices in discovery order, in canonical order (O-16).
# The expectations are worked out by hand from SURVEY.md §8(c); nothing here was produced by the
# oracle or by the CUDA path. Modules 5 ... 18 are 25 mm apart (A1), so mirrored displacements
# about a middle module are exactly collinear.
def _hits(rows):
    x = np.array([r[0] for r in rows], np.float32); y = np.array([r[1] for r in rows], np.float32)
    m = np.array([r[2] for r in rows], np.uint8)
    return x, y, MODULE_Z[m.astype(np.int64)].astype(np.float32), m


def _line_a(first_module, n):
    """x = 10 + 0.1 z, y = 0 on n consecutive modules downwards from first_module (phi16 = 0)."""
    return [(10.0 + 0.1 * float(MODULE_Z[m]), 0.0, m) for m in range(first_module, first_module - n, -1)]


def pin_forward_tie(top=13):
    """O-7 tie -> LOWEST sorted index: the forwarding target module holds the same hit twice
    (A14). Sorted index ties resolve by original index (O-2), so the track ends on hit 3, not 4."""
    rows = _line_a(top, 4)
    rows.append(rows[3])                       # duplicate of the hit on the target module
    return _hits(rows), [(0, 1, 2, 3)]


def pin_forward_window_centre():
    """O-7 window is centred on hb (the LATEST hit), not on ha. The line x = 10, y = 0.0077 z is
    straight (scatter 0) but turns by ~201 phi16 units per module: the module-10 hit lies 201
    units from hb (inside W = 300) and 402 units from ha (outside)."""
    rows = [(10.0, 0.0077 * float(MODULE_Z[m]), m) for m in (13, 12, 11, 10)]
    return _hits(rows), [(0, 1, 2, 3)]


def pin_forward_miss_reset():
    """O-7: n_missed returns to 0 after a found hit. Hits on modules 16, 15, 14, 12, 11, 9, 8: each
    gap is ONE missed module, max_skipped = 1 bridges both -> one 7-hit track."""
    rows = [(10.0 + 0.1 * float(MODULE_Z[m]), 0.0, m) for m in (16, 15, 14, 12, 11, 9, 8)]
    return _hits(rows), [(0, 1, 2, 3, 4, 5, 6)]


def pin_seed_flagged_centre(top=13):
    """O-8: a flagged hit is not a seed centre, and O-6(B): the flags of step s are visible to the
    seeding of the SAME step. Line A on modules top ... top-5 reaches 4 hits in (A) of step top-2,
    which flags its hit on module top-2 (hit 2). Strays U(top-1), U(top-3) mirror each other about
    that hit (exactly collinear through it) and U(top-4) continues their line: if hit 2 seeded at
    step top-2 it would give the 4-hit track (U, 2, U, U). It must not: the strays stay unused."""
    rows = _line_a(top, 6)
    xa = lambda m: 10.0 + 0.1 * float(MODULE_Z[m])
    rows += [(xa(top - 1), 0.2, top - 1), (xa(top - 3), -0.2, top - 3), (xa(top - 4), -0.4, top - 4)]
    return _hits(rows), [(0, 1, 2, 3, 4, 5)]


def pin_seed_flagged_h0(top=13):
    """O-8: a flagged hit is not used as h0. Strays C(top-3), C(top-4), C(top-5) are exactly
    collinear with line A's hit on module top-2 (hit 2, flagged at step top-2). At step top-3 the
    centre C(top-3) has only that flagged hit in its module-(top-2) window -> no seed; at step
    top-4 the three strays seed on their own and survive as a weak 3-hit track (scatter 0)."""
    rows = _line_a(top, 6)
    xa = lambda m: 10.0 + 0.1 * float(MODULE_Z[m])
    rows += [(xa(top - 3), 0.15, top - 3), (xa(top - 4), 0.30, top - 4), (xa(top - 5), 0.45, top - 5)]
    return _hits(rows), [(0, 1, 2, 3, 4, 5), (6, 7, 8)]


def pin_seed_flagged_h2(top=13):
    """O-8: a flagged hit is not used as h2, including one flagged in (A)/(B) of the same step.
    Strays V(top-2) = A + 2d, V(top-3) = A + d are exactly collinear with line A's hit on module
    top-4 (hit 4, picked up and flagged at step top-3), and V(top-5) = A - d continues that line.
    At step top-3 the centre V(top-3) finds only the flagged hit 4 in its module-(top-4) window ->
    no seed; used as h2 it would give the 4-hit track (V, V, 4, V)."""
    rows = _line_a(top, 6)
    xa = lambda m: 10.0 + 0.1 * float(MODULE_Z[m])
    rows += [(xa(top - 2), 0.30, top - 2), (xa(top - 3), 0.15, top - 3), (xa(top - 5), -0.15, top - 5)]
    return _hits(rows), [(0, 1, 2, 3, 4, 5)]


def pin_chi2_track(n):
    """O-12: a track with a known chi2. n hits on modules 12 ... 12-n+1 at y = 0, x = 10 except one
    hit displaced by e = 0.03 mm (n = 3: the middle one; n = 5: the middle one). Unweighted LSQ
    leaves residuals (-e/3, 2e/3, -e/3) resp. (-e/5, -e/5, 4e/5, -e/5, -e/5): sum of squares
    2e^2/3 resp. 4e^2/5; chi2 = that / sigma^2 with sigma^2 = 0.055^2/12; ndof = 2n - 4.
    Returns (event, expected track, chi2 in float64)."""
    e = 0.03
    mods = list(range(12, 12 - n, -1))
    rows = [(10.0 + (e if i == n // 2 else 0.0), 0.0, m) for i, m in enumerate(mods)]
    ss = 2 * e * e / 3 if n == 3 else 4 * e * e / 5
    x = np.array([r[0] for r in rows], np.float32).astype(np.float64)
    ss32 = float(((x - x.mean()) ** 2).sum())          # the same sum on the fp32-rounded inputs
    assert abs(ss32 - ss) < 1e-3 * ss
    return _hits(rows), [tuple(range(n))], ss32 / (0.055 ** 2 / 12.0)


def pin_clone_pair():
    """O-13 on a real pair: two centre hits 0.1 mm apart on module 12 both seed with the same h0
    and h2 (seed scatter 0 and 0.04) and both forward onto the same module-10 hit, giving two
    4-hit candidates that share three hits. The straight one has the lower chi2 and owns the
    shared hits; the other loses 3 of 4 (3*3 > 4*1) and is killed."""
    rows = _line_a(13, 4)
    rows.append((rows[1][0], 0.1, 12))
    return _hits(rows), [(0, 1, 2, 3)]


def pin_clone_tie():
    """O-13 tie: two centre hits mirrored about the line (y = +0.1 and -0.1) give candidates with
    bit-identical chi2; the key falls back to the centre's sorted index, and y < 0 sorts first."""
    a = _line_a(13, 4)
    rows = [a[0], (a[1][0], 0.1, 12), (a[1][0], -0.1, 12), a[2], a[3]]
    return _hits(rows), [(0, 2, 3, 4)]


PIN_EVENTS = [pin_forward_tie, lambda: pin_forward_tie(14), pin_forward_window_centre, pin_forward_miss_reset,
              pin_seed_flagged_centre, lambda: pin_seed_flagged_centre(14), pin_seed_flagged_h0,
              lambda: pin_seed_flagged_h0(14), pin_seed_flagged_h2, lambda: pin_seed_flagged_h2(14),
              lambda: pin_chi2_track(3)[:2], lambda: pin_chi2_track(5)[:2],
              pin_clone_pair, pin_clone_tie]
