"""Hand-made events with STATED expected hit lists (SURVEY.md §8(c) O-6 ... O-13, A11): each pins
one decision of the oracle that no invariant or brute-force restatement reaches — the forwarding
tie-break, the centre of the forwarding window, the reset of the miss counter, the exclusion of
flagged hits from seeding (as centre, as h0), the visibility of a step's flags to the seeding of
the same step, the chi2/ndof cut on both sides of its threshold and at equality, the degenerate
slope threshold, and the clone rule on a real pair. The events and their expectations live in
tests/velo_testlib.py (worked out by hand; tests/test_gpu_parity.py runs the same events through
the CUDA path). CPU only."""
import numpy as np
import pytest

import oracle
from tests import velo_testlib as T

SIGMA = float(np.float32(0.055 / np.sqrt(12.0)))


def tracks_of(ev, params=None):
    x, y, z, m, off = T.batch_of([ev])
    r = oracle.reconstruct(x, y, z, m, off, 26, params)
    assert r["status"] == 0
    return sorted(hits for hits, _ in T.split_tracks(r, 0)), r


# ---------------------------------------------------------------- O-7 forwarding
@pytest.mark.parametrize("top", [13, 14])
def test_forwarding_tie_goes_to_the_lowest_index(top):
    ev, want = T.pin_forward_tie(top)
    got, _ = tracks_of(ev)
    assert got == want


def test_forwarding_window_is_centred_on_the_latest_hit():
    ev, want = T.pin_forward_window_centre()
    # the construction holds: consecutive hits ~200 units apart, hits two modules apart ~400
    phi = oracle.phi16(ev[0], ev[1]).astype(int)
    assert all(150 < phi[i] - phi[i + 1] <= 300 for i in range(3)) and all(phi[i] - phi[i + 2] > 300 for i in range(2))
    got, _ = tracks_of(ev)
    assert got == want


def test_forwarding_miss_counter_resets_after_a_found_hit():
    ev, want = T.pin_forward_miss_reset()
    got, _ = tracks_of(ev)
    assert got == want
    P = oracle.default_params(); P.max_skipped = 0          # without bridging only (16, 15, 14) has
    got0, _ = tracks_of(ev, P)                              # three consecutive modules
    assert got0 == [(0, 1, 2)]


# ---------------------------------------------------------------- O-8 seeding and O-6(B) flags
@pytest.mark.parametrize("top", [13, 14])
def test_flagged_hit_is_not_a_seed_centre_and_same_step_flags_count(top):
    ev, want = T.pin_seed_flagged_centre(top)
    got, r = tracks_of(ev)
    assert got == want
    assert r["n_candidates"] == 1                            # the strays never seed


@pytest.mark.parametrize("top", [13, 14])
def test_flagged_hit_is_not_used_as_h0(top):
    ev, want = T.pin_seed_flagged_h0(top)
    got, r = tracks_of(ev)
    assert got == want
    assert r["n_candidates"] == 2
    c = oracle.event_candidates(*ev, 26)
    orig = [tuple(int(c["perm"][h]) for h in c["hits"][t, :c["n"][t]]) for t in range(c["n_cand"])]
    assert sorted(orig) == want                              # no candidate starts on the flagged hit 2


@pytest.mark.parametrize("top", [13, 14])
def test_flagged_hit_is_not_used_as_h2(top):
    ev, want = T.pin_seed_flagged_h2(top)
    got, r = tracks_of(ev)
    assert got == want
    assert r["n_candidates"] == 1


# ---------------------------------------------------------------- O-12 chi2 / ndof cut
@pytest.mark.parametrize("n", [3, 5])
def test_chi2_cut_both_sides_and_equality(n):
    ev, want, chi2 = T.pin_chi2_track(n)
    ndof = 2 * n - 4
    got, r = tracks_of(ev)
    assert got == want
    chi2_32 = np.float32(r["states"][11, 0])
    assert abs(float(chi2_32) - chi2) < 2e-3 * chi2          # closed form: residual sum of squares / sigma^2
    P = oracle.default_params()
    P.max_chi2_ndof = float(np.float32(chi2 / ndof * 1.04))  # just above chi2/ndof: kept
    assert tracks_of(ev, P)[0] == want
    P.max_chi2_ndof = float(np.float32(chi2 / ndof * 0.96))  # just below: dropped
    assert tracks_of(ev, P)[0] == []
    # ndof = 2n - 4, not 2n - 3: a cut between chi2/(2n-3) and chi2/(2n-4) drops the track
    P.max_chi2_ndof = float(np.float32(chi2 / (ndof + 0.5)))
    assert tracks_of(ev, P)[0] == []
    # equality keeps the track (O-12 drops on chi2 > max * ndof): choose max so that max * ndof
    # reproduces the track's own chi2 bit for bit
    m = np.float32(chi2_32 / np.float32(ndof))
    for cand in (m, np.nextafter(m, np.float32(0)), np.nextafter(m, np.float32(1e9))):
        if np.float32(cand) * np.float32(ndof) == chi2_32:
            P.max_chi2_ndof = float(cand)
            assert tracks_of(ev, P)[0] == want
            break
    else:
        pytest.fail("no float32 threshold reproduces chi2 exactly")


# ---------------------------------------------------------------- A11 degenerate slope threshold
def test_fit_small_but_not_degenerate_slope():
    hz = np.array([126, 101, 76, 51], np.float32)
    # s2 = 1e-8 >= 1e-12: the closest approach is computed, z = -x0/tx = -10000 mm, far from z-bar
    o = oracle.fit((1.0 + 1e-4 * hz.astype(np.float64)).astype(np.float32), np.zeros(4, np.float32), hz, SIGMA)
    assert abs(o[2] - 1e-4) < 2e-7 and abs(o[4] + 10000.0) < 30.0 and abs(o[0]) < 3e-3
    # s2 = 4e-14 < 1e-12: z = z-bar exactly, x = x-bar
    o = oracle.fit((1.0 + 2e-7 * hz.astype(np.float64)).astype(np.float32), np.zeros(4, np.float32), hz, SIGMA)
    assert o[4] == 88.5 and o[6] == 0.0


# ---------------------------------------------------------------- O-13 clone rule on real pairs
def _cands(ev):
    c = oracle.event_candidates(*ev, 26)
    return c, [tuple(int(c["perm"][h]) for h in c["hits"][t, :c["n"][t]]) for t in range(c["n_cand"])]


def test_clone_pair_sharing_three_of_four_hits():
    ev, want = T.pin_clone_pair()
    c, orig = _cands(ev)
    assert sorted(orig) == [(0, 1, 2, 3), (0, 4, 2, 3)]      # two 4-hit candidates, three hits shared
    a, b = orig.index((0, 1, 2, 3)), orig.index((0, 4, 2, 3))
    assert c["pass"][a] and c["pass"][b]
    assert c["states"][a, 11] < c["states"][b, 11]           # the straight one has the lower chi2
    assert c["survive"][a] and not c["survive"][b]
    assert c["lost"][a] == 0 and c["lost"][b] == 3           # 3 * 3 > 4 * 1
    assert tracks_of(ev)[0] == want


def test_clone_pair_equal_chi2_goes_to_the_lower_centre_index():
    ev, want = T.pin_clone_tie()
    c, orig = _cands(ev)
    assert sorted(orig) == [(0, 1, 3, 4), (0, 2, 3, 4)]
    a, b = orig.index((0, 2, 3, 4)), orig.index((0, 1, 3, 4))
    assert c["states"][a, 11:12].view(np.uint32)[0] == c["states"][b, 11:12].view(np.uint32)[0]   # chi2 bits equal
    assert c["centre"][a] < c["centre"][b]                   # y < 0 sorts first (lower phi16)
    assert c["survive"][a] and not c["survive"][b]
    assert tracks_of(ev)[0] == want
