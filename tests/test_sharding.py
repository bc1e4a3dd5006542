"""The N > 1 path on CPU: two `gloo` ranks reconstruct disjoint event ranges (the
oracle stands in for the per-rank engine: the host logic under test is the partition, the
all-gather of counts and the renumbering), and the stitched result equals the one-process result."""
import os
import socket
import tempfile

import numpy as np
import pytest

from paper_2412_05041_b200 import datagen, sharding

M = 26


def test_event_ranges_partition_the_batch():
    for n in (0, 1, 7, 100, 100001):
        for world in (1, 2, 3, 8):
            r = [sharding.event_range(k, world, n) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
    assert sharding.weak_event_range(3, 25000) == (75000, 100000)
    with pytest.raises(ValueError):
        sharding.event_range(2, 2, 10)


def test_slice_events_rebases_offsets():
    d = datagen.generate_config(0, n_events=12)
    s = sharding.slice_events(d, 5, 9)
    off = d["event_offsets"].astype(np.int64)
    assert s["n_events"] == 4 and s["event_offsets"][0] == 0 and s["first_hit"] == off[5]
    np.testing.assert_array_equal(s["event_offsets"], (off[5:10] - off[5]).astype(np.uint32))
    np.testing.assert_array_equal(s["x"], d["x"][off[5]:off[9]])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_events, outdir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        d = datagen.generate_config(0, n_events=n_events)
        e0, e1 = sharding.event_range(rank, world, n_events)
        sl = sharding.slice_events(d, e0, e1)
        res = oracle.reconstruct(sl["x"], sl["y"], sl["z"], sl["module"], sl["event_offsets"], M)
        bases = sharding.global_bases(res["n_tracks"], res["n_track_hits"])
        g = sharding.to_global(res, sl, bases)
        np.savez(os.path.join(outdir, f"rank{rank}.npz"), eto=g["event_track_offsets"], tho=g["track_hit_offsets"],
                 th=g["track_hits"], st=res["states"], bases=np.array([bases[k] for k in (
                     "track_base", "track_hit_base", "total_tracks", "total_track_hits")]))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_equal_one_process():
    import torch.multiprocessing as mp
    import oracle
    n_events, world = 30, 2
    with tempfile.TemporaryDirectory() as tmp:
        mp.spawn(_worker, args=(world, _free_port(), n_events, tmp), nprocs=world, join=True)
        parts = [np.load(os.path.join(tmp, f"rank{r}.npz")) for r in range(world)]
    d = datagen.generate_config(0, n_events=n_events)
    want = oracle.reconstruct(d["x"], d["y"], d["z"], d["module"], d["event_offsets"], M)
    assert int(parts[0]["bases"][2]) == want["n_tracks"] and int(parts[1]["bases"][3]) == want["n_track_hits"]
    assert int(parts[0]["bases"][0]) == 0 and int(parts[1]["bases"][0]) == int(parts[0]["eto"][-1])
    eto = np.concatenate([parts[0]["eto"], parts[1]["eto"][1:]])
    tho = np.concatenate([parts[0]["tho"], parts[1]["tho"][1:]])
    th = np.concatenate([parts[0]["th"], parts[1]["th"]])
    st = np.concatenate([parts[0]["st"], parts[1]["st"]], axis=1)
    np.testing.assert_array_equal(eto, want["event_track_offsets"])
    np.testing.assert_array_equal(tho, want["track_hit_offsets"])
    np.testing.assert_array_equal(th, want["track_hits"])
    np.testing.assert_array_equal(st.view(np.uint32), want["states"].view(np.uint32))
