"""Host-side logic of bench.py that does not need a GPU: the algorithmic-byte table of
SURVEY.md §8(d) and the max-over-ranks timing rule on a world_size-2 gloo group."""
import os
import sys

import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_algorithmic_bytes_match_survey_table():
    import bench
    B = bench.algorithmic_bytes(4096, 5_000_000, 8)
    assert B["row_pass"] == 4096 * 4096 * 8 + 4096 * 2049 * 16
    assert B["col_pass"] == 2 * 4096 * 2049 * 16
    assert B["sample"] == 200_000_000
    assert abs(B["step"] / 1e6 - 737.1) < 0.5            # 537.1 MB of FFT passes + 200 MB
    S = bench.algorithmic_bytes(4096, 5_000_000, 8, "sampleImage")
    assert S["sample"] == 160_000_000
    F = bench.algorithmic_bytes(4096, 5_000_000, 4)
    assert F["step"] * 2 == B["step"]
    # a pruned call, the METHOD's bytes: only columns 0..kumax are written and transformed, only rows
    # kvs_min..kvs_max written back, once; what the implementation moves on top (u, v read again by the extent
    # kernel, values stored twice in the column-pair layout) is not credited
    P = bench.algorithmic_bytes(4096, 5_000_000, 8, extent=(505, 1590, 2282))
    assert P["uv_extent"] == 0
    assert P["row_pass"] == 4096 * 4096 * 8 + 506 * 4096 * 16
    assert P["col_pass"] == 506 * 4096 * 16 + 506 * 693 * 16
    assert P["step"] < B["step"] and P["sample"] == B["sample"]
    assert abs(P["step"] / 1e6 - 406.1) < 0.5
    whole = bench.algorithmic_bytes(4096, 5_000_000, 8, extent=(2048, 0, 4095))
    assert whole == B
    # profile entries read no image; the batch counts C channels
    Pr = bench.algorithmic_bytes(1024, 200_000, 8, "chi2Profile")
    assert Pr["row_pass"] == 1024 * 513 * 16 and abs(Pr["step"] / 1e6 - 33.2) < 0.5
    C4 = bench.algorithmic_bytes(1024, 200_000, 8, "chi2ImageBatch", None, 128)
    assert abs(C4["step"] / 1e9 - 5.33) < 0.01            # 128 x (8.4 image + 3 x 8.4 spectrum + 8.0 per-point) MB


def _worker(rank, world, port, q):
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)
    q.put((rank, ms))
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 1000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == {0: 15.0, 1: 15.0}


def test_max_over_ranks_single():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
