"""Multi-process plumbing of the bench (N > 1): one process per GPU, each searching its own beams,
no data-path collective.  Covered here on CPU with
the gloo backend and world_size 2: the beam partition is exact and the ranks agree on
(max over ranks of the time, sum over ranks of the units) -- the only two numbers they exchange.
"""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

from paper_1811_04165_b200.shard import beam_seed, beams_of_rank, combine, dm_rows_of_rank, gather_rows  # noqa: E402


def test_beam_partition_is_exact_and_balanced():
    for world in (1, 2, 3, 4, 8):
        for n in (0, 1, 7, 8, 9, 64):
            owned = [beams_of_rank(n, r, world) for r in range(world)]
            flat = [b for o in owned for b in o]
            assert flat == list(range(n))                      # every beam exactly once, in order
            sizes = [len(o) for o in owned]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        beams_of_rank(4, 2, 2)
    assert beam_seed(100, 0) == 100 and len({beam_seed(100, b) for b in range(8)}) == 8


def test_dm_row_partition_is_exact_contiguous_and_block_aligned():
    for world in (1, 2, 3, 8):
        for ndm, mult in ((2048, 1), (2048, 32), (37, 1), (96, 8), (0, 1)):
            r = [dm_rows_of_rank(ndm, k, world, mult) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == ndm
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))      # contiguous, every row exactly once
            assert all(lo % mult == 0 and hi % mult == 0 for lo, hi in r)
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= mult
    with pytest.raises(ValueError):
        dm_rows_of_rank(10, 0, 2, 4)
    t = torch.arange(6.0).reshape(3, 2)
    assert gather_rows(t, 3) is t                                          # no process group: identity


def test_plans_of_a_dm_sharded_search_tile_the_one_gpu_plan():
    """plan_for_rank: the delay tables of the ranks' plans, stacked, are the one-GPU plan's tables (direct: rows of
    the delay table; subband: coarse rows of the step-1 table, one shared step-2 table), and every rank needs no
    more input than the whole search."""
    import numpy as np
    import paper_1811_04165_b200 as ddp
    from paper_1811_04165_b200.shard import plan_for_rank
    from synth import configs
    from synth.configs import SubbandPlan
    direct = configs.scaled(configs.apertif_direct(), name="shard_d", nchan=64, nsamp_out=2000, ndm=37, widths=(1, 2, 4))
    sub = configs.scaled(configs.apertif_direct(), name="shard_s", nchan=96, nsamp_out=2000, ndm=7 * 5, widths=(1, 2, 4),
                         subband=SubbandPlan(n_subbands=8, n_coarse=7, coarse_first=0.0, coarse_step=8.0, n_fine=5,
                                             fine_step=0.25))
    for cfg in (direct, sub):
        whole = ddp.plan_from_config(cfg, cache_dir=None)
        wi = whole.query()
        for world in (1, 2, 3, 8):
            tabs, covered = [], 0
            for r in range(world):
                plan, lo, hi = plan_for_rank(cfg, r, world, cache_dir=None)
                assert lo == covered
                covered = hi
                if plan is None:
                    assert lo == hi
                    continue
                i = plan.query()
                assert i.ndm == hi - lo and i.nsamp_in_required <= wi.nsamp_in_required
                if cfg.subband is None:
                    tabs.append(plan.get_delays(0))
                else:
                    tabs.append(plan.get_delays(1))
                    assert np.array_equal(plan.get_delays(2), whole.get_delays(2))
                plan.destroy()
            assert covered == cfg.ndm
            assert np.array_equal(np.concatenate(tabs, axis=0), whole.get_delays(0 if cfg.subband is None else 1))
        whole.destroy()


def test_combine_without_process_group_is_identity():
    assert combine(3.5, 7.0) == (3.5, 7.0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        beams = beams_of_rank(world, rank, world)             # bench: one beam per rank (weak scaling)
        local_ms = 10.0 + 5.0 * rank                          # rank 1 is the slower one
        local_units = 1000.0 * len(beams)
        ms, units = combine(local_ms, local_units, torch.device("cpu"))
        # a DM-sharded search: 5 rows x 3 widths split 3 + 2; row i of the whole table holds i*10 + width index
        lo, hi = dm_rows_of_rank(5, rank, world)
        mine = torch.tensor([[10.0 * i + k for k in range(3)] for i in range(lo, hi)], dtype=torch.float32)
        table = gather_rows(mine, 5)
        dist.barrier()
        out[rank] = (beams, ms, units, table.tolist())
    finally:
        dist.destroy_process_group()


def test_world_size_two_gloo_agrees_on_max_time_and_summed_units():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert out[0][0] == [0] and out[1][0] == [1]
    for r in range(world):
        _, ms, units, table = out[r]
        assert ms == 15.0                                     # max over ranks, never wall clock of rank 0
        assert units == 2000.0                                # whole-job units
        assert table == [[10.0 * i + k for k in range(3)] for i in range(5)]   # every rank holds the whole table
