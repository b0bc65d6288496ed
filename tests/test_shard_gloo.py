"""Multi-rank host logic: q-sharding over ranks with no data-path collective, checked with
world_size-2 `gloo` process groups on CPU.  The per-rank worker here is the CPU oracle (there is no GPU on this box and
the product has no CPU fallback): what is under test is the sharding / gathering / timing plumbing of
paper_2603_10295_b200/shard.py that bench.py and a multi-GPU caller use, not the kernels."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2603_10295_b200 import shard  # noqa: E402


def test_q_ranges_partition():
    for nq in (0, 1, 7, 8, 64, 1000):
        for world in (1, 2, 3, 8):
            r = shard.q_ranges(nq, world)
            assert len(r) == world and r[0][0] == 0 and r[-1][1] == nq
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.q_ranges(4, 0)


def test_q_block_disjoint_within_a_step_and_covers_the_list():
    nq, nq_step, world = 1000, 8, 4
    seen = []
    for step in range(nq // (nq_step * world) + 1):
        blocks = [shard.q_block(step, world, r, nq_step, nq) for r in range(world)]
        flat = np.concatenate(blocks)
        assert len(set(flat.tolist())) == len(flat)  # ranks of one step own disjoint q
        seen.append(flat)
    assert set(np.concatenate(seen).tolist()) == set(range(nq))  # the walk covers every q
    # world = 1 degenerates to consecutive blocks
    assert shard.q_block(3, 1, 0, 8, 1000).tolist() == list(range(24, 32))
    with pytest.raises(ValueError):
        shard.q_block(0, 2, 2, 8, 100)


def test_rp_ranges():
    assert shard.rp_ranges(17, 2) == [(0, 9), (9, 17)]
    assert shard.rp_ranges(343, 8)[-1][1] == 343


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, tmpdir: str):
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle
    import synth

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "1"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.make_custom("shard-test", 3, 3, (1, 1, 0), 1.0, 0.1, 1.0, (3, 2, 1), ("random", 5, 2), seed=11)
        g = w.g_full()
        ranges = shard.q_ranges(w.nq, world)
        a, b = ranges[rank]
        eps_k, eps_kq, omega, g2 = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list[a:b])
        # no collective inside the path; afterwards the caller may gather the small per-q table and its |g|^2 slices
        omega_all = shard.all_gather_rows(torch.from_numpy(omega), ranges, dist)
        g2_all = shard.all_gather_rows(torch.from_numpy(g2), ranges, dist)
        epskq_all = shard.all_gather_rows(torch.from_numpy(eps_kq), ranges, dist)
        t = shard.max_over_ranks_ms(10.0 + rank, dist)
        assert t == 10.0 + world - 1
        if rank == 0:
            ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)
            np.testing.assert_array_equal(omega_all.numpy(), ref[2])
            np.testing.assert_array_equal(g2_all.numpy(), ref[3])
            np.testing.assert_array_equal(epskq_all.numpy(), ref[1])
            np.testing.assert_array_equal(eps_k, ref[0])
            open(os.path.join(tmpdir, "ok"), "w").write("ok")
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_q_sharded_run_world2_gloo(tmp_path):
    """Two ranks interpolate disjoint q ranges of one workload and gather: identical to the single-rank result,
    bit for bit (outputs are per-q, nothing is reduced across ranks)."""
    import torch.multiprocessing as mp

    port = _free_port()
    mp.spawn(_worker, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok").exists()


def _worker_rp(rank: int, world: int, port: int, tmpdir: str):
    """Rp-sharded variant: partial Eq. 9 per rank, all-reduce(SUM) of g(Re,q), then each rank
    interpolates its share of the k-points.  Worker = the oracle; under test: rp_ranges / k_ranges / the collective."""
    import torch
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import oracle
    import synth

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "1"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.make_custom("rp-shard", 2, 3, (1, 1, 0), 1.0, 0.1, 1.0, (3, 2, 1), ("random", 2, 2), seed=12)
        g = w.g_full()
        a, b = shard.rp_ranges(w.np_, world)[rank]
        ka, kb = shard.k_ranges(w.nk, world)[rank]
        g2_local = []
        for q in w.q_list:
            part = oracle.rp_to_q(g[a:b], w.Rp[a:b], w.w_p[a:b], q)           # this rank's slabs only
            t = torch.from_numpy(part.view(np.float64).copy())
            dist.all_reduce(t, op=dist.ReduceOp.SUM)                          # the one exchange step of the path
            g1 = t.numpy().view(np.complex128).reshape(part.shape)
            e_cm, om = oracle.phonon(w.D_R, w.Rp, w.w_p, q)
            g2_local.append(np.stack([oracle.pair(g1, w.H_R, w.Re, w.w_e, e_cm, om, k, q)[0] for k in w.k_list[ka:kb]]))
        g2_local = torch.from_numpy(np.stack(g2_local, axis=1))               # [nk_local][nq]...
        g2_all = shard.all_gather_rows(g2_local, shard.k_ranges(w.nk, world), dist)
        if rank == 0:
            ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, w.q_list)[3]
            got = np.swapaxes(g2_all.numpy(), 0, 1)
            assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
            open(os.path.join(tmpdir, "ok_rp"), "w").write("ok")
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_rp_sharded_run_world2_gloo(tmp_path):
    import torch.multiprocessing as mp

    port = _free_port()
    mp.spawn(_worker_rp, args=(2, port, str(tmp_path)), nprocs=2, join=True)
    assert (tmp_path / "ok_rp").exists()
