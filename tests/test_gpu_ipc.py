"""NEXT-1 (g(Re,Rp) split by Rp over ranks) ACROSS A PROCESS BOUNDARY.

Two processes on cuda:0, each with one Rp-shard handle.  Every process owns the g(Re,q) buffers of its q-points, exports
them with CUDA IPC (torch's CUDA tensor pickling: cudaIpcGetMemHandle in the owner, cudaIpcOpenMemHandle in the peer) and
fills the destination table of epw_interp_rp_to_q_scatter_add with its own pointers and the MAPPED FOREIGN pointers of the
peer -- what the table holds on a multi-GPU node, where the mapping goes over NVLink instead of staying on one device.
Every process adds its partial sums into both owners' buffers; after a host-side barrier each owner checks its summed
g(Re,q) against the oracle's Eq. 9 and runs the rest of the path on it.  No kernel waits on another kernel (the processes
meet at host barriers only), so the two contexts may time-slice the GPU in any order.
"""
import os
import sys
import traceback

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

WORLD = 2
TIMEOUT_S = 240


def _workload():
    import synth

    # 12 q: S1 batches of 8 and 4 -> the bulk-TMA kernel (NQ = 8) and the register-staged one (NQ = 4)
    return synth.make_custom("si-ipc", 8, 6, (2, 2, 2), 1.5, 0.1, 1.5, (6, 5, 4), ("random", 12, 3), seed=57)


def _rank_main(rank, send_q, recv_q, barrier, result_q):
    """One rank = one process = one CUDA context on cuda:0."""
    try:
        import torch

        sys.path.insert(0, os.path.join(ROOT, "tests"))
        import oracle
        import paper_2603_10295_b200 as epw
        import synth
        from paper_2603_10295_b200 import shard
        from parity import assert_path_close

        synth.build()
        oracle.build()
        torch.cuda.set_device(0)
        w = _workload()
        rows = w.nbnd * w.nbnd * w.nmodes * w.ne
        lo, hi = shard.rp_ranges(w.np_, WORLD)[rank]
        h = epw.EpwInterp(w.nbnd, w.nmodes, w.ne, w.np_)
        h.set_operators_from_host(w, rp_range=(lo, hi))
        mine = [iq for iq in range(w.nq) if iq % WORLD == rank]          # owner of q-point iq = rank iq % WORLD
        own = torch.zeros((len(mine), rows, 2), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        send_q.put(own)                 # CUDA IPC export of my buffer ...
        peer = recv_q.get(timeout=TIMEOUT_S)   # ... and the peer's buffer mapped into this process
        assert peer.is_cuda and peer.shape == (w.nq - len(mine), rows, 2)
        assert peer.data_ptr() != own.data_ptr()
        barrier.wait(TIMEOUT_S)         # both buffers are zeroed and mapped on both sides
        bufs = {rank: own, 1 - rank: peer}
        dst = [bufs[iq % WORLD][iq // WORLD] for iq in range(w.nq)]
        q_d = torch.from_numpy(w.q_list).cuda()
        epw.epw_interp_rp_to_q_scatter_add(h.h, q_d, w.nq, dst)
        epw.epw_interp_sync(h.h)
        barrier.wait(TIMEOUT_S)         # every rank's additions have landed in every owner's buffer
        g = w.g_full()
        got = own.cpu().numpy().view(np.complex128).reshape(len(mine), rows)
        g1_ref = np.stack([oracle.rp_to_q(g, w.Rp, w.w_p, w.q_list[iq]) for iq in mine]).reshape(len(mine), rows)
        err = float(np.abs(got - g1_ref).max() / np.abs(g1_ref).max())
        assert err <= 1e-13, f"rank {rank}: summed g(Re,q) off by {err:.3e}"
        # the rest of the path on my q-points, from the summed g(Re,q)
        q_mine = np.ascontiguousarray(w.q_list[mine])
        epw.epw_interp_set_gq(h.h, own)
        out = h.interpolate_grid(w.k_grid, torch.from_numpy(q_mine).cuda())
        epw.epw_interp_sync(h.h)
        epw.epw_interp_set_gq(h.h, None)
        ref = oracle.interpolate(w.H_R, w.D_R, g, w.Re, w.w_e, w.Rp, w.w_p, w.k_list, q_mine)
        worst = assert_path_close([t.cpu().numpy() for t in out], ref)
        barrier.wait(TIMEOUT_S)         # nobody unmaps or frees while the other still reads
        h.close()
        del peer, bufs, dst
        result_q.put(("ok", rank, err, float(worst)))
    except BaseException:  # noqa: BLE001 -- reported to the parent, which fails the test
        try:
            barrier.abort()
        except Exception:  # noqa: BLE001
            pass
        result_q.put(("fail", rank, traceback.format_exc(), 0.0))


def test_rp_sharded_scatter_add_across_two_processes_cuda_ipc():
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q01, q10, results = ctx.Queue(), ctx.Queue(), ctx.Queue()
    barrier = ctx.Barrier(WORLD)
    procs = [ctx.Process(target=_rank_main, args=(0, q01, q10, barrier, results)),
             ctx.Process(target=_rank_main, args=(1, q10, q01, barrier, results))]
    for p in procs:
        p.start()
    got = []
    try:
        for _ in procs:
            got.append(results.get(timeout=TIMEOUT_S + 60))
    finally:
        for p in procs:
            p.join(timeout=30)
            if p.is_alive():
                p.kill()   # the exact process this test started
    for status, rank, a, b in got:
        assert status == "ok", f"rank {rank} failed:\n{a}"
        print(f"rank {rank}: summed g(Re,q) rel. error {a:.2e}, worst |g|^2 deviation {b:.3f} x tolerance")
    assert sorted(r for _, r, _, _ in got) == [0, 1]
