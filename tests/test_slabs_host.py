"""Host-side logic of the z-slab decomposition on CPU: the exchange plan of paper_1809_00995_b200/slabs.py carried
out over gloo between two processes, checked against a single-rank oracle run.  (The kernels' side of the same rules is checked on
the GPU by tests/test_gpu_parity.py::test_slab_group_*.)"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_layout_and_plan_are_consistent():
    from paper_1809_00995_b200 import slabs
    for N, P in ((16, 1), (16, 2), (16, 4), (128, 8), (1024, 8)):
        lay = slabs.layout(N, P)
        assert [s.z_offset for s in lay] == [r * N // P for r in range(P)] and all(s.nz == N // P for s in lay)
        owned = sorted(z for s in lay for z in range(s.z_offset, s.z_offset + s.nz))
        assert owned == list(range(N))                                        # every plane exactly once
        plan = slabs.exchange_plan(N, P)
        assert len(plan) == 2 * P
        filled = {}
        for src, sp, dst, dp, fields in plan:
            zg = lay[src].z_offset + sp - 1                                  # the global plane that travels
            assert lay[dst].ghost_planes()[dp] == zg % N                     # ... is the one the ghost mirrors (periodic wrap included)
            assert set(slabs.FACE_FIELDS) <= set(fields)
            filled[(dst, dp)] = fields
        assert set(filled) == {(s.rank, g) for s in lay for g in s.ghost_planes()}          # every ghost filled once
        assert all((slabs.GAUSS_FIELD in f) == (dp == 0) for (dst, dp), f in filled.items())  # eps_2 only into the ghost below
    with pytest.raises(ValueError):
        slabs.layout(16, 3)
    assert [slabs.owner(r, 4, 2) for r in range(4)] == [0, 0, 1, 1]


def _worker(rank, world, port, N, P, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from oracle import ahs_oracle as O
    from paper_1809_00995_b200 import slabs
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        import torch
        p = O.Params(N=N, m=1.0, s=0.0)
        full = O.initial_condition(p, 5)
        O.step(p, full, 0, 3)                                                # the single-rank oracle run both processes can afford
        lay = slabs.layout(N, P)
        mine = [s for s in lay if slabs.owner(s.rank, P, world) == rank]
        ok = True
        for nstep in (3, 4):
            # my slabs: own planes from the snapshot, ghosts poisoned
            local = {}
            for s in mine:
                a = np.full((10, s.nz_alloc, N, N), np.nan)
                a[:, 1:s.nz + 1] = full[:, s.z_offset:s.z_offset + s.nz]
                local[s.rank] = a
            for src, sp, dst, dp, fields in slabs.exchange_plan(N, P):       # the same order on every rank: no deadlock
                so, do = slabs.owner(src, P, world), slabs.owner(dst, P, world)
                idx = list(fields)
                if so == rank and do == rank:
                    local[dst][idx, dp] = local[src][idx, sp]
                elif so == rank:
                    dist.send(torch.from_numpy(np.ascontiguousarray(local[src][idx, sp])), dst=do)
                elif do == rank:
                    buf = torch.empty((len(idx), N, N), dtype=torch.float64)
                    dist.recv(buf, src=so)
                    local[dst][idx, dp] = buf.numpy()
            for s in mine:                                                   # ghosts against the oracle's planes
                for g, zg in s.ghost_planes().items():
                    want = list(slabs.FACE_FIELDS) + ([slabs.GAUSS_FIELD] if g == 0 else [])
                    ok = ok and np.array_equal(local[s.rank][want, g], full[want, zg])
                    rest = [k for k in range(10) if k not in want]
                    ok = ok and bool(np.isnan(local[s.rank][rest, g]).all())  # nothing else travels
            O.step(p, full, nstep, 1)                                        # next step of the single-rank run, exchange again
        t = torch.tensor([1.0 if ok else 0.0])
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
        if rank == 0:
            out.put(float(t.item()))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("P", [2, 4])
def test_exchange_plan_over_gloo_matches_a_single_rank_oracle_run(P):
    import torch.multiprocessing as mp
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 16, P, out)) for r in range(2)]
    for pr in procs:
        pr.start()
    for pr in procs:
        pr.join(timeout=240)
        assert pr.exitcode == 0
    assert out.get(timeout=5) == 1.0
