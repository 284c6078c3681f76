"""Host logic of the T-slab sharded path (paper_1412_1498_b200/sharded.py) on CPU ranks:
the product's schedule and transport (torch.distributed, gloo, world_size 2) drive slabs whose arithmetic is the
oracle's; the assembled lattice must equal the oracle's sweep of the whole lattice."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _run_sharded(dims, n_slabs, gauge, storage, omega, sweeps, rough, seed, reunit_every=0):
    """On the calling rank (or alone): returns ({slab: links}, (F, theta), fixer counters)."""
    import gf_inputs as gi
    from _slab_oracle import OracleSlabEngine
    from paper_1412_1498_b200.sharded import ShardedGaugeFixer

    U = gi.make_links(dims, rough, seed, dtype=np.float64)
    sh = ShardedGaugeFixer(dims, n_slabs, device=None,
                           engine_factory=lambda ld, s: OracleSlabEngine(ld, s, gauge, storage))
    sh.set_reunit_every(reunit_every)
    sh.set_links_global(torch.from_numpy(U))
    sh.ovr_sweep(sweeps, omega)
    links = {s: t.numpy() for s, t in sh.get_links().items()}
    return links, sh.measure(), (sh.messages_sent, sh.copies)


def _expected(dims, gauge, storage, omega, sweeps, rough, seed, reunit_every=0):
    import gf_inputs as gi
    import oracle

    U = gi.make_links(dims, rough, seed, dtype=np.float64)
    if storage == 12:
        oracle.project12(U, dims)
    oracle.sweeps(U, dims, gauge, omega, n=sweeps, storage=storage, reunit_every=reunit_every)
    return U, oracle.measure(U, dims, gauge)


def _worker(rank, world, port, case, out):
    os.environ["OMP_NUM_THREADS"] = "1"
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    links, meas, counters = _run_sharded(*case)
    out[rank] = (links, meas, counters)
    dist.barrier()
    dist.destroy_process_group()


CASES = [  # dims, n_slabs, gauge, storage, omega, sweeps, roughness, seed, reunit_every
    ((4, 4, 4, 8), 2, "landau", 18, 1.7, 2, 0.4, 11, 0),   # one slab per rank: both neighbours are the same peer
    ((4, 4, 4, 8), 4, "landau", 12, 1.8, 2, 0.5, 12, 0),   # two slabs per rank (copy + send), lt = 2: border only
    ((4, 2, 4, 12), 2, "coulomb", 18, 1.7, 2, 0.5, 13, 1),  # Coulomb, lt = 6, reunitarisation + ghost refresh
]


@pytest.mark.parametrize("case", CASES)
def test_sharded_schedule_world2_equals_whole_lattice_oracle(case):
    dims, n_slabs, gauge, storage, omega, sweeps, rough, seed, reunit = case
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, _free_port(), case, out), nprocs=2, join=True)
        res = dict(out)
    Uexp, (Fexp, thexp) = _expected(dims, gauge, storage, omega, sweeps, rough, seed, reunit)
    V = int(np.prod(dims)) // n_slabs
    seen = set()
    for rank in (0, 1):
        links, (F, th), (sent, copies) = res[rank]
        assert sorted(links) == list(range(rank * n_slabs // 2, (rank + 1) * n_slabs // 2))
        for s, L in links.items():
            seen.add(s)
            assert np.array_equal(L.reshape(-1), Uexp[s * V:(s + 1) * V].reshape(-1)), f"slab {s} differs"
        assert abs(F - Fexp) <= 1e-13 * abs(Fexp) and abs(th - thexp) <= 1e-11 * thexp
        assert sent > 0
        assert (copies > 0) == (n_slabs > 2)
    assert seen == set(range(n_slabs))
    assert res[0][1] == res[1][1]  # every rank holds the same F, theta (same stop decision)


@pytest.mark.parametrize("n_slabs", [1, 2, 3])
def test_sharded_schedule_single_process(n_slabs):
    dims = (4, 4, 2, 12)
    links, (F, th), (sent, copies) = _run_sharded(dims, n_slabs, "landau", 18, 1.75, 2, 0.5, 21)
    Uexp, (Fexp, thexp) = _expected(dims, "landau", 18, 1.75, 2, 0.5, 21)
    got = np.concatenate([links[s].reshape(-1) for s in range(n_slabs)])
    assert np.array_equal(got, Uexp.reshape(-1))
    assert abs(F - Fexp) <= 1e-13 * abs(Fexp) and abs(th - thexp) <= 1e-11 * thexp
    assert sent == 0 and copies > 0


def test_send_and_receive_order_agree_between_every_pair_of_ranks():
    """A tag-less transport (NCCL) matches the k-th send A -> B with the k-th receive B posts from A."""
    from paper_1412_1498_b200.sharded import halo_messages, local_slabs, slab_owner

    for n_slabs, world in [(1, 1), (2, 1), (2, 2), (4, 2), (6, 2), (3, 3), (6, 3), (8, 4), (8, 8), (16, 8)]:
        sends, recvs = {}, {}
        for rank in range(world):
            mine = local_slabs(rank, n_slabs, world)
            for kind, src, dst in halo_messages(0, mine, n_slabs):
                a, b = slab_owner(src, n_slabs, world), slab_owner(dst, n_slabs, world)
                if a == b:
                    assert a == rank  # a local copy is seen by its owner only
                    continue
                if a == rank:
                    sends.setdefault((a, b), []).append((kind, src, dst))
                if b == rank:
                    recvs.setdefault((a, b), []).append((kind, src, dst))
        assert sends == recvs, (n_slabs, world)
        n_remote = sum(len(v) for v in sends.values())
        assert n_remote == (0 if world == 1 else 2 * world)  # one "ret" and one "fwd" across every rank boundary


def test_bad_partitions_are_rejected():
    from paper_1412_1498_b200.sharded import ShardedGaugeFixer

    for dims, n in [((4, 4, 4, 8), 3), ((4, 4, 4, 6), 2), ((4, 4, 4, 8), 8), ((4, 4, 4, 8), 0)]:
        with pytest.raises(ValueError):
            ShardedGaugeFixer(dims, n, device=None, engine_factory=lambda ld, s: None)
