"""Direct delivery of the halo messages between PROCESSES (missing 2(i)): two ranks share
the one GPU of the test box, each owns slabs of the lattice, the neighbours' halo workspaces are mapped with CUDA IPC
(gf_ipc_export / gf_ipc_open) and the border kernels store into them (gf_slab_set_peer_targets).  gloo is the control
plane (NCCL refuses two ranks on one device); no kernel waits on another process - the ranks meet in a host barrier
after a stream synchronisation.  The assembled links must be bit-identical to the single-context sweep."""
import os
import socket
import sys

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, case, out):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import gf_inputs as gi
    import paper_1412_1498_b200 as gf

    torch.cuda.set_device(0)
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    dims, n_slabs, gauge, prec, storage, sweeps, reunit, mode = case
    U = gi.make_links(dims, 0.5, 77, dtype=np.float32 if prec == "f32" else np.float64)
    sh = gf.ShardedGaugeFixer(dims, n_slabs, gauge=gauge, prec=prec, storage=storage, device="cuda:0", mode=mode)
    assert sh.mode == (mode or "flags"), "the CUDA-IPC mapping of the neighbours' workspaces was not made"
    sh.set_reunit_every(reunit)
    sh.set_links_global(torch.from_numpy(U).cuda())
    done, hist = sh.fix(1.7, 0.0, sweeps, 2)
    links = {s: t.cpu().numpy() for s, t in sh.get_links().items()}
    launches, sent = sh.kernel_launches(), sh.messages_sent
    sh.close()
    out[rank] = (links, hist, launches, sent)
    dist.barrier()
    dist.destroy_process_group()


# mode None = the default ("flags": neighbours ordered by stream-ordered flag writes / waits, the sweep is one libgf call);
# "ipc" = the same delivery with a barrier between the ranks per half-sweep
CASES = [((8, 8, 8, 8), 2, "landau", "f64", 18, 4, 0, None),    # one slab per rank: both neighbours are the other rank
         ((8, 6, 4, 8), 4, "coulomb", "f64", 12, 4, 3, None),   # two slabs per rank (local and remote neighbours), lt = 2, reunit
         ((6, 4, 4, 8), 2, "landau", "f32", 12, 3, 0, None),
         # 100 sweeps in 50 calls of gf_slab_group_sweep (F/theta every 2 sweeps), reunitarisation every 7: the arrival
         # counters, the entry signals and the ghost refresh over many epochs, between two CUDA contexts
         ((8, 8, 8, 8), 4, "landau", "f64", 18, 100, 7, None),
         ((32, 32, 32, 16), 2, "landau", "f32", 12, 100, 50, None),  # config 2's local volume per rank, 32^3 x 8
         ((8, 8, 8, 8), 2, "landau", "f64", 18, 4, 0, "ipc"),
         ((8, 6, 4, 8), 4, "coulomb", "f64", 12, 4, 3, "ipc")]


@pytest.mark.parametrize("case", CASES)
def test_ipc_direct_delivery_two_processes_bit_identical(case):
    import torch
    import torch.multiprocessing as mp

    import gf_inputs as gi
    import paper_1412_1498_b200 as gf

    dims, n_slabs, gauge, prec, storage, sweeps, reunit, mode = case
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, _free_port(), case, out), nprocs=2, join=True)
        res = {r: out[r] for r in (0, 1)}
    U = gi.make_links(dims, 0.5, 77, dtype=np.float32 if prec == "f32" else np.float64)
    fx = gf.GaugeFixer(dims, gauge=gauge, prec=prec, storage=storage)
    fx.set_links(torch.from_numpy(U).cuda())
    fx.set_reunit_every(reunit)
    done = fx.fix(1.7, 0.0, sweeps, 2)
    single = fx.get_links().cpu().numpy()
    hist = fx.history()
    fx.close()
    V = single.shape[0] // n_slabs
    seen = set()
    for r in (0, 1):
        links, h, launches, sent = res[r]
        assert sent == 0 and launches > 0  # no halo message went through torch.distributed
        for s, a in links.items():
            assert np.array_equal(a.reshape(-1), single[s * V:(s + 1) * V].reshape(-1)), f"slab {s} of rank {r}"
            seen.add(s)
        assert [x[0] for x in h] == [x[0] for x in hist]
        for (_, F, th), (_, Fs, ths) in zip(h, hist):
            assert abs(F - Fs) <= 1e-12 * abs(Fs) + (0 if prec == "f64" else 1e-6) and abs(th - ths) <= 1e-6 * ths
    assert seen == set(range(n_slabs))
    assert res[0][1] == res[1][1]  # every rank took its decisions from the same numbers
