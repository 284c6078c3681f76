"""T-slab sharding of the overrelaxation sweep over several GPUs (include/gf.h "T-slab sharding").

The lattice nx*ny*nz*nt is cut along t into `n_slabs` slabs of lt = nt/n_slabs time slices (lt even).  Every slab is a
libgf context with a halo workspace attached; all arithmetic (border / interior half-sweeps, packing and scattering of
the top-slice temporal links, F and theta) runs in libgf's kernels.  This module is the plumbing between them: which
buffer goes to which neighbour and when, on which stream, over which transport

  * direct delivery (default on GPUs): the border kernel of a slab stores its two halo messages straight into the
    neighbours' workspaces - plain pointers for slabs of the same process (gf_slab_set_targets), CUDA-IPC mappings of the
    other ranks' workspaces between processes on one node (gf_ipc_export / gf_ipc_open, gf_slab_set_peer_targets), i.e.
    stores over NVLink from inside the update kernel; what is left per half-sweep is one ordering point between ranks
    (a one-element all-reduce queued on the streams with NCCL; stream synchronisation + barrier with gloo),
  * transport (direct=False, or where the mappings cannot be made): device-to-device copies between slabs of one
    process, torch.distributed send / recv between ranks,

and the driver loop of Algorithm 1 around it, whose decisions (stop test, sweeps to the next measurement, the global
F and theta from the slabs' values) are taken by libgf (gf_fix_plan, gf_combine_slabs); the one data-path collective is
an all-gather of each slab's F and theta.

Per half-sweep of parity p (include/gf.h steps 1-4), for every local slab s with lower neighbour s-1 and upper s+1:
    border(p)    -> ghost[1-p] updated in place, top_out = top-slice U_t of the parity-p sites
    interior(p)  -> overlaps with the transport, which runs on its own stream
    ghost[1-p] --"ret"--> top_in of slab s-1          top_out --"fwd"--> ghost[p] of slab s+1
    unpack_top(1-p)
"""
from __future__ import annotations

import contextlib

from . import binding as _b


# ---- one slab on a GPU ------------------------------------------------------------------------------------------------------
class GpuSlabEngine:
    """A libgf context on the local lattice (nx, ny, nz, lt) with its halo workspace.  Marshals arguments only."""

    def __init__(self, local_dims, gauge, prec, storage, device, stream=None):
        import torch

        self.torch = torch
        self.fx = _b.GaugeFixer(local_dims, gauge=gauge, prec=prec, storage=storage, device=device, stream=stream)
        self.device = self.fx.device
        self.stream = self.fx.stream
        B = _b.gf_slab_halo_bytes(self.fx.ctx)
        self.halo_bytes = B
        with torch.cuda.device(self.device), torch.cuda.stream(self.stream):  # tied to the stream its kernels run on
            # 4 halo buffers + the two synchronisation words of gf_slab_set_peer_flags (same allocation: one IPC handle)
            self.halo = torch.zeros(4 * B + 256, dtype=torch.uint8, device=self.device)
        self.flags_offset = 4 * B
        self.fx._check(_b.gf_slab_attach(self.fx.ctx, self.halo.data_ptr(), 4 * B))
        self.ghost = [self.halo[0:B], self.halo[B:2 * B]]
        self.top_out = self.halo[2 * B:3 * B]
        self.top_in = self.halo[3 * B:4 * B]

    def set_links(self, links):
        self.fx.set_links(links)

    def get_links(self, out=None):
        return self.fx.get_links(out)

    def set_targets(self, upper_ghost0, upper_ghost1, lower_top_in):
        """Device tensors of the neighbours' halo workspaces the border kernel stores into (None x 3: back to top_out)."""
        ptr = [t.data_ptr() if t is not None else 0 for t in (upper_ghost0, upper_ghost1, lower_top_in)]
        self.fx._check(_b.gf_slab_set_targets(self.fx.ctx, *ptr))

    def set_peer_targets(self, upper_base: int, lower_base: int):
        """Device addresses of the upper and lower neighbours' halo workspaces (own process or CUDA-IPC mappings)."""
        B = self.halo_bytes
        self.fx._check(_b.gf_slab_set_peer_targets(self.fx.ctx, upper_base, upper_base + B, lower_base + 3 * B,
                                                   lower_base + 2 * B))

    def set_peer_flags(self, upper_base: int, lower_base: int):
        """The neighbours' workspaces again: this slab signals into the upper one's "from below" word and the lower
        one's "from above" word (gf_slab_set_peer_flags)."""
        off = self.flags_offset
        self.fx._check(_b.gf_slab_set_peer_flags(self.fx.ctx, self.halo.data_ptr() + off, upper_base + off + 4, lower_base + off))

    def pack_top(self, parity):
        self.fx._check(_b.gf_slab_pack_top(self.fx.ctx, int(parity)))

    def unpack_top(self, parity):
        self.fx._check(_b.gf_slab_unpack_top(self.fx.ctx, int(parity)))

    def border(self, parity, omega):
        self.fx._check(_b.gf_slab_halfsweep_border(self.fx.ctx, int(parity), float(omega)))

    def interior(self, parity, omega):
        self.fx._check(_b.gf_slab_halfsweep_interior(self.fx.ctx, int(parity), float(omega)))

    def measure(self):
        return self.fx.measure()

    def reunitarize(self):
        self.fx.reunitarize()

    def kernel_launches(self):
        return self.fx.kernel_launches()

    # stream hand-offs between the compute stream of this slab and the process's transport stream
    def mark(self):
        ev = self.torch.cuda.Event()
        ev.record(self.stream)
        return ev

    def wait(self, event):
        if event is not None:
            self.stream.wait_event(event)

    def close(self):
        self.fx.close()


# ---- who owns which slab ---------------------------------------------------------------------------------------------------
def slab_owner(slab: int, n_slabs: int, world: int) -> int:
    """Slabs are dealt to the ranks in contiguous runs of n_slabs / world (neighbouring slabs on the same or the next GPU)."""
    return slab // (n_slabs // world)


def local_slabs(rank: int, n_slabs: int, world: int):
    k = n_slabs // world
    return list(range(rank * k, (rank + 1) * k))


def halo_messages(p: int, slabs, n_slabs: int):
    """The messages of one half-sweep of parity p that involve the given slabs, as (kind, src_slab, dst_slab):
    "ret": ghost[1-p] of src -> top_in of dst = src - 1;   "fwd": top_out of src -> ghost[p] of dst = src + 1.
    (p does not change who talks to whom, only which ghost buffer is meant.)"""
    out = []
    for s in slabs:
        out.append(("ret", s, (s - 1) % n_slabs))
        out.append(("fwd", s, (s + 1) % n_slabs))
        out.append(("ret", (s + 1) % n_slabs, s))
        out.append(("fwd", (s - 1) % n_slabs, s))
    # One global order (kind, destination) on every rank: between any two ranks the sends are posted in the order the
    # matching receives are, which is what a tag-less transport (NCCL) matches by.
    return sorted(set(out), key=lambda m: (m[0], m[2]))


def message_tag(kind: str, dst_slab: int) -> int:
    return 2 * dst_slab + (1 if kind == "fwd" else 0)


class ShardedGaugeFixer:
    """Overrelaxation gauge fixing of one lattice spread over n_slabs T-slabs.

    dims: the GLOBAL lattice (nx, ny, nz, nt).  With torch.distributed initialised every rank constructs the same object
    and owns n_slabs / world_size consecutive slabs; without it (or with group=False) all slabs live in this process.
    engine_factory(local_dims, slab_index) builds one slab (default: GpuSlabEngine on `device`).
    mode: how the halo messages travel and how neighbours are ordered.
      "flags" (default wherever the slabs are libgf contexts on GPUs): the border kernels store the messages straight into
        the neighbours' workspaces - plain pointers within a process, CUDA-IPC mappings between the processes of a node -
        and neighbours are ordered by stream-ordered flag writes / waits; ovr_sweep(n) is ONE libgf call
        (gf_slab_group_sweep): no Python, host wait or collective per half-sweep.  If the mappings cannot be made (e.g.
        an allocator with virtual-memory segments) a warning is issued and the transport is used.
      "ipc": the same delivery, ranks ordered by a one-element all-reduce (NCCL) or a barrier (gloo) per half-sweep.
      "events": all slabs in this process, delivery by plain pointers, kernels ordered by CUDA events (round 1).
      "transport": device copies within a process, torch.distributed send / recv between ranks.
    slab_streams: None = every local slab on the current stream; "own" = each local slab on a CUDA stream of its own, so
      that the kernels of neighbouring slabs of ONE process overlap on the device the way those of neighbouring ranks do
      and every ordering between them goes through the flags (what the multi-rank schedule is tested with on one GPU).
    direct (older spelling): True = "events" / "ipc", False = "transport".  (device=None with an engine_factory is the seam the CPU schedule test uses to
    drive this schedule with host-side slabs.)
    """

    def __init__(self, dims, n_slabs, gauge="landau", prec="f64", storage=18, device="cuda:0", group=None,
                 engine_factory=None, direct=None, mode=None, slab_streams=None):
        import torch

        self.torch = torch
        self.dims = tuple(int(d) for d in dims)
        self.n_slabs = int(n_slabs)
        nx, ny, nz, nt = self.dims
        if self.n_slabs < 1 or nt % self.n_slabs or (nt // self.n_slabs) % 2 or nt // self.n_slabs < 2:
            raise ValueError("nt must split into n_slabs slabs of an even number (>= 2) of time slices")
        self.local_dims = (nx, ny, nz, nt // self.n_slabs)
        self.local_volume = nx * ny * nz * (nt // self.n_slabs)
        self.dist = None
        self.group = None
        self.rank, self.world = 0, 1
        if group is not False:
            import torch.distributed as dist

            if dist.is_available() and dist.is_initialized():
                self.dist, self.group = dist, group
                self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        if self.n_slabs % self.world:
            raise ValueError("n_slabs must be a multiple of the number of ranks")
        self.slabs = local_slabs(self.rank, self.n_slabs, self.world)
        self.device = torch.device(device) if device is not None else torch.device("cpu")
        self.on_gpu = self.device.type == "cuda"
        if slab_streams not in (None, "own"):
            raise ValueError("slab_streams must be None or 'own'")
        self.own_streams = slab_streams == "own"
        if engine_factory is None:
            def engine_factory(local_dims, slab):
                stream = None
                if self.own_streams:
                    with torch.cuda.device(self.device):
                        stream = torch.cuda.Stream(self.device)
                return GpuSlabEngine(local_dims, gauge, prec, storage, self.device, stream=stream)
        self.engines = {s: engine_factory(self.local_dims, s) for s in self.slabs}
        self.comm_stream = None
        if self.on_gpu:
            with torch.cuda.device(self.device):
                self.comm_stream = torch.cuda.Stream(self.device)
        gpu_slabs = self.on_gpu and all(hasattr(e, "set_targets") for e in self.engines.values())
        if mode is None:
            if direct is None:
                mode = "flags" if gpu_slabs else "transport"
            elif direct:
                mode = "events" if self.world == 1 else "ipc"
            else:
                mode = "transport"
        if mode not in ("flags", "events", "ipc", "transport"):
            raise ValueError("mode must be flags, events, ipc or transport")
        if mode != "transport" and not gpu_slabs:
            raise ValueError("direct delivery needs libgf slabs on GPUs")
        if mode == "events" and self.world > 1:
            raise ValueError("mode 'events' orders kernels with CUDA events: all slabs must live in this process")
        self._ipc_mapped = {}
        if mode == "events":
            for s, e in self.engines.items():
                up, lo = self.engines[(s + 1) % self.n_slabs], self.engines[(s - 1) % self.n_slabs]
                e.set_targets(up.ghost[0], up.ghost[1], lo.top_in)
        elif mode in ("flags", "ipc"):
            if not self._map_neighbours(with_flags=mode == "flags"):
                import warnings

                warnings.warn("ShardedGaugeFixer: CUDA IPC mapping of the neighbours' halo workspaces failed; halo messages "
                              "go through torch.distributed send/recv")
                mode = "transport"
        self.mode = mode
        self.direct = mode == "events"   # in-process direct delivery, kernels ordered by CUDA events
        self.ipc = mode == "ipc"         # direct delivery between processes, ranks ordered by a collective / barrier
        self.flags = mode == "flags"     # direct delivery, neighbours ordered by stream-ordered flags; the sweep is one C call
        self._after_unpack = {}
        self.reunit_every = 0
        self.sweeps_total = 0
        self.messages_sent = 0  # remote (torch.distributed) messages posted by this rank
        self.copies = 0         # local device-to-device copies

    # ---- direct delivery between processes -----------------------------------------------------------------------------------
    def _map_neighbours(self, with_flags=False):
        """Exchange CUDA-IPC handles of every slab's halo workspace, map the ones of this rank's remote neighbours and
        give every local slab its two neighbours' addresses.  All ranks agree on the outcome."""
        torch, dist = self.torch, self.dist
        table = {}
        if self.world > 1:
            mine, ok = {}, True
            for s, e in self.engines.items():
                rc, handle, off = _b.gf_ipc_export(e.halo.data_ptr())
                ok = ok and rc == _b.GF_OK
                mine[s] = (handle, off)
            gathered = [None] * self.world
            dist.all_gather_object(gathered, (ok, mine), group=self.group)
            if not all(g[0] for g in gathered):
                return False
            for _, d in gathered:
                table.update(d)

        def base(slab):
            if slab in self.engines:
                return self.engines[slab].halo.data_ptr()
            handle, off = table[slab]
            if handle not in self._ipc_mapped:  # several slabs of a rank may sit in one allocation: map it once
                with torch.cuda.device(self.device):
                    rc, ptr = _b.gf_ipc_open(handle, 0)
                self._ipc_mapped[handle] = ptr if rc == _b.GF_OK else None
            return None if self._ipc_mapped[handle] is None else self._ipc_mapped[handle] + off

        bases = {s: (base((s + 1) % self.n_slabs), base((s - 1) % self.n_slabs)) for s in self.slabs}
        good = all(u is not None and l is not None for u, l in bases.values())
        if self.world > 1:
            agreed = [None] * self.world
            dist.all_gather_object(agreed, good, group=self.group)
            good = all(agreed)
        if not good:
            return False
        for s, (u, l) in bases.items():
            self.engines[s].set_peer_targets(u, l)
            if with_flags:
                self.engines[s].set_peer_flags(u, l)  # zeroes this slab's two words and synchronises its stream
        if self.world > 1:
            dist.barrier(group=self.group)  # every rank's words are zero before anybody signals
        self._token = torch.zeros(1, dtype=torch.float32, device=self.device)
        return True

    def _ctxs(self):
        return [self.engines[s].fx.ctx for s in self.slabs]

    def _rank_sync(self):
        """One ordering point between all ranks' streams: what every rank queued before it is complete before anything
        queued after it starts.  NCCL: a one-element all-reduce on the transport stream between the compute streams (no
        host wait); other backends: stream synchronisation and a barrier."""
        torch, dist = self.torch, self.dist
        if dist is None or self.world == 1:
            self.synchronize()
            return
        if dist.get_backend(self.group) == "nccl":
            for s in self.slabs:
                self.comm_stream.wait_event(self.engines[s].mark())
            with torch.cuda.stream(self.comm_stream):
                dist.all_reduce(self._token, group=self.group)
            done = torch.cuda.Event()
            done.record(self.comm_stream)
            for s in self.slabs:
                self.engines[s].wait(done)
        else:
            self.synchronize()
            dist.barrier(group=self.group)

    # ---- transport ------------------------------------------------------------------------------------------------------
    def _buffer(self, kind, end, slab, p):
        e = self.engines[slab]
        if kind == "ret":
            return e.ghost[1 - p] if end == "src" else e.top_in
        return e.top_out if end == "src" else e.ghost[p]

    def _exchange(self, p, kinds=("ret", "fwd"), after=None):
        """Move this half-sweep's messages on the transport stream.  `after`: events the transport waits for (default:
        everything queued so far on the local compute streams).  On return every local compute stream waits for the
        transport, so neither a source nor a destination buffer is touched by a later kernel before it is done."""
        torch = self.torch
        ctx = contextlib.nullcontext()
        if self.on_gpu:
            for ev in (after if after is not None else [self.engines[s].mark() for s in self.slabs]):
                self.comm_stream.wait_event(ev)
            ctx = torch.cuda.stream(self.comm_stream)
        with ctx:
            ops = []
            for kind, src, dst in halo_messages(p, self.slabs, self.n_slabs):
                if kind not in kinds:
                    continue
                src_local, dst_local = src in self.engines, dst in self.engines
                if src_local and dst_local:
                    self._buffer(kind, "dst", dst, p).copy_(self._buffer(kind, "src", src, p), non_blocking=True)
                    self.copies += 1
                elif src_local:
                    peer = self._global_rank(slab_owner(dst, self.n_slabs, self.world))
                    ops.append(self.dist.P2POp(self.dist.isend, self._buffer(kind, "src", src, p), peer, self.group,
                                               message_tag(kind, dst)))
                    self.messages_sent += 1
                elif dst_local:
                    peer = self._global_rank(slab_owner(src, self.n_slabs, self.world))
                    ops.append(self.dist.P2POp(self.dist.irecv, self._buffer(kind, "dst", dst, p), peer, self.group,
                                               message_tag(kind, dst)))
            if ops:
                for req in self.dist.batch_isend_irecv(ops):
                    req.wait()
        if self.on_gpu:
            done = torch.cuda.Event()
            done.record(self.comm_stream)
            for s in self.slabs:
                self.engines[s].wait(done)

    def _global_rank(self, group_rank):
        if self.group is None:
            return group_rank
        return self.dist.get_global_rank(self.group, group_rank)

    def _join_neighbours(self, events):
        """Direct delivery: slab s goes on once its two neighbours' kernels behind `events` are done."""
        for s in self.slabs:
            for nb in {(s - 1) % self.n_slabs, (s + 1) % self.n_slabs} - {s}:
                self.engines[s].wait(events.get(nb))

    def refresh_ghosts(self):
        """Fill both ghost buffers of every slab from its lower neighbour's top slice (after set_links, reunitarize)."""
        if self.flags:
            rc = _b.gf_slab_group_refresh(self._ctxs())
            if rc != _b.GF_OK:
                raise _b.GFError(rc, _b.gf_last_error(self._ctxs()[0]))
            return
        if self.direct:  # pack_top writes into the upper neighbour's ghost buffer: wait for whatever it still runs
            self._join_neighbours({s: self.engines[s].mark() for s in self.slabs})
        if self.ipc:
            self._rank_sync()
        for q in (0, 1):
            for s in self.slabs:
                self.engines[s].pack_top(q)
            if self.direct:
                self._join_neighbours({s: self.engines[s].mark() for s in self.slabs})
            elif not self.ipc:
                self._exchange(q, kinds=("fwd",))
        if self.ipc:
            self._rank_sync()

    # ---- links in / out ---------------------------------------------------------------------------------------------------
    def set_links(self, links_by_slab):
        """links_by_slab: {slab: canonical (V_local,4,3,3,2) tensor} for the local slabs."""
        if self.own_streams:  # the tensors were produced on the caller's stream, the slabs read them on theirs
            self.torch.cuda.current_stream(self.device).synchronize()
        for s in self.slabs:
            self.engines[s].set_links(links_by_slab[s])
        self.sweeps_total = 0
        self.refresh_ghosts()

    def set_links_global(self, links):
        """links: the canonical array of the WHOLE lattice (t is the slowest index, so a slab is a contiguous run of sites)."""
        V = self.local_volume
        self.set_links({s: links[s * V:(s + 1) * V].contiguous() for s in self.slabs})

    def get_links(self):
        out = {s: self.engines[s].get_links() for s in self.slabs}
        if self.own_streams:  # written on the slabs' streams, read by the caller on its own
            self.synchronize()
        return out

    # ---- Algorithm 1 ---------------------------------------------------------------------------------------------------------
    def half_sweep(self, p, omega):
        if self.direct:
            # the border kernels deliver: a slab's border kernel writes its neighbours' ghost[p] / top_in, so it starts
            # after their last unpack, and the unpack after the neighbours' border kernels
            self._join_neighbours(self._after_unpack)
            for s in self.slabs:
                self.engines[s].border(p, omega)
            after = {s: self.engines[s].mark() for s in self.slabs}
            for s in self.slabs:
                self.engines[s].interior(p, omega)
            self._join_neighbours(after)
            for s in self.slabs:
                self.engines[s].unpack_top(1 - p)
            self._after_unpack = {s: self.engines[s].mark() for s in self.slabs}
            return
        if self.ipc or self.flags:  # (flags: a single half-sweep outside ovr_sweep takes the host-ordered schedule)
            # Between processes: the border kernels store both messages in the neighbours' mapped workspaces (top_in is
            # double-buffered by parity, gf_slab_set_peer_targets), then ONE ordering point between the ranks; the next
            # border kernel only writes buffers whose last readers ran before it.
            for s in self.slabs:
                self.engines[s].border(p, omega)
            self._rank_sync()
            for s in self.slabs:
                self.engines[s].interior(p, omega)
            for s in self.slabs:
                self.engines[s].unpack_top(1 - p)
            return
        for s in self.slabs:
            self.engines[s].border(p, omega)
        # the transport starts as soon as the border kernels are done, beside the interior kernels queued behind them
        after = [self.engines[s].mark() for s in self.slabs] if self.on_gpu else None
        for s in self.slabs:
            self.engines[s].interior(p, omega)
        self._exchange(p, after=after)
        for s in self.slabs:
            self.engines[s].unpack_top(1 - p)

    def reunitarize(self):
        for s in self.slabs:
            self.engines[s].reunitarize()
        self.refresh_ghosts()

    def set_reunit_every(self, k):
        self.reunit_every = int(k)

    def ovr_sweep(self, n, omega):
        """n sweeps, even half-sweep first; reunitarisation cadence as gf_ovr_sweep."""
        if _b.gf_fix_plan(float(omega), 0.0, int(n), 1, 0, 1.0)[0] != _b.GF_OK:
            raise ValueError("omega outside [1,2) or n < 0")
        if self.flags:  # the whole schedule, reunitarisation cadence included, is one asynchronous libgf call
            rc = _b.gf_slab_group_sweep(self._ctxs(), int(n), float(omega), self.reunit_every, self.sweeps_total)
            if rc != _b.GF_OK:
                raise _b.GFError(rc, _b.gf_last_error(self._ctxs()[0]))
            self.sweeps_total += int(n)
            return
        for _ in range(int(n)):
            self.half_sweep(0, omega)
            self.half_sweep(1, omega)
            self.sweeps_total += 1
            if self.reunit_every > 0 and self.sweeps_total % self.reunit_every == 0:
                self.reunitarize()

    def measure(self):
        """Global F and theta: the mean over all slabs (equal volumes) of each slab's gf_measure, added in slab order on
        every rank, so all ranks take the same stop decision."""
        torch = self.torch
        local = torch.tensor([list(self.engines[s].measure()) for s in self.slabs], dtype=torch.float64)
        if self.world > 1:
            # gf_measure's results are host numbers; NCCL moves device memory only
            buf = local.to(self.device) if self.on_gpu else local
            parts = [torch.empty_like(buf) for _ in range(self.world)]
            self.dist.all_gather(parts, buf, group=self.group)
            local = torch.cat(parts).cpu()
        rows = local.tolist()
        rc, F, theta = _b.gf_combine_slabs([r[0] for r in rows], [r[1] for r in rows])
        if rc != _b.GF_OK:
            raise _b.GFError(rc, "global F / theta from the slabs' values")
        return F, theta

    def fix(self, omega, eps, max_sweeps, check_every):
        """Algorithm 1 with a measurement cadence (as gf_fix).  Returns (sweeps_done, [(sweep, F, theta), ...])."""
        def plan(done, theta):  # Algorithm 1 l.2 and the cadence: decided by libgf, as in gf_fix
            rc, n = _b.gf_fix_plan(float(omega), float(eps), int(max_sweeps), int(check_every), done, theta)
            if rc != _b.GF_OK:
                raise ValueError("need omega in [1,2), check_every >= 1, max_sweeps >= 0, eps >= 0")
            return n

        plan(0, 1.0)
        done = 0
        F, th = self.measure()
        history = [(0, F, th)]
        while True:
            n = plan(done, th)
            if n == 0:
                break
            self.ovr_sweep(n, omega)
            done += n
            F, th = self.measure()
            history.append((done, F, th))
        return done, history

    def kernel_launches(self):
        return sum(e.kernel_launches() for e in self.engines.values())

    def synchronize(self):
        if self.on_gpu:
            for e in self.engines.values():
                e.stream.synchronize()
            self.comm_stream.synchronize()

    def close(self):
        if self._ipc_mapped:
            self.synchronize()
            if self.dist is not None:
                self.dist.barrier(group=self.group)  # no rank unmaps while a neighbour's kernels may still store into it
            for ptr in self._ipc_mapped.values():
                if ptr:
                    _b.gf_ipc_close(ptr, 0)
            self._ipc_mapped = {}
        for e in self.engines.values():
            e.close()
        self.engines = {}
