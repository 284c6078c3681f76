"""A T-slab held on the CPU whose arithmetic is the oracle's (oracle.site_update on a lattice two slices taller than the
slab: slice 0 carries the ghost links, the last slice is never read).  Test infrastructure: it plugs into
paper_1412_1498_b200.sharded.ShardedGaugeFixer through engine_factory, so that the product's exchange schedule and
transport run on CPU ranks (gloo) and their result can be compared with the oracle's sweep of the whole lattice."""
import numpy as np
import torch

import oracle


class OracleSlabEngine:
    def __init__(self, local_dims, slab, gauge="landau", storage=18):
        self.ld = tuple(local_dims)
        nx, ny, nz, lt = self.ld
        self.ext = (nx, ny, nz, lt + 2)
        self.gauge, self.storage, self.slab = gauge, storage, slab
        self.V3 = nx * ny * nz
        self.U = np.zeros((self.V3 * (lt + 2), 4, 3, 3, 2))
        self.U[:, :, [0, 1, 2], [0, 1, 2], 0] = 1.0
        s = np.arange(self.V3)
        self.par3 = (s % nx + (s // nx) % ny + s // (nx * ny)) & 1  # parity of (x, y, z)
        n = self.V3 // 2 * 18
        self.ghost = [torch.zeros(n, dtype=torch.float64), torch.zeros(n, dtype=torch.float64)]
        self.top_out = torch.zeros(n, dtype=torch.float64)
        self.top_in = torch.zeros(n, dtype=torch.float64)
        self.launches = 0

    # sites of parity q in local time slice t (global parity = local parity: lt is even), as indices into self.U
    def _sites(self, t, q):
        return (t + 1) * self.V3 + np.nonzero((self.par3 + t) % 2 == q)[0]

    def set_links(self, links):
        lt = self.ld[3]
        self.U[self.V3:(lt + 1) * self.V3] = links.numpy().reshape(-1, 4, 3, 3, 2)
        if self.storage == 12:
            oracle.project12(self.U, self.ext)

    def get_links(self, out=None):
        lt = self.ld[3]
        return torch.from_numpy(self.U[self.V3:(lt + 1) * self.V3].copy())

    def _ghost_sites(self, q):
        return self._sites(-1, q)

    def _update(self, ts, p, omega):
        for t in ts:
            for site in self._sites(t, p):
                oracle.site_update(self.U, self.ext, self.gauge, int(site), omega, self.storage)

    def pack_top(self, q):
        self.top_out.copy_(torch.from_numpy(self.U[self._sites(self.ld[3] - 1, q), 3].reshape(-1)))

    def unpack_top(self, q):
        self.U[self._sites(self.ld[3] - 1, q), 3] = self.top_in.numpy().reshape(-1, 3, 3, 2)

    def border(self, p, omega):
        lt = self.ld[3]
        for q in (0, 1):  # whatever the transport delivered since the last call
            self.U[self._ghost_sites(q), 3] = self.ghost[q].numpy().reshape(-1, 3, 3, 2)
        self._update(sorted({0, lt - 1}), p, omega)
        self.ghost[1 - p].copy_(torch.from_numpy(self.U[self._ghost_sites(1 - p), 3].reshape(-1)))
        self.pack_top(p)
        self.launches += 1

    def interior(self, p, omega):
        self._update(range(1, self.ld[3] - 1), p, omega)
        self.launches += 1

    def measure(self):
        lt = self.ld[3]
        for q in (0, 1):
            self.U[self._ghost_sites(q), 3] = self.ghost[q].numpy().reshape(-1, 3, 3, 2)
        nd = 4 if self.gauge == "landau" else 3
        f = th = 0.0
        for t in range(lt):
            for q in (0, 1):
                for site in self._sites(t, q):
                    if q == 0:
                        f += np.trace(oracle.site_K(self.U, self.ext, self.gauge, int(site))).real
                    D = oracle.site_delta(self.U, self.ext, self.gauge, int(site))
                    th += (abs(D) ** 2).sum()
        V = self.V3 * lt
        return f / (nd * 3.0 * V), th / (3.0 * V)

    def reunitarize(self):
        oracle.reunitarize(self.U, self.ext)

    def kernel_launches(self):
        return self.launches

    def close(self):
        pass
