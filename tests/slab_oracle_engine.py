"""A CPU engine for paper_1209_4008_b200.slab.SlabRunner built on the oracle (test infrastructure): one t-slab of a
configuration in the canonical layout, owned slices followed by one ghost slice, updated site by site with
orc_site_overrelax on the local lattice (whose periodic wrap in t sends the first slice to the ghost -- exactly the
layout of a gf_create_slab context).  It lets the CPU tests drive the product's schedule and transports without a GPU."""
import numpy as np
import torch

import oracle


class OracleSlab:
    def __init__(self, dims, t_begin, t_end, U_global, gauge=oracle.LANDAU):
        assert t_begin % 2 == 0 and t_end % 2 == 0
        self.dims = tuple(dims)
        self.Nt = t_end - t_begin
        self.Vs = dims[0] * dims[1] * dims[2]
        self.ldims = (dims[0], dims[1], dims[2], self.Nt + 1)
        self.gauge = gauge
        self.U = np.zeros(((self.Nt + 1) * self.Vs, 4, 3, 3), dtype=np.complex128)
        self.U[: self.Nt * self.Vs] = U_global[t_begin * self.Vs: t_end * self.Vs]
        self.U[self.Nt * self.Vs:] = np.nan  # the ghost starts undefined: every use must follow a refresh
        s = np.arange((self.Nt + 1) * self.Vs)
        x, y, z, t = s % dims[0], (s // dims[0]) % dims[1], (s // (dims[0] * dims[1])) % dims[2], s // self.Vs
        # the ghost slice (local t = Nt, even) stands for the global slice t_begin - 1 (odd): its sites have the other parity
        self.parity = (x + y + z + t + (t == self.Nt)) & 1
        self.slice = t

    def owned(self):
        return self.U[: self.Nt * self.Vs]

    def new_face(self):
        return torch.empty(self.Vs // 2 * 18, dtype=torch.float64)

    def _sites(self, t, block_parity):
        return np.nonzero((self.slice == t) & (self.parity == block_parity))[0]

    def pack_face(self, which, block_parity, buf):
        t = self.Nt - 1 if which == 0 else self.Nt
        buf.copy_(torch.from_numpy(self.U[self._sites(t, block_parity), 3].reshape(-1).view(np.float64).copy()))
        return buf

    def unpack_face(self, which, block_parity, buf):
        t = self.Nt - 1 if which == 0 else self.Nt
        self.U[self._sites(t, block_parity), 3] = buf.numpy().view(np.complex128).reshape(-1, 3, 3)

    def begin(self):
        pass

    def half_sweep(self, kind, parity, sweep, t_first, t_count):
        assert kind[0] == "relax" and kind[1] == 0  # second-order overrelaxation (no site index in its arithmetic)
        sel = (self.slice >= t_first) & (self.slice < t_first + t_count) & (self.parity == parity)
        for s in np.nonzero(sel)[0]:
            oracle.site_overrelax(self.U, self.ldims, int(s), kind[2], self.gauge)

    def raw_sums(self):
        nd = 3 if self.gauge == oracle.COULOMB else 4
        own = self.owned()
        F = float(np.trace(own[:, :nd], axis1=-2, axis2=-1).real.sum())
        th = sum(oracle.site_theta(self.U, self.ldims, s, self.gauge) for s in range(self.Nt * self.Vs))
        return F, th

    def theta_slices(self):
        per = np.array([oracle.site_theta(self.U, self.ldims, s, self.gauge) for s in range(self.Nt * self.Vs)])
        return list(per.reshape(self.Nt, self.Vs).sum(axis=1) / (3.0 * self.Vs))
