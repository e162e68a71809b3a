"""The CPU oracle as the per-slab engine of paper_2404_17057_b200/slab.py (test infrastructure: the multi-process gloo
test drives the REAL decomposition logic with it and compares with the single-domain oracle).  Same duck-typed interface as
slab.CudaSlabEngine; the phases are the oracle's own line-by-line functions of Algorithm 1:
    set_particles : load + l.2 grid reset + l.3 first P2G (raw sums, before any boundary condition)
    phase_gather  : l.4 BC, l.5 momentum advance, l.6-7 G2P + velocity update, l.8 second P2G (raw)
    phase_update  : l.9 BC, l.10 particle update, l.13 CFL maxima, l.11 advection
"""
import numpy as np
import torch

from oracle import pyoracle as po


class OracleSlabEngine:
    device = "cpu"

    def __init__(self, cfg):
        self.o = po.Oracle(cfg)
        self.dim = cfg["dim"]
        self.plane = self.o.num_nodes // self.o.nn[self.dim - 1]
        self.loaded = False
        self.gid = np.zeros(0, dtype=np.int64)

    def set_particles(self, x, v, mass, rho, e, q, gid):
        self.gid = gid.numpy().astype(np.int64)
        self.o.load_particles(x.numpy(), v.numpy(), mass.numpy(), rho.numpy(), e.numpy(), q.numpy(), ids=self.gid,
                              keep_time=self.loaded)
        self.loaded = True
        self.o.grid_reset()
        self.o.p2g1()

    def get_particles(self):
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
        o = self.o
        if o.n == 0:
            z = torch.zeros(0, dtype=torch.float64)
            zz = torch.zeros((self.dim, 0), dtype=torch.float64)
            return {"x": zz, "v": zz.clone(), "mass": z, "rho": z.clone(), "e": z.clone(), "q": z.clone(), "gid": torch.zeros(0, dtype=torch.int64)}
        return {"x": t(o.particles(po.P_X)), "v": t(o.particles(po.P_V)), "mass": t(o.particles(po.P_M)),
                "rho": t(o.particles(po.P_RHO)), "e": t(o.particles(po.P_E)), "q": t(o.particles(po.P_Q)), "gid": t(self.gid)}

    def halo_export(self, which, side):
        buf = np.zeros(((1 + 2 * self.dim) if which == 0 else self.dim, self.plane))
        self.o.halo(which, side, 0, buf)
        return torch.from_numpy(buf)

    def halo_add(self, which, side, buf):
        self.o.halo(which, side, 1, np.ascontiguousarray(buf.numpy()))

    def phase_gather(self, dt):
        self.dt = dt
        o = self.o
        o.grid_bc(); o.grid_advance(dt); o.g2p_velocity(dt); o.p2g2()

    def phase_update(self):
        o = self.o
        o.grid_bc2(); o.particle_update(self.dt); o.cfl(0.0); o.advect(self.dt)
        o.advance_time(self.dt)

    def maxima(self):
        s = self.o.stats()
        self._left = getattr(self, "_left", 0) + 1      # the oracle engine does not count leavers: always hand over
        return s.vmax, s.cmax, self._left

    def stats(self):
        return self.o.stats()
