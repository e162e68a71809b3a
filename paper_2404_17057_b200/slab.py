"""Slab decomposition of the particle-grid cycle over several GPUs (the paper's own plan: domain
decomposition with one SoA per device).

The grid is cut into slabs of whole cell layers along the LAST axis; slab s owns the cells [z0_s, z1_s) and the particles
inside them, on its own solver handle (one per GPU; `mpm_config.bc` = MPM_BC_OPEN on the interfaces).  Q1 hats reach one cell, so
neighbouring slabs share exactly one node plane.  One time step:

    1. halo SUM-exchange of the shared plane's raw first-P2G sums m, mv, f        (Alg. 1 l.3 is complete on every slab)
    2. GATHER phase on every slab with the global dt: l.4-8                         (mpm_step_phase)
    3. halo SUM-exchange of the shared plane's mv2                                  (l.8 is complete)
    4. UPDATE phase: l.9-13
    5. all-reduce(max) of v_max and c_max -> the next global dt = alpha h / (v_max + c_max)   (eq. 25/29)
    6. if any particle anywhere left its slab (a device-side counter, all-reduced with the maxima): particles that left their slab (<= 1 cell per step by the CFL condition; anywhere for a recycled
       particle) are handed to the slab that now contains them; every slab replaces its particle set, which re-orders it
       and redoes the first P2G of the next step (mpm_load_particles_ex with MPM_LOAD_KEEP_TIME and the global ids, on
       which the recycling generator of reading A8 is keyed).

This module holds the HOST logic only -- who owns what, which planes pair up, where a particle goes -- over two small
interfaces: an *engine* per slab (the CUDA solver: `CudaSlabEngine`; anything with the same methods in the tests) and a
*transport* (`LocalTransport`: all slabs in this process; `DistTransport`: torch.distributed point-to-point, NCCL between
GPUs or gloo between CPU processes).  No method arithmetic happens here: particle fields are only selected, concatenated
and shifted by the slab origin (a multiple of h).

Status: first correct multi-GPU path.  Step 6 re-sorts every slab's particles on every step (about one extra particle
sweep); a ghost-cell layer that lets arrivals join the fused re-ordering is the next step.  Measured scaling: none in this
environment (one GPU); DistTransport over NCCL is covered by construction and by the gloo test of the same code.
"""
import numpy as np


# ----------------------------------------------------------------------------------------------------------- geometry
def slab_ranges(n_last, num_slabs, tile=1):
    """Cell ranges [z0, z1) of `num_slabs` slabs along an axis of n_last cells: as even as possible in whole multiples
    of `tile` cells (the tile depth of the kernels, so that no tile straddles an interface), every slab non-empty."""
    units = -(-n_last // tile)
    if num_slabs < 1 or num_slabs > units:
        raise ValueError("more slabs than %d-cell layers" % tile)
    cuts = [min(n_last, tile * ((units * s) // num_slabs)) for s in range(num_slabs + 1)]
    return [(cuts[s], cuts[s + 1]) for s in range(num_slabs)]


def slab_config(cfg, z0, z1, first, last):
    """Solver configuration of the slab [z0, z1) of the domain described by `cfg` (the dict of inputs.py workloads)."""
    d = cfg["dim"]
    a = d - 1
    c = dict(cfg)
    n = list(cfg["n"][:d])
    nz = n[a]
    n[a] = z1 - z0
    c["n"] = n
    bc = [list(b) for b in cfg["bc"][:d]]
    periodic = bc[a][0] == 0
    single = first and last
    if not (single and periodic):
        bc[a] = [bc[a][0] if (first and not periodic) else 4, bc[a][1] if (last and not periodic) else 4]
    c["bc"] = bc
    c["slab_global_n"], c["slab_offset"] = nz, z0
    nn_other = [n[b] if cfg["bc"][b][0] == 0 else n[b] + 1 for b in range(a)]
    plane = int(np.prod(nn_other)) if nn_other else 1
    cells_other = int(np.prod(n[:a])) if a > 0 else 1
    if cfg.get("obstacle_mask") is not None:
        m = np.ascontiguousarray(cfg["obstacle_mask"], dtype=np.uint8).reshape(nz, cells_other)
        c["obstacle_mask"] = np.ascontiguousarray(m[z0:z1]).ravel()
        if cfg.get("node_normals") is None:
            raise ValueError("a decomposed obstacle needs node_normals (normals derived from a mask need the neighbours' cells)")
        nn_last = nz if periodic else nz + 1
        nrm = np.ascontiguousarray(cfg["node_normals"], dtype=np.float64).reshape(d, nn_last, plane)
        c["node_normals"] = np.ascontiguousarray(nrm[:, z0:z1 + 1]).reshape(d, -1)
    return c


# ----------------------------------------------------------------------------------------------------------- transports
# A message is one tensor, keyed (src_slab, dst_slab, tag).  The receiver knows shape and dtype of everything it is to get.
class LocalTransport:
    """All slabs live in this process (several handles on one GPU, or the host-logic tests)."""
    rank, world = 0, 1

    def owner(self, slab):
        return 0

    def route(self, messages, recv_specs):
        assert set(messages) == set(recv_specs)
        return dict(messages)

    def allreduce_max(self, values):
        return [float(v) for v in values]

    def allgather_counts(self, counts):
        return counts


class DistTransport:
    """One process per GPU (torch.distributed, backend nccl) or per CPU (gloo); slab s lives on rank s % world.
    Point-to-point isend / irecv in the same (sorted-key) order on both sides of every pair of processes."""

    def __init__(self, device="cpu"):
        import torch
        import torch.distributed as dist
        self.torch, self.dist, self.device = torch, dist, device
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def owner(self, slab):
        return slab % self.world

    def route(self, messages, recv_specs):
        """messages: {(src, dst, tag): tensor} of the local source slabs; recv_specs: {(src, dst, tag): (shape, dtype)} of
        every message with a local destination.  Returns {key: tensor} for the local destinations."""
        torch, dist = self.torch, self.dist
        out, ops, keep = {}, [], []
        for key in sorted(set(messages) | set(recv_specs)):
            src, dst, _ = key
            if key in messages and self.owner(dst) == self.rank:
                out[key] = messages[key]
            elif key in messages:
                t = messages[key].contiguous()
                keep.append(t)
                if t.numel():
                    ops.append(dist.isend(t, self.owner(dst)))
            else:
                shape, dtype = recv_specs[key]
                buf = torch.empty(shape, dtype=dtype, device=self.device)
                if buf.numel():
                    ops.append(dist.irecv(buf, self.owner(src)))
                out[key] = buf
        for op in ops:
            op.wait()
        return out

    def allreduce_max(self, values):
        t = self.torch.tensor([float(v) for v in values], dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return t.tolist()

    def allgather_counts(self, counts):
        """counts: [num_slabs, num_slabs] int64 with this process's rows filled in, zeros elsewhere -> the full matrix"""
        t = self.torch.as_tensor(counts, dtype=self.torch.int64, device=self.device).clone()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return t.cpu().numpy()


# ----------------------------------------------------------------------------------------------------------- CUDA engine
class CudaSlabEngine:
    """One slab on the CUDA solver (TILED family).  Tensors are torch CUDA tensors; nothing is computed here."""

    def __init__(self, cfg, device=0):
        import torch
        from . import binding as mpm
        self.mpm, self.torch = mpm, torch
        self.solver = mpm.Solver(cfg, sort_every=1, variant=mpm.VARIANT_TILED, device=device)
        self.dim = cfg["dim"]
        self.device = self.solver.device
        self.plane = self.solver.num_nodes // self.solver.nn[self.dim - 1]
        self.loaded = False

    def set_particles(self, x, v, mass, rho, e, q, gid):
        """torch tensors on self.device: x, v [dim, n]; the rest [n]; gid int64 = the global particle ids"""
        c = lambda t: t.contiguous()
        self.solver.load_particles(c(x), c(v), c(mass), c(rho), c(e), c(q), location=self.mpm.DEVICE, ids=c(gid),
                                   keep_time=self.loaded)
        self.loaded = True

    def get_particles(self):
        """dict of torch tensors (storage order) with 'gid' = the global ids (int64)"""
        m = self.mpm
        p = self.solver.read_particles(m.P_X | m.P_V | m.P_M | m.P_RHO | m.P_E | m.P_Q | m.P_ID, order=1, location=m.DEVICE)
        p["gid"] = p.pop("id").to(self.torch.int64)
        return p

    def halo_export(self, which, side):
        nch = (1 + 2 * self.dim) if which == 0 else self.dim
        buf = self.torch.empty((nch, self.plane), dtype=self.torch.float64, device=self.device)
        self.solver.halo(which, side, self.mpm.HALO_EXPORT, buf)
        return buf

    def halo_add(self, which, side, buf):
        self.solver.halo(which, side, self.mpm.HALO_ADD, buf.contiguous())

    def phase_gather(self, dt):
        self.solver.step_phase(self.mpm.PHASE_GATHER, dt)

    def phase_update(self):
        self.solver.step_phase(self.mpm.PHASE_UPDATE)

    def maxima(self):
        """(v_max, c_max, cumulative number of particles that ended a step beyond an interface)"""
        vmax, cmax, left, _ = self.solver.peek()
        return vmax, cmax, left

    def stats(self):
        return self.solver.stats()

    def close(self):
        self.solver.close()


# ----------------------------------------------------------------------------------------------------------- driver
class SlabDomain:
    """The decomposed solver: the slabs this process owns, stepped in lock step with everybody else's."""

    def __init__(self, cfg, num_slabs, transport=None, engine_factory=None, tile_depth=None):
        import torch
        self.torch = torch
        self.cfg, self.dim = cfg, cfg["dim"]
        self.axis = self.dim - 1
        self.h = cfg["dx"]
        self.n_last = cfg["n"][self.axis]
        self.periodic = cfg["bc"][self.axis][0] == 0
        self.transport = transport or LocalTransport()
        if tile_depth is None:
            tile_depth = 4 if self.dim == 3 else 16          # TileGeo: no tile straddles an interface
        self.ranges = slab_ranges(self.n_last, num_slabs, tile_depth)
        self.num_slabs = num_slabs
        self.local = [s for s in range(num_slabs) if self.transport.owner(s) == self.transport.rank]
        factory = engine_factory or (lambda c, s: CudaSlabEngine(c))
        self.engines = {}
        for s in self.local:
            z0, z1 = self.ranges[s]
            self.engines[s] = factory(slab_config(cfg, z0, z1, s == 0, s == num_slabs - 1), s)
        self.vmax = self.cmax = 0.0
        self.t, self.step_count, self.dt_last = 0.0, 0, 0.0
        self.n_migrated = 0
        self._left_seen = {}
        # interfaces (lower slab, upper slab): the lower one's HIGH plane is the upper one's LOW plane
        self.interfaces = [(s, s + 1) for s in range(num_slabs - 1)]
        if self.periodic and num_slabs > 1:
            self.interfaces.append((num_slabs - 1, 0))

    # -- ownership
    def _dest_slab(self, z_global):
        """destination slab of a coordinate along the slab axis (torch tensor), and the coordinate after the periodic wrap"""
        torch = self.torch
        L = self.n_last * self.h
        if self.periodic:
            z_global = z_global - L * torch.floor(z_global / L)
            z_global = torch.where(z_global >= L, torch.zeros_like(z_global), z_global)
        cell = torch.clamp(torch.floor(z_global / self.h), 0, self.n_last - 1).to(torch.int64)
        starts = torch.tensor([r[0] for r in self.ranges[1:]], dtype=torch.int64, device=z_global.device)
        return torch.bucketize(cell, starts, right=True), z_global

    def load_particles(self, x, v, mass, rho, e, q=None):
        """Every process passes the GLOBAL arrays (numpy, load order = global id) and keeps its slabs' share."""
        torch = self.torch
        x = np.asarray(x, dtype=np.float64)
        v, mass, rho, e = (np.asarray(t, dtype=np.float64) for t in (v, mass, rho, e))
        q = np.zeros_like(mass) if q is None else np.asarray(q, dtype=np.float64)
        dest, _ = self._dest_slab(torch.from_numpy(np.ascontiguousarray(x[self.axis])))
        dest = dest.numpy()
        for s in self.local:
            sel = np.nonzero(dest == s)[0]
            eng = self.engines[s]
            dev = getattr(eng, "device", "cpu")
            xs = x[:, sel].copy()
            xs[self.axis] -= self.ranges[s][0] * self.h          # slab-local coordinate (exact for the power-of-two h of the configs)
            up = lambda t: torch.from_numpy(np.ascontiguousarray(t)).to(dev)
            eng.set_particles(up(xs), up(v[:, sel]), up(mass[sel]), up(rho[sel]), up(e[sel]), up(q[sel]), up(sel.astype(np.int64)))
        self._reduce_maxima()

    def _reduce_maxima(self):
        """global CFL maxima (eq. 25/29); returns whether any particle, anywhere, left its slab since the last hand-over"""
        vm = cm = 0.0
        left = 0
        for s in self.local:
            v, c, l = self.engines[s].maxima()
            vm, cm = max(vm, v), max(cm, c)
            left += l - self._left_seen.get(s, 0)
            self._left_seen[s] = l
        self.vmax, self.cmax, any_left = self.transport.allreduce_max([vm, cm, float(left > 0)])
        return any_left > 0.0

    # -- halo SUM-exchange of the shared node planes; which = 0: m, mv, f of the first P2G, 1: mv2 of the second
    def _halo_exchange(self, which):
        torch = self.torch
        nch = (1 + 2 * self.dim) if which == 0 else self.dim
        msgs, specs = {}, {}
        for lo, hi in self.interfaces:
            # tag = the plane of the DESTINATION the message is added to: 0 = its low plane, 1 = its high plane
            if lo in self.engines:
                msgs[(lo, hi, 0)] = self.engines[lo].halo_export(which, 1)
            if hi in self.engines:
                msgs[(hi, lo, 1)] = self.engines[hi].halo_export(which, 0)
            if hi in self.engines:
                specs[(lo, hi, 0)] = ((nch, self.engines[hi].plane), torch.float64)
            if lo in self.engines:
                specs[(hi, lo, 1)] = ((nch, self.engines[lo].plane), torch.float64)
        got = self.transport.route(msgs, specs)
        for (src, dst, side), plane in sorted(got.items(), key=lambda kv: kv[0]):
            self.engines[dst].halo_add(which, side, plane)        # mine + theirs on both sides: the same sum bit for bit

    # -- hand-over of the particles that left their slab
    def _migrate(self):
        torch = self.torch
        d, a = self.dim, self.axis
        R = self.num_slabs
        counts = np.zeros((R, R), dtype=np.int64)
        packed, stay = {}, {}
        for s in self.local:
            p = self.engines[s].get_particles()
            z0 = self.ranges[s][0] * self.h
            dest, zg = self._dest_slab(p["x"][a] + z0)
            rows = [p["x"][b] for b in range(d)] + [p["v"][b] for b in range(d)] + [p["mass"], p["rho"], p["e"], p["q"],
                                                                                      p["gid"].to(torch.float64)]
            allf = torch.stack(rows)                               # [2 d + 5, n]; ids < 2^53 are exact in fp64
            allf[a] = zg                                           # global (wrapped) coordinate; made slab-local on arrival
            for t in range(R):
                sel = torch.nonzero(dest == t).flatten()
                if t == s:
                    stay[s] = allf[:, sel]
                elif sel.numel():
                    packed[(s, t, 0)] = allf[:, sel]
                    counts[s, t] = int(sel.numel())
        counts = np.asarray(self.transport.allgather_counts(counts))
        specs = {}
        for t in self.local:
            dev = stay[t].device
            for s in range(R):
                if s != t and counts[s, t] > 0:
                    specs[(s, t, 0)] = ((2 * d + 5, int(counts[s, t])), torch.float64)
        msgs = {k: v for k, v in packed.items()}
        got = self.transport.route(msgs, specs)
        for t in self.local:
            parts = [stay[t]] + [got[k] for k in sorted(got) if k[1] == t]
            f = torch.cat([x.to(stay[t].device) for x in parts], dim=1)
            f[a] = f[a] - self.ranges[t][0] * self.h
            self.engines[t].set_particles(f[0:d], f[d:2 * d], f[2 * d], f[2 * d + 1], f[2 * d + 2], f[2 * d + 3],
                                          f[2 * d + 4].to(torch.int64))
        self.n_migrated += int(counts.sum())

    def step(self, cfl, nsteps=1, dt=0.0):
        """nsteps time steps with dt = cfl h / (v_max + c_max) over ALL slabs (eq. 25/29), or a fixed dt > 0"""
        for _ in range(nsteps):
            step_dt = dt if dt > 0.0 else cfl * self.h / (self.vmax + self.cmax)
            self._halo_exchange(0)
            for s in self.local:
                self.engines[s].phase_gather(step_dt)
            self._halo_exchange(1)
            for s in self.local:
                self.engines[s].phase_update()
            if self._reduce_maxima():      # nobody crossed an interface: the fused re-ordering and P2G#1 stand, nothing to do
                self._migrate()
            self.t += step_dt
            self.dt_last = step_dt
            self.step_count += 1
        return self.dt_last

    def gather_particles(self):
        """The local slabs' particles with GLOBAL coordinates and ids: dict of numpy arrays (+ 'gid'), unordered."""
        torch = self.torch
        out = {k: [] for k in ("x", "v", "mass", "rho", "e", "q", "gid")}
        for s in self.local:
            p = self.engines[s].get_particles()
            x = p["x"].clone()
            x[self.axis] = x[self.axis] + self.ranges[s][0] * self.h
            for k in ("v", "mass", "rho", "e", "q"):
                out[k].append(p[k].cpu().numpy())
            out["x"].append(x.cpu().numpy())
            out["gid"].append(p["gid"].cpu().numpy())
        return {k: np.concatenate(vals, axis=-1) for k, vals in out.items()}

    def close(self):
        for e in self.engines.values():
            if hasattr(e, "close"):
                e.close()
