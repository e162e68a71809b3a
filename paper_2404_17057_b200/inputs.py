"""Seeded synthetic workloads (numpy only) shaped like the paper's test cases.

This module holds NONE of the method's arithmetic (no shape functions, no P2G/G2P, no time stepping):
it only draws positions and initial states.  It is the one module both the CPU oracle's tests and the
CUDA path's tests / bench.py import, so that both sides see bit-identical inputs.

The five recipes follow BASELINE.json `configs` and SURVEY.md section 8(d); each stands in for the
paper's own input files (Sod tube PAPER.md:528-535, Mach-3 cylinder PAPER.md:543-554, uniform random
particle placement PAPER.md:526, ppc 4/9/16 PAPER.md:598-606, "3D" PAPER.md:729-733), which are not
available.  Every workload is a dict:

    cfg        dict for mpm_create / oracle_create (dim, n, dx, gamma, c0, c1, bc, inflow_*, obstacle_mask,
               node_normals, recycle_seed, ppc_inflow)
    x, v       float64 [dim, N]   positions, velocities (component-major SoA)
    mass, rho, e   float64 [N]
    cfl        alpha of eq. (25)/(29) used by the config
    steps      number of steps the config asks for
    name       workload name
"""
import numpy as np

BC_PERIODIC, BC_REFLECT, BC_INFLOW, BC_OUTFLOW = 0, 1, 2, 3


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _base_cfg(dim, n, dx, gamma, bc):
    return dict(dim=dim, n=[int(v) for v in n], dx=float(dx), gamma=float(gamma), c0=1.0, c1=1.0,
                visc_form=0, bc=bc, inflow_rho=1.0, inflow_p=1.0, inflow_v=[0.0, 0.0, 0.0],
                obstacle_mask=None, node_normals=None, recycle_seed=0, ppc_inflow=1.0)


def _lattice_positions(n, h, sub, jitter, rng, jitter_axes=None):
    """Cell-ordered (x fastest) sub-lattice of `sub` points per axis per cell, at (i+1/2)/sub of the cell,
    plus U(-jitter, jitter)*h per axis.  Returns [dim, N] with N = prod(n) * sub**dim, index = cell*sub**dim + s."""
    dim = len(n)
    ns = sub ** dim
    shape = tuple(reversed(n)) + (ns,)           # (nz, ny, nx, ns): x fastest among cells
    out = np.empty((dim,) + (int(np.prod(n)) * ns,), dtype=np.float64)
    s_idx = np.arange(ns)
    for a in range(dim):
        cell = np.arange(n[a], dtype=np.float64)
        view = [1] * (dim + 1)
        view[dim - 1 - a] = n[a]
        sub_a = ((s_idx // (sub ** a)) % sub + 0.5) / sub
        pos = cell.reshape(view) + sub_a.reshape([1] * dim + [ns])
        pos = np.broadcast_to(pos, shape).astype(np.float64)
        if jitter > 0 and (jitter_axes is None or a in jitter_axes):
            pos = pos + rng.uniform(-jitter, jitter, size=shape)
        else:
            pos = pos.copy()
        out[a] = (pos * h).ravel()
    return out


def sod(nx=256, ny=4, seed=1001, jitter=0.1, jitter_y=True, steps=100):
    """Config 1: 2D Sod shock tube, nx x ny cells, dx = 1/nx, 4 particles/cell on a jittered 2x2 lattice,
    left rho=1 p=1, right rho=0.125 p=0.1, at rest; reflecting x walls, periodic y, CFL 0.3."""
    h = 1.0 / nx
    gamma = 1.4
    cfg = _base_cfg(2, [nx, ny], h, gamma, [[BC_REFLECT, BC_REFLECT], [BC_PERIODIC, BC_PERIODIC]])
    rng = _rng(seed)
    x = _lattice_positions([nx, ny], h, 2, jitter, rng, jitter_axes=None if jitter_y else (0,))
    n = x.shape[1]
    left = x[0] < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    mass = rho * h * h / 4.0
    e = p / ((gamma - 1.0) * rho)
    v = np.zeros((2, n))
    return dict(name=f"sod2d_{nx}x{ny}", cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.3, steps=steps)


def periodic_box(n=512, seed=2002, perm_seed=None, steps=200, ppc=4):
    """Config 2: 2D periodic gas box, n x n cells, ppc particles/cell uniform in cell, rho = 1 + 0.01 N(0,1),
    p = 1, V ~ N(0, 0.1).  perm_seed != None shuffles the particle order (locality / contention sweep)."""
    h = 1.0 / n
    gamma = 1.4
    cfg = _base_cfg(2, [n, n], h, gamma, [[BC_PERIODIC, BC_PERIODIC], [BC_PERIODIC, BC_PERIODIC]])
    rng = _rng(seed)
    N = n * n * ppc
    cx = np.tile(np.repeat(np.arange(n, dtype=np.float64), ppc), n)
    cy = np.repeat(np.arange(n, dtype=np.float64), n * ppc)
    x = np.empty((2, N))
    x[0] = (cx + rng.uniform(0.0, 1.0, N)) * h
    x[1] = (cy + rng.uniform(0.0, 1.0, N)) * h
    np.clip(x, 0.0, np.nextafter(1.0, 0.0), out=x)
    rho = 1.0 + 0.01 * rng.standard_normal(N)
    p = np.ones(N)
    v = 0.1 * rng.standard_normal((2, N))
    mass = rho * h * h / ppc
    e = p / ((gamma - 1.0) * rho)
    if perm_seed is not None:
        perm = _rng(perm_seed).permutation(N)
        x, v, mass, rho, e = x[:, perm], v[:, perm], mass[perm], rho[perm], e[perm]
        x, v = np.ascontiguousarray(x), np.ascontiguousarray(v)
    name = f"box2d_{n}" + ("_shuffled" if perm_seed is not None else "")
    return dict(name=name, cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.3, steps=steps)


def cylinder(nx=2048, ny=1024, seed=3003, recycle_seed=3004, ppc=9, steps=500):
    """Config 3: Mach-3 flow past a solid cylinder on [0,4]x[0,2] (nx = 2 ny), radius 64/2048*nx cells centred
    at cell coordinates (nx/4, ny/2), given as a cell mask; ppc particles uniform in every unmasked cell;
    rho=1.4, p=1, V=(3,0); inflow x-low, outflow x-high, reflecting y; analytic radial node normals."""
    h = 4.0 / nx
    gamma = 1.4
    cfg = _base_cfg(2, [nx, ny], h, gamma, [[BC_INFLOW, BC_OUTFLOW], [BC_REFLECT, BC_REFLECT]])
    cfg.update(inflow_rho=1.4, inflow_p=1.0, inflow_v=[3.0, 0.0, 0.0], recycle_seed=recycle_seed,
               ppc_inflow=float(ppc))
    r_cells = 64.0 * nx / 2048.0
    ccx, ccy = nx / 4.0, ny / 2.0
    ix = np.arange(nx) + 0.5
    iy = np.arange(ny) + 0.5
    mask = ((ix[None, :] - ccx) ** 2 + (iy[:, None] - ccy) ** 2) <= r_cells ** 2   # [ny, nx], x fastest
    cfg["obstacle_mask"] = mask.astype(np.uint8).ravel()
    gx = np.arange(nx + 1, dtype=np.float64)[None, :] - ccx
    gy = np.arange(ny + 1, dtype=np.float64)[:, None] - ccy
    r = np.sqrt(gx * gx + gy * gy)
    r_safe = np.where(r > 0, r, 1.0)
    normals = np.stack([np.broadcast_to(gx / r_safe, r.shape).ravel(),
                        np.broadcast_to(gy / r_safe, r.shape).ravel()])
    cfg["node_normals"] = np.ascontiguousarray(normals)
    rng = _rng(seed)
    free = np.flatnonzero(~mask.ravel())
    N = free.size * ppc
    cell = np.repeat(free, ppc)
    x = np.empty((2, N))
    x[0] = ((cell % nx) + rng.uniform(0.0, 1.0, N)) * h
    x[1] = ((cell // nx) + rng.uniform(0.0, 1.0, N)) * h
    rho = np.full(N, 1.4)
    v = np.zeros((2, N))
    v[0] = 3.0
    mass = rho * h * h / ppc
    e = np.full(N, 1.0 / ((gamma - 1.0) * 1.4))
    return dict(name=f"cylinder2d_{nx}x{ny}", cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.3, steps=steps)


def sphere_tunnel(nx=48, ny=24, nz=24, seed=6006, recycle_seed=6007, ppc=8, steps=60, mach=2.0):
    """3D counterpart of the cylinder case (PAPER.md:543-554 with the z repetition of PAPER.md:729-733): supersonic flow
    past a solid sphere, radius ny/6 cells, centred at (nx/3, ny/2, nz/2) cells, given as a cell mask WITHOUT node normals
    (the library derives them from the mask, reading A7); inflow x-low, outflow x-high with recycling,
    reflecting y and z; ppc particles uniform in every free cell.  A parity workload, not one of the BASELINE configs."""
    h = 1.0 / ny
    gamma = 1.4
    u = mach * np.sqrt(gamma * 1.0 / 1.4)
    cfg = _base_cfg(3, [nx, ny, nz], h, gamma, [[BC_INFLOW, BC_OUTFLOW], [BC_REFLECT, BC_REFLECT], [BC_REFLECT, BC_REFLECT]])
    cfg.update(inflow_rho=1.4, inflow_p=1.0, inflow_v=[u, 0.0, 0.0], recycle_seed=recycle_seed, ppc_inflow=float(ppc))
    ix, iy, iz = np.arange(nx) + 0.5, np.arange(ny) + 0.5, np.arange(nz) + 0.5
    r_cells = ny / 6.0
    mask = ((ix[None, None, :] - nx / 3.0) ** 2 + (iy[None, :, None] - ny / 2.0) ** 2 +
            (iz[:, None, None] - nz / 2.0) ** 2) <= r_cells ** 2                    # [nz, ny, nx], x fastest
    cfg["obstacle_mask"] = mask.astype(np.uint8).ravel()
    rng = _rng(seed)
    free = np.flatnonzero(~mask.ravel())
    N = free.size * ppc
    cell = np.repeat(free, ppc)
    x = np.empty((3, N))
    x[0] = ((cell % nx) + rng.uniform(0.0, 1.0, N)) * h
    x[1] = (((cell // nx) % ny) + rng.uniform(0.0, 1.0, N)) * h
    x[2] = ((cell // (nx * ny)) + rng.uniform(0.0, 1.0, N)) * h
    rho = np.full(N, 1.4)
    v = np.zeros((3, N))
    v[0] = u
    mass = rho * h ** 3 / ppc
    e = np.full(N, 1.0 / ((gamma - 1.0) * 1.4))
    return dict(name=f"sphere3d_{nx}x{ny}x{nz}", cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.3, steps=steps)


def sedov(n=256, seed=4004, jitter=0.1, steps=100, e_total=1.0, p_ambient=1e-5):
    """Config 4: 3D Sedov-type blast, n^3 cells, 8 particles/cell on a jittered 2x2x2 lattice, rho=1,
    p=1e-5, total energy 1 deposited on the particles within 2 cells of the centre; reflecting walls, CFL 0.25."""
    h = 1.0 / n
    gamma = 1.4
    cfg = _base_cfg(3, [n, n, n], h, gamma, [[BC_REFLECT, BC_REFLECT]] * 3)
    cfg["visc_form"] = 1     # eq. (4) as printed heats at a rate ~ 1/rho and diverges in the evacuated centre (A3)
    rng = _rng(seed)
    x = _lattice_positions([n, n, n], h, 2, jitter, rng)
    N = x.shape[1]
    rho = np.ones(N)
    mass = np.full(N, h ** 3 / 8.0)
    e = np.full(N, p_ambient / (gamma - 1.0))
    r2 = (x[0] - 0.5) ** 2
    r2 += (x[1] - 0.5) ** 2
    r2 += (x[2] - 0.5) ** 2
    hot = np.flatnonzero(r2 <= (2.0 * h) ** 2)
    e[hot] = e_total / (hot.size * mass[0])
    v = np.zeros((3, N))
    return dict(name=f"sedov3d_{n}", cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.25, steps=steps)


def clumps(n=128, num_particles=1 << 26, seed=5005, nclumps=32, sigma_cells=3.0, steps=50):
    """Config 5: 3D clustered contention stress, n^3 periodic cells, particles drawn from `nclumps` Gaussian clumps
    (sigma = 3 cells, centres uniform), mass 1/N, p proportional to rho (p = rho), gamma = 5/3, V ~ N(0, 0.5).
    rho_k is the analytic density of the sampling mixture at X_k (nearest periodic image), so that no
    particle-grid arithmetic is needed to build the input."""
    h = 1.0 / n
    gamma = 5.0 / 3.0
    cfg = _base_cfg(3, [n, n, n], h, gamma, [[BC_PERIODIC, BC_PERIODIC]] * 3)
    cfg["visc_form"] = 1     # densities span orders of magnitude: use the dimensionally consistent form (A3)
    rng = _rng(seed)
    N = int(num_particles)
    centres = rng.uniform(0.0, 1.0, (nclumps, 3))
    which = rng.integers(0, nclumps, N)
    sigma = sigma_cells * h
    x = np.empty((3, N))
    for a in range(3):
        xa = centres[which, a] + sigma * rng.standard_normal(N)
        xa -= np.floor(xa)
        np.clip(xa, 0.0, np.nextafter(1.0, 0.0), out=xa)
        x[a] = xa
    # rho(X) = (1/nclumps) sum_j prod_a N(d_a; sigma) with d_a the nearest-image distance, total mass 1
    rho = np.zeros(N)
    norm = 1.0 / (nclumps * (np.sqrt(2.0 * np.pi) * sigma) ** 3)
    chunk = 1 << 20
    for s in range(0, N, chunk):
        sl = slice(s, min(N, s + chunk))
        acc = np.zeros(sl.stop - sl.start)
        for j in range(nclumps):
            r2 = np.zeros_like(acc)
            for a in range(3):
                dd = x[a, sl] - centres[j, a]
                dd -= np.rint(dd)
                r2 += dd * dd
            acc += np.exp(-0.5 * r2 / (sigma * sigma))
        rho[sl] = norm * acc
    rho = np.maximum(rho, 1e-12)
    mass = np.full(N, 1.0 / N)
    e = np.full(N, 1.0 / (gamma - 1.0))          # p = rho  ->  e = p / ((gamma-1) rho)
    v = 0.5 * rng.standard_normal((3, N))
    return dict(name=f"clumps3d_{n}_{N}", cfg=cfg, x=x, v=v, mass=mass, rho=rho, e=e, cfl=0.3, steps=steps)


def by_name(name, **kw):
    """The five BASELINE.json configs at full size (kw overrides sizes for reduced parity cases)."""
    table = {"sod": sod, "box": periodic_box, "cylinder": cylinder, "sedov": sedov, "clumps": clumps}
    return table[name](**kw)
