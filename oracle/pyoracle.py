"""ctypes driver for the CPU oracle (oracle/mpm_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It shares no code with, and never
imports, the CUDA path (paper_2404_17057_b200/).  Argument marshalling only; all arithmetic is in C.
"""
import ctypes as C
import os
import importlib.util

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

BC_PERIODIC, BC_REFLECT, BC_INFLOW, BC_OUTFLOW, BC_OPEN = 0, 1, 2, 3, 4
VISC_PRINTED, VISC_STANDARD = 0, 1
BASIS_Q1, BASIS_QUADRATIC = 0, 1
G_MASS, G_MOM, G_FORCE, G_MOM2, G_NORMAL, G_FLAG = 0, 1, 2, 3, 4, 5
P_X, P_V, P_M, P_RHO, P_E, P_Q, P_VBAR, P_ACC, P_DIV = range(9)


class _Config(C.Structure):
    _fields_ = [
        ("dim", C.c_int), ("n", C.c_int * 3), ("dx", C.c_double), ("gamma", C.c_double),
        ("c0", C.c_double), ("c1", C.c_double), ("visc_form", C.c_int),
        ("bc", (C.c_int * 2) * 3),
        ("inflow_rho", C.c_double), ("inflow_p", C.c_double), ("inflow_v", C.c_double * 3),
        ("obstacle_mask", C.c_void_p), ("node_normals", C.c_void_p),
        ("recycle_seed", C.c_ulonglong), ("ppc_inflow", C.c_double), ("basis", C.c_int),
        ("slab_global_n", C.c_int), ("slab_offset", C.c_int),
    ]


class Stats(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt_last", C.c_double), ("dt_next", C.c_double), ("step", C.c_longlong),
        ("vmax", C.c_double), ("cmax", C.c_double), ("n_recycled", C.c_longlong),
        ("n_clamped", C.c_longlong), ("n_negjac", C.c_longlong), ("n_nonfinite", C.c_longlong),
    ]


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    spec = importlib.util.spec_from_file_location("_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    # MPM_ORACLE_LIB: a differently built copy of the same source (tests/test_oracle_sanitizers.py: ASan + UBSan)
    lib = C.CDLL(os.environ.get("MPM_ORACLE_LIB") or mod.build())
    vp, dp = C.c_void_p, C.POINTER(C.c_double)
    lib.oracle_create.restype = vp
    lib.oracle_create.argtypes = [C.POINTER(_Config)]
    lib.oracle_destroy.argtypes = [vp]
    lib.oracle_num_nodes.restype = C.c_longlong
    lib.oracle_num_nodes.argtypes = [vp, C.POINTER(C.c_int * 3)]
    lib.oracle_num_particles.restype = C.c_longlong
    lib.oracle_num_particles.argtypes = [vp]
    lib.oracle_load_particles.argtypes = [vp, C.c_longlong, vp, vp, vp, vp, vp, vp]
    lib.oracle_load_particles_ex.argtypes = [vp, C.c_longlong, vp, vp, vp, vp, vp, vp, vp, C.c_int]
    lib.oracle_halo.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp]
    lib.oracle_shape.argtypes = [vp, vp, vp, vp, vp]
    lib.oracle_shape_quadratic.argtypes = [vp, vp, vp, vp, vp]
    for name in ("oracle_grid_reset", "oracle_p2g1", "oracle_grid_bc", "oracle_p2g2", "oracle_grid_bc2"):
        getattr(lib, name).argtypes = [vp]
        getattr(lib, name).restype = None
    for name in ("oracle_grid_advance", "oracle_g2p_velocity", "oracle_particle_update", "oracle_advect",
                 "oracle_cfl", "oracle_advance_time"):
        getattr(lib, name).argtypes = [vp, C.c_double]
        getattr(lib, name).restype = None
    lib.oracle_mix64.restype = C.c_ulonglong
    lib.oracle_mix64.argtypes = [C.c_ulonglong]
    lib.oracle_recycle_uniform.restype = C.c_double
    lib.oracle_recycle_uniform.argtypes = [C.c_ulonglong, C.c_longlong, C.c_longlong, C.c_int]
    lib.oracle_step.argtypes = [vp, C.c_double, C.c_double, C.c_int, dp]
    lib.oracle_read_particles.argtypes = [vp, C.c_int, vp]
    lib.oracle_read_grid.argtypes = [vp, C.c_int, vp]
    lib.oracle_grid_diagnostic.argtypes = [vp, C.c_int, vp]
    lib.oracle_get_stats.argtypes = [vp, C.POINTER(Stats)]
    _lib = lib
    return lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def mix64(z):
    return int(_load().oracle_mix64(int(z) & 0xFFFFFFFFFFFFFFFF))


def recycle_uniform(seed, pid, step, j):
    return float(_load().oracle_recycle_uniform(int(seed), int(pid), int(step), int(j)))


class Oracle:
    """Thin handle around oracle_t.  `cfg` is a dict with the keys of oracle_config
    (dim, n, dx, gamma, c0, c1, visc_form, bc, inflow_rho, inflow_p, inflow_v, obstacle_mask,
    node_normals, recycle_seed, ppc_inflow, basis); missing keys take the documented defaults."""

    def __init__(self, cfg):
        lib = _load()
        self._lib = lib
        c = _Config()
        d = int(cfg["dim"])
        c.dim = d
        n = list(cfg["n"]) + [1] * (3 - len(cfg["n"]))
        for a in range(3):
            c.n[a] = int(n[a])
        c.dx = float(cfg["dx"])
        c.gamma = float(cfg.get("gamma", 1.4))
        c.c0 = float(cfg.get("c0", 1.0))
        c.c1 = float(cfg.get("c1", 1.0))
        c.visc_form = int(cfg.get("visc_form", VISC_PRINTED))
        bc = cfg.get("bc", [[BC_PERIODIC, BC_PERIODIC]] * 3)
        for a in range(3):
            for s in range(2):
                c.bc[a][s] = int(bc[a][s]) if a < len(bc) else BC_PERIODIC
        c.inflow_rho = float(cfg.get("inflow_rho", 1.0))
        c.inflow_p = float(cfg.get("inflow_p", 1.0))
        iv = list(cfg.get("inflow_v", [0.0, 0.0, 0.0])) + [0.0] * 3
        for a in range(3):
            c.inflow_v[a] = float(iv[a])
        self._keep = []
        mask = cfg.get("obstacle_mask")
        if mask is not None:
            mask = np.ascontiguousarray(mask, dtype=np.uint8).ravel()
            self._keep.append(mask)
            c.obstacle_mask = mask.ctypes.data
        normals = cfg.get("node_normals")
        if normals is not None:
            normals = _f64(normals).ravel()
            self._keep.append(normals)
            c.node_normals = normals.ctypes.data
        c.recycle_seed = int(cfg.get("recycle_seed", 0))
        c.ppc_inflow = float(cfg.get("ppc_inflow", 1.0))
        c.basis = int(cfg.get("basis", BASIS_Q1))
        c.slab_global_n = int(cfg.get("slab_global_n", 0)); c.slab_offset = int(cfg.get("slab_offset", 0))
        self.dim = d
        self._h = lib.oracle_create(C.byref(c))
        if not self._h:
            raise ValueError("oracle_create rejected the configuration")
        nn = (C.c_int * 3)()
        self.num_nodes = int(lib.oracle_num_nodes(self._h, C.byref(nn)))
        self.nn = tuple(int(v) for v in nn)
        self.n = 0

    def close(self):
        if getattr(self, "_h", None):
            self._lib.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        self.close()

    # ---- particles
    def load_particles(self, x, v, mass, rho, e, q=None, ids=None, keep_time=False):
        x, v, mass, rho, e = _f64(x), _f64(v), _f64(mass), _f64(rho), _f64(e)
        n = mass.shape[0]
        assert x.shape == (self.dim, n) and v.shape == (self.dim, n)
        qq = _f64(q) if q is not None else None
        ii = np.ascontiguousarray(ids, dtype=np.int64) if ids is not None else None
        rc = self._lib.oracle_load_particles_ex(self._h, n, x.ctypes.data, v.ctypes.data, mass.ctypes.data,
                                                rho.ctypes.data, e.ctypes.data,
                                                qq.ctypes.data if qq is not None else None,
                                                ii.ctypes.data if ii is not None else None, 1 if keep_time else 0)
        assert rc == 0
        self.n = n

    def halo(self, which, side, op, buf):
        """buf: C-contiguous float64 [channels, plane nodes]; op 0 = export into buf, 1 = add buf to the plane"""
        assert buf.dtype == np.float64 and buf.flags["C_CONTIGUOUS"]
        assert self._lib.oracle_halo(self._h, int(which), int(side), int(op), buf.ctypes.data) == 0

    def shape(self, X):
        X = _f64(X)
        nb = 1 << self.dim
        node = np.zeros(nb, dtype=np.int64)
        phi = np.zeros(nb)
        grad = np.zeros((nb, self.dim))
        self._lib.oracle_shape(self._h, X.ctypes.data, node.ctypes.data, phi.ctypes.data, grad.ctypes.data)
        return node, phi, grad

    def shape_quadratic(self, X):
        X = _f64(X)
        nb = 3 ** self.dim
        node = np.zeros(nb, dtype=np.int64)
        phi = np.zeros(nb)
        grad = np.zeros((nb, self.dim))
        self._lib.oracle_shape_quadratic(self._h, X.ctypes.data, node.ctypes.data, phi.ctypes.data, grad.ctypes.data)
        return node, phi, grad

    # ---- Algorithm 1, line by line
    def grid_reset(self): self._lib.oracle_grid_reset(self._h)
    def p2g1(self): self._lib.oracle_p2g1(self._h)
    def grid_bc(self): self._lib.oracle_grid_bc(self._h)
    def grid_advance(self, dt): self._lib.oracle_grid_advance(self._h, float(dt))
    def g2p_velocity(self, dt): self._lib.oracle_g2p_velocity(self._h, float(dt))
    def p2g2(self): self._lib.oracle_p2g2(self._h)
    def grid_bc2(self): self._lib.oracle_grid_bc2(self._h)
    def particle_update(self, dt): self._lib.oracle_particle_update(self._h, float(dt))
    def advect(self, dt): self._lib.oracle_advect(self._h, float(dt))
    def cfl(self, alpha): self._lib.oracle_cfl(self._h, float(alpha))
    def advance_time(self, dt): self._lib.oracle_advance_time(self._h, float(dt))

    def step(self, dt=0.0, cfl=0.3, nsteps=1):
        out = C.c_double(0.0)
        rc = self._lib.oracle_step(self._h, float(dt), float(cfl), int(nsteps), C.byref(out))
        assert rc == 0
        return out.value

    # ---- read-back
    def particles(self, field):
        nc = self.dim if field in (P_X, P_V, P_VBAR, P_ACC) else 1
        out = np.zeros((nc, self.n))
        rc = self._lib.oracle_read_particles(self._h, int(field), out.ctypes.data)
        assert rc == 0
        return out if nc > 1 else out[0]

    def grid(self, field):
        nc = self.dim if field in (G_MOM, G_FORCE, G_MOM2, G_NORMAL) else 1
        out = np.zeros((nc, self.num_nodes))
        rc = self._lib.oracle_read_grid(self._h, int(field), out.ctypes.data)
        assert rc == 0
        return out if nc > 1 else out[0]

    def grid_diagnostic(self, which):
        """mass-weighted nodal mean of rho (0) or E (1), reading A18"""
        out = np.zeros(self.num_nodes)
        assert self._lib.oracle_grid_diagnostic(self._h, int(which), out.ctypes.data) == 0
        return out

    def stats(self):
        s = Stats()
        self._lib.oracle_get_stats(self._h, C.byref(s))
        return s
