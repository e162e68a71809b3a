"""Thin ctypes binding over libmpm_b200.so (include/mpm.h).  Argument marshalling ONLY: every step of the
particle-grid cycle runs in the CUDA kernels of csrc/.  PyTorch supplies device memory (the allocator callbacks
hand out torch caching-allocator blocks), the CUDA stream and pinned host buffers -- nothing else.

There is no CPU fallback: load() raises if the library has not been built or no CUDA device is present.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# MPM_B200_LIB: another build of the same sources (tests: the checked build libmpm_b200_checked.so)
LIB_PATH = os.environ.get("MPM_B200_LIB") or os.path.join(_HERE, "libmpm_b200.so")

OK, E_ARG, E_CUDA, E_OOM, E_STATE, E_NONFINITE = 0, -1, -2, -3, -4, -5
HOST, DEVICE = 0, 1
BC_PERIODIC, BC_REFLECT, BC_INFLOW, BC_OUTFLOW, BC_OPEN = 0, 1, 2, 3, 4
PHASE_GATHER, PHASE_UPDATE = 0, 1
HALO_P2G1, HALO_P2G2 = 0, 1
HALO_EXPORT, HALO_ADD = 0, 1
VISC_PRINTED, VISC_STANDARD = 0, 1
VARIANT_AUTO, VARIANT_ATOMIC, VARIANT_SORTED_RETIRED, VARIANT_TILED = 0, 1, 2, 3
ACCUM_FP64, ACCUM_FP32 = 0, 1
STREAM_CP_ASYNC, STREAM_BULK = 0, 1
BASIS_Q1, BASIS_QUADRATIC = 0, 1
IDS_TRACK, IDS_NONE = 0, 1
P2G_RED, P2G_COLOUR_G2P, P2G_COLOUR_UPDATE, P2G_COLOUR_BOTH = 0, 1, 2, 3
P_X, P_V, P_M, P_RHO, P_E, P_Q, P_ID = 1, 2, 4, 8, 16, 32, 64
LOAD_KEEP_TIME = 1
G_MASS, G_MOMENTUM, G_FORCE, G_MOMENTUM2, G_NORMAL, G_FLAG, G_RHO_GRID, G_E_GRID = 0, 1, 2, 3, 4, 5, 6, 7

K_P2G1, K_NODE1, K_G2P_P2G2, K_NODE2, K_UPDATE, K_SORT, K_MISC = range(7)
KERNEL_NAMES = ["p2g1", "node1", "g2p_p2g2", "node2", "update", "sort", "misc"]

EXPORTS = ["mpm_peek", "mpm_step_phase", "mpm_halo", "mpm_load_particles_ex", "mpm_set_profiling", "mpm_abi_version", "mpm_create", "mpm_load_particles", "mpm_step", "mpm_read_particles",
           "mpm_read_grid", "mpm_get_stats", "mpm_last_error", "mpm_destroy"]

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Config(C.Structure):
    _fields_ = [
        ("dim", C.c_int32), ("n", C.c_int32 * 3), ("dx", C.c_double), ("gamma", C.c_double),
        ("c0", C.c_double), ("c1", C.c_double), ("visc_form", C.c_int32), ("bc", (C.c_int32 * 2) * 3),
        ("inflow_rho", C.c_double), ("inflow_p", C.c_double), ("inflow_v", C.c_double * 3),
        ("obstacle_mask", C.c_void_p), ("node_normals", C.c_void_p),
        ("recycle_seed", C.c_uint64), ("ppc_inflow", C.c_double),
        ("sort_every", C.c_int32), ("variant", C.c_int32), ("device", C.c_int32), ("grid_accum", C.c_int32),
        ("particle_stream", C.c_int32), ("p2g_mode", C.c_int32),
        ("stream", C.c_void_p), ("alloc", ALLOC_FN), ("free", FREE_FN), ("alloc_user", C.c_void_p),
        ("basis", C.c_int32), ("slab_global_n", C.c_int32), ("slab_offset", C.c_int32), ("particle_ids", C.c_int32),
    ]


class Stats(C.Structure):
    _fields_ = [
        ("t", C.c_double), ("dt_last", C.c_double), ("dt_next", C.c_double), ("step", C.c_int64),
        ("vmax", C.c_double), ("cmax", C.c_double),
        ("n_recycled", C.c_int64), ("n_clamped", C.c_int64), ("n_negjac", C.c_int64), ("n_nonfinite", C.c_int64),
        ("sum_mass", C.c_double), ("sum_momentum", C.c_double * 3), ("sum_energy", C.c_double),
        ("num_particles", C.c_int64), ("num_nodes", C.c_int64), ("nn", C.c_int32 * 3), ("variant", C.c_int32),
        ("launches", C.c_int64), ("kernel_ms", C.c_double * 8), ("kernel_calls", C.c_int64 * 8),
        ("n_cell_changes", C.c_int64), ("n_out_of_cell", C.c_int64), ("n_bad_dt", C.c_int64), ("n_left_slab", C.c_int64),
    ]


_lib = None


def load_library():
    """dlopen libmpm_b200.so and declare the prototypes (works without a GPU; no compute call is made)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2404_17057_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    lib.mpm_abi_version.restype = C.c_int
    lib.mpm_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
    lib.mpm_load_particles.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp, vp, C.c_int]
    lib.mpm_step.argtypes = [vp, C.c_double, C.c_double, C.c_int32, C.POINTER(C.c_double)]
    lib.mpm_load_particles_ex.argtypes = [vp, C.c_int64, vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_int]
    lib.mpm_step_phase.argtypes = [vp, C.c_int, C.c_double]
    lib.mpm_peek.argtypes = [vp, C.POINTER(C.c_double * 4)]
    lib.mpm_halo.argtypes = [vp, C.c_int, C.c_int, C.c_int, vp, C.c_int]
    lib.mpm_read_particles.argtypes = [vp, C.c_uint32, vp, C.c_int, C.c_int]
    lib.mpm_read_grid.argtypes = [vp, C.c_int, vp, C.c_int]
    lib.mpm_get_stats.argtypes = [vp, C.POINTER(Stats)]
    lib.mpm_set_profiling.argtypes = [vp, C.c_int]
    lib.mpm_last_error.restype = C.c_char_p
    lib.mpm_last_error.argtypes = [vp]
    lib.mpm_destroy.argtypes = [vp]
    lib.mpm_destroy.restype = None
    _lib = lib
    return lib


def load():
    """Library + a usable CUDA device, or a loud failure."""
    lib = load_library()
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2404_17057_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
    return lib


class MpmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"mpm error {code}: {msg}")
        self.code = code


class Solver:
    """mpm_handle wrapper.  `cfg` is the dict of inputs.py workloads (`w["cfg"]`); extra keyword arguments
    (sort_every, variant, device, grid_accum, particle_stream, p2g_mode, particle_ids) select the execution options of mpm_config."""

    def __init__(self, cfg, sort_every=0, variant=VARIANT_AUTO, device=0, use_torch_allocator=True, grid_accum=0,
                 particle_stream=STREAM_CP_ASYNC, p2g_mode=P2G_RED, particle_ids=IDS_TRACK):
        import torch
        self._lib = load()
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.dim = int(cfg["dim"])
        c = Config()
        c.dim = self.dim
        n = list(cfg["n"]) + [1] * (3 - len(cfg["n"]))
        for a in range(3):
            c.n[a] = int(n[a])
        c.dx = float(cfg["dx"]); c.gamma = float(cfg.get("gamma", 1.4))
        c.c0 = float(cfg.get("c0", 1.0)); c.c1 = float(cfg.get("c1", 1.0))
        c.visc_form = int(cfg.get("visc_form", VISC_PRINTED))
        bc = cfg.get("bc", [[BC_PERIODIC, BC_PERIODIC]] * 3)
        for a in range(3):
            for s in range(2):
                c.bc[a][s] = int(bc[a][s]) if a < len(bc) else BC_PERIODIC
        c.inflow_rho = float(cfg.get("inflow_rho", 1.0)); c.inflow_p = float(cfg.get("inflow_p", 1.0))
        iv = list(cfg.get("inflow_v", [0.0] * 3)) + [0.0] * 3
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
            normals = np.ascontiguousarray(normals, dtype=np.float64).ravel()
            self._keep.append(normals)
            c.node_normals = normals.ctypes.data
        c.recycle_seed = int(cfg.get("recycle_seed", 0)); c.ppc_inflow = float(cfg.get("ppc_inflow", 1.0))
        c.sort_every = int(sort_every); c.variant = int(variant); c.device = int(device)
        c.grid_accum = int(grid_accum)
        c.particle_stream = int(particle_stream)
        c.p2g_mode = int(p2g_mode)
        c.particle_ids = int(particle_ids)
        c.basis = int(cfg.get("basis", BASIS_Q1))
        c.slab_global_n = int(cfg.get("slab_global_n", 0)); c.slab_offset = int(cfg.get("slab_offset", 0))
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream()
        c.stream = self.stream.cuda_stream
        self._blocks = {}
        if use_torch_allocator:
            def _alloc(nbytes, stream, user):
                try:
                    t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
                except Exception:
                    return None
                self._blocks[t.data_ptr()] = t
                return t.data_ptr()

            def _free(ptr, user):
                self._blocks.pop(ptr, None)

            self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)
            c.alloc, c.free = self._alloc_cb, self._free_cb
        self._cfg = c
        h = C.c_void_p()
        rc = self._lib.mpm_create(C.byref(c), C.byref(h))
        if rc != OK:
            raise MpmError(rc, self._lib.mpm_last_error(None).decode())
        self._h = h
        self.n = 0
        st = self.stats()
        self.num_nodes = int(st.num_nodes)
        self.nn = tuple(int(v) for v in st.nn)
        # mpm.h MPM_IDS_NONE: honoured by the TILED family on grids without an INFLOW face
        inflow = any(int(c.bc[a][sd]) == BC_INFLOW for a in range(self.dim) for sd in range(2))
        self.ids_tracked = not (int(particle_ids) == IDS_NONE and int(st.variant) == VARIANT_TILED and not inflow)

    # ------------------------------------------------------------------ plumbing
    def _check(self, rc):
        if rc != OK:
            raise MpmError(rc, self._lib.mpm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._lib.mpm_destroy(self._h)
            self._h = None
            self._blocks.clear()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _ptr(a):
        if isinstance(a, np.ndarray):
            return a.ctypes.data
        return a.data_ptr()          # torch tensor (host pinned or device)

    # ------------------------------------------------------------------ the C-ABI calls
    def load_particles(self, x, v, mass, rho, e, q=None, location=HOST, ids=None, keep_time=False):
        """x, v: [dim, N]; mass, rho, e, q: [N].  numpy arrays / pinned torch tensors (HOST) or CUDA tensors (DEVICE).
        ids (int64, same location) / keep_time: mpm_load_particles_ex (caller-chosen persistent ids; time, step and
        counters kept)."""
        d = self.dim
        n = int(mass.shape[0])
        if location == HOST:
            cv = (lambda a: np.ascontiguousarray(a, dtype=np.float64)) if isinstance(mass, np.ndarray) else (lambda a: a.contiguous())
            x, v, mass, rho, e = cv(x), cv(v), cv(mass), cv(rho), cv(e)
            q = cv(q) if q is not None else None
        xp = (C.c_void_p * d)(*[self._ptr(x[a]) for a in range(d)])
        vp = (C.c_void_p * d)(*[self._ptr(v[a]) for a in range(d)])
        if ids is None and not keep_time:
            self._check(self._lib.mpm_load_particles(self._h, n, xp, vp, self._ptr(mass), self._ptr(rho), self._ptr(e),
                                                     self._ptr(q) if q is not None else None, location))
        else:
            if ids is not None and isinstance(ids, np.ndarray):
                ids = np.ascontiguousarray(ids, dtype=np.int64)
            self._check(self._lib.mpm_load_particles_ex(self._h, n, xp, vp, self._ptr(mass), self._ptr(rho), self._ptr(e),
                                                        self._ptr(q) if q is not None else None,
                                                        self._ptr(ids) if ids is not None else None, location,
                                                        LOAD_KEEP_TIME if keep_time else 0))
        self.n = n

    def step_phase(self, phase, dt=0.0):
        self._check(self._lib.mpm_step_phase(self._h, int(phase), float(dt)))

    def peek(self):
        """(v_max, c_max, particles that left through OPEN faces so far, t) without the reductions of stats()"""
        out = (C.c_double * 4)()
        self._check(self._lib.mpm_peek(self._h, C.byref(out)))
        return out[0], out[1], int(out[2]), out[3]

    def halo(self, which, side, op, buf, location=DEVICE):
        """buf: [channels, plane nodes] float64, contiguous (CUDA tensor for DEVICE, numpy / pinned tensor for HOST)."""
        self._check(self._lib.mpm_halo(self._h, int(which), int(side), int(op), self._ptr(buf), location))

    def step(self, dt=0.0, cfl=0.3, nsteps=1, sync=True):
        if sync:
            out = C.c_double(0.0)
            self._check(self._lib.mpm_step(self._h, float(dt), float(cfl), int(nsteps), C.byref(out)))
            return out.value
        self._check(self._lib.mpm_step(self._h, float(dt), float(cfl), int(nsteps), None))
        return None

    def read_particles(self, mask=P_X | P_V | P_M | P_RHO | P_E | P_Q, order=None, out=None, location=HOST):
        """Returns a dict name -> array ([dim, N] for X and V).  `out` may supply preallocated buffers
        (numpy / pinned torch for HOST, CUDA tensors for DEVICE) under the same names.  order: 0 = load order (by
        persistent id), 1 = storage order; default 0, or 1 for a solver created with IDS_NONE."""
        if order is None:
            order = 0 if self.ids_tracked else 1
        d, n = self.dim, self.n
        names = [("x", P_X, d), ("v", P_V, d), ("mass", P_M, 1), ("rho", P_RHO, 1), ("e", P_E, 1), ("q", P_Q, 1), ("id", P_ID, 1)]
        res, ptrs = {}, []
        for name, bit, nc in names:
            if not mask & bit:
                continue
            if out is not None and name in out:
                buf = out[name]
            elif location == HOST:
                buf = np.empty((nc, n) if nc > 1 else (n,), dtype=np.float64)
            else:
                buf = self._torch.empty((nc, n) if nc > 1 else (n,), dtype=self._torch.float64, device=self.device)
            res[name] = buf
            if nc > 1:
                ptrs += [self._ptr(buf[a]) for a in range(nc)]
            else:
                ptrs.append(self._ptr(buf))
        arr = (C.c_void_p * len(ptrs))(*ptrs)
        self._check(self._lib.mpm_read_particles(self._h, mask, arr, int(order), location))
        return res

    def read_grid(self, field):
        nc = self.dim if field in (G_MOMENTUM, G_FORCE, G_MOMENTUM2, G_NORMAL) else 1
        out = np.empty((nc, self.num_nodes), dtype=np.float64)
        self._check(self._lib.mpm_read_grid(self._h, int(field), out.ctypes.data, HOST))
        return out if nc > 1 else out[0]

    def set_profiling(self, on=True):
        self._check(self._lib.mpm_set_profiling(self._h, 1 if on else 0))

    def stats(self):
        s = Stats()
        self._check(self._lib.mpm_get_stats(self._h, C.byref(s)))
        return s
