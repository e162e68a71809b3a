/*
 * mpm.h -- C ABI of libmpm_b200.so: the per-time-step particle-grid cycle of the compressible-flow
 * Material Point Method of arXiv 2404.17057 (Section 3, steps (i)-(xiv), and
 * Algorithm 1), implemented as hand-written CUDA kernels for sm_100a (B200).
 *
 * Shape of the interface = the paper's problem statement: an object is constructed ONCE from the grid,
 * boundary flags and obstacle normals and the particles are copied to the device ONCE;
 * the time loop then runs entirely on the device; data come back only on request
 * (PAPER.md:381, :385).
 *
 * Conventions
 *   - plain C, no exceptions or aborts cross the ABI; every call returns MPM_OK (0) or a negative MPM_E_* code,
 *     and mpm_last_error() gives a human-readable reason.
 *   - inputs are COPIED (caller keeps ownership); outputs are written into caller-allocated buffers; the handle
 *     owns all device memory it allocates (through the allocator callbacks if given, else cudaMalloc).
 *   - every pointer argument says whether it is HOST or DEVICE memory; `ptr_location` arguments select at run
 *     time (MPM_HOST: cudaMemcpyAsync from/to host memory, pinned recommended; MPM_DEVICE: device-to-device).
 *   - all arithmetic is fp64.  Vector particle/grid fields are component-major SoA: one
 *     pointer per component (particles) or [ncomp][N_n] (grid), x fastest in node/cell indices:
 *     node i = ix + NX (iy + NY iz), NX = n[0] (periodic axis) or n[0]+1.
 *   - calls are asynchronous on `stream` except mpm_read_*, mpm_get_stats and mpm_step with dt_last != NULL,
 *     which synchronise the stream.  A handle is not thread-safe.
 *   - there is NO CPU fallback: without a CUDA device mpm_create fails with MPM_E_CUDA.
 */
#ifndef MPM_B200_H
#define MPM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MPM_ABI_VERSION 2   /* 2: mpm_stats grew three counters, mpm_config two fields; the SORTED kernel family was retired */

#if defined(__GNUC__)
#define MPM_API __attribute__((visibility("default")))
#else
#define MPM_API
#endif

/* return codes */
enum { MPM_OK = 0, MPM_E_ARG = -1, MPM_E_CUDA = -2, MPM_E_OOM = -3, MPM_E_STATE = -4, MPM_E_NONFINITE = -5 };
/* pointer location */
enum { MPM_HOST = 0, MPM_DEVICE = 1 };
/* boundary condition of a domain face, bc[axis][side], side 0 = low, 1 = high.
 * PERIODIC must be set on both sides of an axis.  REFLECT: v.n = 0 (eq. 30), normal components of
 * nodal momentum and force zeroed.  INFLOW: Dirichlet, nodal momentum = m v_in, force = 0.
 * OUTFLOW: nodal momentum untouched, normal force zeroed; particles that pass the face are recycled at the
 * first INFLOW face with the inflow state. */
enum { MPM_BC_PERIODIC = 0, MPM_BC_REFLECT = 1, MPM_BC_INFLOW = 2, MPM_BC_OUTFLOW = 3 };
/* artificial viscosity q of eq. (4): as printed, or the textbook rho (c0 h^2 D^2 - c1 h c_s D) */
enum { MPM_VISC_PRINTED = 0, MPM_VISC_STANDARD = 1 };
/* kernel family.  AUTO = TILED when sort_every == 1, else ATOMIC.
 * ATOMIC: one thread per particle, global fp64 atomics (the paper's design); any particle order;
 *         sort_every = k > 0 adds a separate cell-key counting sort every k steps.
 * TILED:  particles are kept exactly cell-sorted every step, in tile-major cell order with even-aligned cell slots
 *         (128-bit particle loads); the re-ordering is fused into the sweeps; one cell per group of 2^dim / 2 lanes,
 *         contributions summed inside the group before they reach the grid; shared-memory grid tiles: the node
 *         velocities of a tile are formed once per block from the raw sums (BC, momentum advance and quotients
 *         included); two particle sweeps per step (the next step's first P2G is fused into the particle update).
 *         Ignores sort_every (always 1).
 * (2 was the SORTED family of ABI version 1, an intermediate of TILED; mpm_create now rejects it.) */
enum { MPM_VARIANT_AUTO = 0, MPM_VARIANT_ATOMIC = 1, MPM_VARIANT_SORTED_RETIRED = 2, MPM_VARIANT_TILED = 3 };
/* precision of the node sums m, mv, f, mv2 ("the code supports different choices"): FP64 (default), or FP32
 * = the fp32 grid-accumulation variant of the clustered stress workload: the scatters reduce in fp32 and the sums are
 * kept in fp32, all particle arithmetic stays fp64.  TILED family only (MPM_E_ARG otherwise). */
enum { MPM_ACCUM_FP64 = 0, MPM_ACCUM_FP32 = 1 };
/* how the TILED kernels bring the next pass's particle fields into shared memory: CP_ASYNC (default) = per-thread
 * 16-byte cp.async; BULK = one bulk asynchronous copy (cp.async.bulk, the non-tensor form of TMA) per field, warp and pass,
 * tracked by an mbarrier (a tile's particles are one contiguous run of slots).  Same results bit for bit.  TILED only. */
enum { MPM_STREAM_CP_ASYNC = 0, MPM_STREAM_BULK = 1 };
/* particle fields (bit mask for mpm_read_particles; output pointers are consumed in this order, a vector field
 * takes `dim` pointers) */
enum { MPM_P_X = 1, MPM_P_V = 2, MPM_P_M = 4, MPM_P_RHO = 8, MPM_P_E = 16, MPM_P_Q = 32 };
/* grid fields for mpm_read_grid, as left by the LAST completed step (Algorithm 1):
 *   MASS       m_i                         after l.3   (1 component)
 *   MOMENTUM   (mv)'_i = mv_i + dt f_i     after l.5   (dim components)
 *   FORCE      f_i after BC/obstacle       after l.4   (dim)
 *   MOMENTUM2  second momentum P2G, after BC   l.9     (dim)
 *   NORMAL     obstacle normals n_i (static)           (dim)
 *   FLAG       1.0 at obstacle nodes, else 0 (static)  (1)  */
enum { MPM_G_MASS = 0, MPM_G_MOMENTUM = 1, MPM_G_FORCE = 2, MPM_G_MOMENTUM2 = 3, MPM_G_NORMAL = 4, MPM_G_FLAG = 5 };

/* device allocator callbacks (e.g. torch's caching allocator).  `stream` is the cudaStream_t of the handle. */
typedef void *(*mpm_alloc_fn)(size_t bytes, void *stream, void *user);
typedef void (*mpm_free_fn)(void *ptr, void *user);

typedef struct mpm_config {
    int32_t dim;              /* 2 or 3 (PAPER.md:729-733 for 3D) */
    int32_t n[3];             /* cells per axis; n[2] ignored when dim == 2 */
    double dx;                /* cell size h (cubic cells) */
    double gamma;             /* eq. (3) */
    double c0, c1;            /* eq. (4); the paper's runs use 1, 1 */
    int32_t visc_form;        /* MPM_VISC_* */
    int32_t bc[3][2];         /* MPM_BC_* */
    double inflow_rho, inflow_p, inflow_v[3];
    const uint8_t *obstacle_mask; /* HOST, one byte per cell, x fastest, non-zero = solid; NULL = none; copied */
    const double *node_normals;   /* HOST, [dim][N_n], outward unit normals at nodes; NULL = derive
                                     from the mask (windowed signed distance, reading A7); copied */
    uint64_t recycle_seed;    /* counter-based generator for particle recycling (reading A8) */
    double ppc_inflow;        /* recycled particle mass = inflow_rho h^dim / ppc_inflow */
    int32_t sort_every;       /* 0 = never re-order; k > 0 = cell-key re-ordering every k steps */
    int32_t variant;          /* MPM_VARIANT_* */
    int32_t device;           /* CUDA device ordinal */
    int32_t grid_accum;       /* MPM_ACCUM_* (this field was `reserved`, 0, in ABI version 1) */
    int32_t particle_stream;  /* MPM_STREAM_* (ABI version 2) */
    int32_t reserved2;        /* must be 0 */
    void *stream;             /* cudaStream_t; NULL = the legacy default stream */
    mpm_alloc_fn alloc;       /* NULL = cudaMalloc */
    mpm_free_fn free;         /* NULL = cudaFree */
    void *alloc_user;
} mpm_config;

/* kernel classes for the optional per-kernel timers (mpm_set_profiling) */
enum { MPM_K_P2G1 = 0, MPM_K_NODE1 = 1, MPM_K_G2P_P2G2 = 2, MPM_K_NODE2 = 3, MPM_K_UPDATE = 4, MPM_K_SORT = 5,
       MPM_K_MISC = 6, MPM_K_COUNT = 8 };

typedef struct mpm_stats {
    double t;                 /* simulated time */
    double dt_last;           /* dt of the last completed step */
    double dt_next;           /* alpha h / (vmax + cmax) from the last CFL reduction (eq. 29) */
    int64_t step;
    double vmax, cmax;        /* max_k max(|V'_k|, |Vbar_k|) and max_k sqrt(gamma P'_k / rho'_k) */
    int64_t n_recycled, n_clamped, n_negjac, n_nonfinite; /* cumulative counters; negjac = 1 + dt D <= 0 */
    double sum_mass, sum_momentum[3], sum_energy;         /* sum_k M, M V, M (E + |V|^2/2) of the current state */
    int64_t num_particles, num_nodes;
    int32_t nn[3];            /* nodes per axis */
    int32_t variant;          /* the kernel family actually in use */
    int64_t launches;         /* kernels launched by this handle so far */
    double kernel_ms[8];      /* with profiling on: device time per kernel class (MPM_K_*), CUDA events on `stream` */
    int64_t kernel_calls[8];  /* ... and how many timed launches (groups) went into it */
    /* ABI version 2 */
    int64_t n_cell_changes;   /* cumulative: particles whose cell changed in a step (Alg. 1 l.12); TILED family only */
    int64_t n_out_of_cell;    /* cumulative: particles a TILED kernel found outside their group's cell (debug counter of
                                 the exact-sort invariant; must be 0) */
    int64_t n_bad_dt;         /* cumulative: CFL steps with v_max + c_max = 0 or non-finite; such a step runs with dt = 0 */
} mpm_stats;

typedef struct mpm_handle mpm_handle;

/* Construct the solver for a grid (PAPER.md:299-300 step 2).  cfg: HOST.  *out receives the handle. */
MPM_API int mpm_create(const mpm_config *cfg, mpm_handle **out);

/* Copy n particles to the device (replaces any previous set; persistent id = load index) and perform the first
 * CFL reduction from the loaded state.  x, v: arrays of `dim` pointers; q may be NULL (Q = 0).  All data
 * pointers are HOST or DEVICE according to ptr_location; the pointer arrays themselves are HOST. */
MPM_API int mpm_load_particles(mpm_handle *h, int64_t n, const double *const *x, const double *const *v,
                       const double *mass, const double *rho, const double *e, const double *q,
                       int ptr_location);

/* Advance nsteps time steps of Algorithm 1.  dt > 0: fixed step.  dt <= 0: CFL mode, each step uses
 * dt = cfl * h / (vmax + cmax) from the latest device-side reduction (eq. 25/29); `cfl` is alpha.
 * dt_last: HOST, NULL = do not synchronise.  With dt_last != NULL the call returns MPM_E_NONFINITE if a non-finite
 * particle state or a CFL step without a positive finite dt (mpm_stats.n_bad_dt) has been seen so far. */
MPM_API int mpm_step(mpm_handle *h, double dt, double cfl, int32_t nsteps, double *dt_last);

/* Read particle fields selected by field_mask (MPM_P_*).  out: HOST array of pointers (see MPM_P_* order), each
 * to n doubles, HOST or DEVICE per ptr_location.  order 0 = by persistent id (load order), 1 = storage order. */
MPM_API int mpm_read_particles(mpm_handle *h, uint32_t field_mask, double *const *out, int order, int ptr_location);

/* Read one grid field (MPM_G_*) of the last completed step: out[ncomp][N_n], HOST or DEVICE. */
MPM_API int mpm_read_grid(mpm_handle *h, int field, double *out, int ptr_location);

/* Time, step, dt, CFL maxima, counters, conserved sums (computed on the device on demand).  out: HOST. */
MPM_API int mpm_get_stats(mpm_handle *h, mpm_stats *out);

/* Switch per-kernel-class CUDA-event timers on (1) / off (0); switching on clears the accumulated times.  With the
 * timers on, mpm_step brackets every kernel class with events on `stream` (a few microseconds of overhead per
 * launch) -- use it for roofline measurements, not inside a throughput measurement. */
MPM_API int mpm_set_profiling(mpm_handle *h, int on);

/* Last error message of this handle (or of the last failed mpm_create when h == NULL).  Never NULL. */
MPM_API const char *mpm_last_error(const mpm_handle *h);

MPM_API void mpm_destroy(mpm_handle *h);

MPM_API int mpm_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif
