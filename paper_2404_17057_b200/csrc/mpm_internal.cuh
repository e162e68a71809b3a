// mpm_internal.cuh -- internal types and device helpers of libmpm_b200.so (CUDA path; NOT shared with oracle/).
//
// Notation follows the paper (arXiv 2404.17057): particles k carry X, V, M, rho, E, Q;
// nodes i carry m, mv, f.  All arithmetic fp64.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/mpm.h"

// Checked build (nvcc -DMPM_CHECKED=1, libmpm_b200_checked.so): every index the tile kernels form -- particle slots, node
// indices, cell keys, window offsets, group and item records -- is tested against its bound and the kernel traps on a
// violation (the next CUDA call then fails loudly).  compute-sanitizer is not available on the GPU pool, so this build
// run through the parity tests is the memory-safety evidence (tests/test_gpu_parity.py::test_checked_build).
#if defined(MPM_CHECKED) && MPM_CHECKED
#define MPM_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define MPM_CHECK(cond) ((void)0)
#endif

namespace mpm {

// ---------------------------------------------------------------------------------------------- descriptors

struct GridDesc {
    int dim;
    int nc[3];        // cells per axis (1 on unused axes)
    int nn[3];        // nodes per axis: n (periodic) or n+1
    int per[3];       // periodic axis?
    int bc[3][2];     // MPM_BC_*
    double h, inv_h;  // cell size and its reciprocal (A4, A19)
    double L[3];      // domain lengths
    long long Nn, Nc;
    double gamma, c0, c1;
    int visc_form;
    int has_obstacle;
    // inflow / recycling (reading A8)
    double inflow_v[3];
    double inflow_rho, inflow_e, inflow_mass;
    int in_axis, in_side;   // first INFLOW face, -1 = none
    unsigned long long recycle_seed;
    // TILED family: cell keys are tile-major (see TileGeo); ntile = tiles per axis, Nkeys = size of the key space
    int tiled;
    int ntile[3];
    long long Nkeys;
    // TILED: every loaded particle has the same mass (bit for bit; with an inflow face, the recycled mass too): the
    // kernels then take M from here and neither read nor write the mass array (it stays filled with this value)
    int uniform_mass;
    double um;
    // TILED: node accumulators m, mv, f, mv2 are fp32 (mpm_config.grid_accum = MPM_ACCUM_FP32)
    int acc32;
    // TILED: particle fields are streamed with bulk asynchronous copies + mbarriers instead of per-thread cp.async
    // (mpm_config.particle_stream = MPM_STREAM_BULK)
    int bulk_stream;
    // TILED: which scatters accumulate in a shared-memory tile by cell colour (mpm_config.p2g_mode, MPM_P2G_* bits)
    int p2g_mode;
    // slab decomposition: this grid is cells [slab_offset, slab_offset + nc[dim-1]) of slab_global_n along the last axis
    // (0 = not a slab); only the recycling position needs to know
    int slab_global_n, slab_offset;
    int has_open;       // some face is MPM_BC_OPEN (particles beyond it are out of their cell until the caller hands them over)
    int quadratic;      // ATOMIC family: quadratic B-spline basis instead of Q1 (mpm_config.basis), periodic grids only
    int colour_major;   // layout of the cell numbering inside a tile (TileGeo): 1 when p2g_mode != 0
    // TILED: allocated slots per particle array and capacities of the group / item lists (bounds of the checked build)
    long long slots, max_groups, max_items;
    // TILED: the persistent particle ids travel with the particles (mpm_config.particle_ids; always with an INFLOW face, whose
    // recycling generator is keyed on them, reading A8).  0: the sweeps neither read nor write the id arrays
    int track_ids;
};

// TILED family: the grid is cut into tiles of T0 x T1 (x T2) cells; the cell key is (tile index, cell inside the
// tile): tiles x fastest, cells inside a tile x fastest or colour-major (see below), so that the particles of one tile are contiguous
// in the cell-sorted order (PAPER.md:745-748 applied per tile) and one thread block can keep the tile's (T+1)^d nodes in
// shared memory.
template <int DIM>
struct TileGeo {
    static constexpr int LT0 = (DIM == 3) ? 3 : 4;
    static constexpr int LT1 = (DIM == 3) ? 3 : 4;
    static constexpr int LT2 = (DIM == 3) ? 2 : 0;
    static constexpr int T0 = 1 << LT0, T1 = 1 << LT1, T2 = 1 << LT2;
    static constexpr int LTC = LT0 + LT1 + LT2;
    static constexpr int TC = 1 << LTC;                      // cells per tile
    static constexpr int N0 = T0 + 1, N1 = T1 + 1, N2 = (DIM == 3) ? T2 + 1 : 1;
    static constexpr int NN = N0 * N1 * N2;                  // nodes per tile
    // Numbering of the cells inside a tile (the low LTC bits of the cell key), two layouts:
    //   natural (default): x fastest, then y, then z;
    //   colour-major (cm, used when a scatter accumulates by cell colour, mpm_config.p2g_mode): colour = parities of the
    //     tile-local cell coordinates (the 2^d colouring the paper proposes for an atomics-free P2G: cells
    //     of one colour share no node), then the position among the cells of that colour, x fastest.  Consecutive keys --
    //     and hence the groups a block works on in one pass -- then belong to one colour: their corner nodes are disjoint.
    static constexpr int NCOL = 1 << DIM;                    // colours
    static constexpr int LCC = LTC - DIM;                    // log2(cells per colour)
    __host__ __device__ static constexpr int local_of(int lx, int ly, int lz, bool cm)
    {
        return cm ? ((((lx & 1) | ((ly & 1) << 1) | ((DIM == 3 ? (lz & 1) : 0) << 2)) << LCC) |
                     (lx >> 1) | ((ly >> 1) << (LT0 - 1)) | ((DIM == 3 ? (lz >> 1) : 0) << (LT0 + LT1 - 2)))
                  : (lx | (ly << LT0) | ((DIM == 3 ? lz : 0) << (LT0 + LT1)));
    }
    __host__ __device__ static constexpr int colour_of(int local) { return local >> LCC; }      // colour-major layout only
    __host__ __device__ static constexpr int lx_of(int local, bool cm)
    {
        return cm ? ((((local & ((1 << (LT0 - 1)) - 1))) << 1) | ((local >> LCC) & 1)) : (local & (T0 - 1));
    }
    __host__ __device__ static constexpr int ly_of(int local, bool cm)
    {
        return cm ? ((((local >> (LT0 - 1)) & ((1 << (LT1 - 1)) - 1)) << 1) | ((local >> (LCC + 1)) & 1)) : ((local >> LT0) & (T1 - 1));
    }
    __host__ __device__ static constexpr int lz_of(int local, bool cm)
    {
        return DIM != 3 ? 0
               : cm ? ((((local >> (LT0 + LT1 - 2)) & ((1 << (LT2 > 0 ? LT2 - 1 : 0)) - 1)) << 1) | ((local >> (LCC + 2)) & 1))
                    : (local >> (LT0 + LT1));
    }
    // tile-local node index of the cell's corner 0
    __host__ __device__ static constexpr int node0_of(int local, bool cm)
    {
        return lx_of(local, cm) + N0 * (ly_of(local, cm) + N1 * lz_of(local, cm));
    }
};

// Order of the tiles = order of their particles in memory = order in which the blocks of the tile kernels are scheduled:
// x fastest over the whole grid.  (Measured in round 2, profiles/r02_experiments.md section 7: numbering the tiles in compact
// super-tiles of 4 x 4 x 4, so that the node planes neighbouring tiles share are still in L2 when the second tile needs
// them, changes neither kernel's time on configs 4 and 5.)
template <int DIM>
__host__ __device__ __forceinline__ int tile_index(const GridDesc &gd, int tx, int ty, int tz)
{
    int tile = tx + gd.ntile[0] * ty;
    if (DIM == 3) tile += gd.ntile[0] * gd.ntile[1] * tz;
    return tile;
}
template <int DIM>
__host__ __device__ __forceinline__ void tile_coords(const GridDesc &gd, int tile, int t[3])
{
    t[0] = tile % gd.ntile[0];
    t[1] = (tile / gd.ntile[0]) % gd.ntile[1];
    t[2] = (DIM == 3) ? tile / (gd.ntile[0] * gd.ntile[1]) : 0;
}

// cm: colour-major numbering inside the tile (a compile-time constant in the tile kernels, gd.colour_major elsewhere)
template <int DIM>
__host__ __device__ __forceinline__ int tiled_key_of_cell(const GridDesc &gd, const int c[DIM], bool cm)
{
    using TG = TileGeo<DIM>;
    const int tile = tile_index<DIM>(gd, c[0] >> TG::LT0, c[1] >> TG::LT1, DIM == 3 ? (c[DIM - 1] >> TG::LT2) : 0);
    const int local = TG::local_of(c[0] & (TG::T0 - 1), c[1] & (TG::T1 - 1), DIM == 3 ? (c[DIM - 1] & (TG::T2 - 1)) : 0, cm);
    return (tile << TG::LTC) | local;
}
template <int DIM>
__host__ __device__ __forceinline__ int tiled_key_of_cell(const GridDesc &gd, const int c[DIM])
{
    return tiled_key_of_cell<DIM>(gd, c, gd.colour_major != 0);
}

template <int DIM>
__host__ __device__ __forceinline__ void tiled_cell_of_key(const GridDesc &gd, int key, int c[DIM])
{
    using TG = TileGeo<DIM>;
    const int tile = key >> TG::LTC, local = key & (TG::TC - 1);
    const bool cm = gd.colour_major != 0;
    int t[3];
    tile_coords<DIM>(gd, tile, t);
    c[0] = (t[0] << TG::LT0) | TG::lx_of(local, cm);
    c[1] = (t[1] << TG::LT1) | TG::ly_of(local, cm);
    if (DIM == 3) c[DIM - 1] = (t[2] << TG::LT2) | TG::lz_of(local, cm);
}

// particle SoA.  P, Vbar, A, grad V are transient and never stored.
struct PArr {
    double *x[3];
    double *v[3];
    double *m, *rho, *e, *q;
    int *id;   // persistent id = load index
};

// node SoA.  vbar = mv'/m, acc = f/m, v2 = mv2/m are the node velocities the gathers of the ATOMIC family read (ratio := 0
// where m = 0, A5), component-major; NULL in the TILED family, which forms them per tile node in shared memory.
struct GArr {
    double *m;
    double *mv[3], *f[3], *mv2[3];
    double *vbar[3], *acc[3], *v2[3];
    const unsigned char *flag;   // 1 = obstacle node, NULL when there is no obstacle
    const double *normal[3];
};

// device-resident scalars of the time loop: nothing in mpm_step needs the host
struct DevScalars {
    double dt;          // dt of the step being executed
    double t;
    double dt_next;     // alpha h / (vmax + cmax)
    double alpha;
    double dt_fixed;    // > 0: fixed-step mode
    double vmax, cmax;  // finalised maxima of the last reduction
    unsigned long long vmax_bits, cmax_bits;   // running maxima (non-negative doubles compared as integers)
    long long step;
    unsigned long long n_recycled, n_clamped, n_negjac, n_nonfinite;
    // cumulative: particles that changed cell in a step (l.12), particles found outside their group's cell by a tile
    // kernel (must stay 0: the TILED family's weights rely on the exact sort), steps whose CFL dt was not a positive
    // finite number (v_max + c_max = 0 or non-finite: dt := 0 for that step)
    unsigned long long n_cell_changes, n_out_of_cell, n_bad_dt;
    unsigned long long n_left_slab;   // cumulative: particles that ended a step beyond an MPM_BC_OPEN face (to be handed over)
    double sum_mass, sum_mom[3], sum_energy;   // filled by the stats reduction on demand
};

// ---------------------------------------------------------------------------------------------- device helpers

// Cell and local coordinate of a position along one axis (readings A6, A19).  The product is rounded on
// its own (no contraction into s - c): every kernel that bins a position gets the same cell for it.
__device__ __forceinline__ void cell_1d(double X, double inv_h, int ncell, int &c, double &xi)
{
    double s = __dmul_rn(X, inv_h);
    int ci = (int)floor(s);
    ci = max(0, min(ci, ncell - 1));
    c = ci;
    xi = s - (double)ci;
}

template <int DIM>
__device__ __forceinline__ void particle_cell(const GridDesc &gd, const double X[DIM], int c[DIM], double xi[DIM])
{
#pragma unroll
    for (int a = 0; a < DIM; ++a) cell_1d(X[a], gd.inv_h, gd.nc[a], c[a], xi[a]);
}

// global node index of corner b (bit a of ib = b_a) of cell c; periodic: node n == node 0 (A11)
template <int DIM>
__device__ __forceinline__ long long corner_node(const GridDesc &gd, const int c[DIM], int ib)
{
    long long idx = 0;
    long long stride = 1;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int i = c[a] + ((ib >> a) & 1);
        if (gd.per[a] && i == gd.nc[a]) i = 0;
        idx += stride * (long long)i;
        stride *= (long long)gd.nn[a];
    }
    return idx;
}

// phi_b = prod_a w_a(b_a), w_a(0) = 1 - xi_a, w_a(1) = xi_a
template <int DIM>
__device__ __forceinline__ double corner_phi(const double xi[DIM], int ib)
{
    double p = 1.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) p *= ((ib >> a) & 1) ? xi[a] : (1.0 - xi[a]);
    return p;
}

// d_a phi_b = (+-1/h) prod_{a' != a} w_a'(b_a')
template <int DIM>
__device__ __forceinline__ double corner_dphi(const double xi[DIM], int ib, int a, double inv_h)
{
    double q = ((ib >> a) & 1) ? inv_h : -inv_h;
#pragma unroll
    for (int a2 = 0; a2 < DIM; ++a2)
        if (a2 != a) q *= ((ib >> a2) & 1) ? xi[a2] : (1.0 - xi[a2]);
    return q;
}

// splitmix64 output function (Steele, Lea & Flood 2014), restated here independently of the oracle (A8)
__host__ __device__ __forceinline__ unsigned long long mix64(unsigned long long z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__host__ __device__ __forceinline__ double recycle_uniform(unsigned long long seed, long long id, long long step, int j)
{
    unsigned long long z = mix64(seed);
    z = mix64(z ^ (unsigned long long)id);
    z = mix64(z ^ (unsigned long long)step);
    z = mix64(z ^ (unsigned long long)j);
    return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}

__device__ __forceinline__ void atomic_max_nonneg(unsigned long long *addr, double v)
{
    // non-negative doubles order like their bit patterns; NaN (0x7ff8...) wins, which is what we want to see
    atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

// cell-sorted order: off[c] .. off[c+1] are the particles of cell c; every cell is cut into groups of <= 2^dim particles.
// One 16-byte record per group: {first particle, count, linear cell, packed cell coordinates}.
struct SortedMap {
    const int4 *groups;     // [n_groups]
    const int *n_groups;    // device scalar
};

// ---------------------------------------------------------------------------------------------- launchers

// ATOMIC family (one thread per particle, global fp64 atomics; any particle order) -- mpm_kernels_atomic.cu
void launch_p2g1_atomic(const GridDesc &gd, const PArr &p, const GArr &g, long long n, cudaStream_t s);
void launch_g2p_p2g2_atomic(const GridDesc &gd, const PArr &p, const GArr &g, const DevScalars *sc, long long n,
                            cudaStream_t s);
void launch_update_atomic(const GridDesc &gd, const PArr &p, const GArr &g, DevScalars *sc, long long n,
                          cudaStream_t s);

// TILED family (tile-major cell order, even-aligned cell slots, tile nodes in shared memory) -- mpm_kernels_tiled.cu
// Alg. 1 l.12 bookkeeping in one kernel: per-key counts -> even-aligned slot offsets off[Nkeys + 1], group records, work
// items of the tile kernels (one block per item = <= Chunk::GROUPS groups of one tile).  `state`: scratch of
// cell_map_state_bytes(gd) bytes (zeroed by the launcher).
size_t cell_map_state_bytes(const GridDesc &gd);
void launch_cell_map_tiled(const GridDesc &gd, const int *count, int *off, int4 *groups, int *n_groups, int4 *items, int *n_items,
                           void *state, cudaStream_t s);
// P2G#1 after a load (every later step gets it from launch_update_tiled of the step before); g.m, g.mv, g.f must be zero
void launch_p2g1_tiled(const GridDesc &gd, const PArr &p, const GArr &g, const SortedMap &map, long long max_groups, cudaStream_t s);
// flag[0] |= 1 if any of m[0..n) differs from m[0] bit for bit (flag zeroed by the caller); fill: m[0..n) = value
void launch_mass_differs(const double *m, long long n, int *flag, cudaStream_t s);
void launch_fill(double *m, long long n, double value, cudaStream_t s);
// fp32 accumulators (node-major: src32.m = nm[N_n][8], src32.mv2[0] = v2[N_n][4]) widened into the component-major fp64 arrays of
// dst64 for mpm_read_grid
void launch_widen(const GridDesc &gd, const GArr &src32, const GArr &dst64, cudaStream_t s);
// dst[i] += src[i], i < n (halo sum-exchange of a node plane)
void launch_add_into(double *dst, const double *src, long long n, cudaStream_t s);
long long max_items_tiled(const GridDesc &gd, long long max_groups);   // upper bound of the item count (launch size)
// g: the node accumulators m, mv, f of this step (raw P2G#1) and mv2; the kernels apply l.4-5 / l.9 while staging a tile
void launch_g2p_p2g2_tiled(const GridDesc &gd, const PArr &p, const GArr &g, const DevScalars *sc,
                           const SortedMap &map, const int4 *items, const int *n_items, long long max_items, int *count,
                           unsigned *dest, cudaStream_t s);
// update + re-ordering + P2G#1 of the next step into g_next.m, g_next.mv, g_next.f (zeroed by the caller).  store_q:
// write Q' to memory (only needed when the state can be read back or re-loaded before the next step: the fused P2G#1
// has already consumed it)
void launch_update_tiled(const GridDesc &gd, const PArr &p, const PArr &q, const GArr &g, DevScalars *sc,
                         const SortedMap &map, const int4 *items, const int *n_items, long long max_items, const int *off_new,
                         const unsigned *dest, const GArr &g_next, bool store_q, cudaStream_t s);
// dst[id] = src[slot] for every occupied slot; with coff (exclusive scan of the per-key counts) and off (slot offsets):
// dst[compact storage index] = src[slot] instead
void launch_gather_by_id_groups(const double *src, const int *id, double *dst, const SortedMap &map, long long max_groups,
                                const int *coff, const int *off, cudaStream_t s);
void launch_stats_reduce_groups(const GridDesc &gd, const PArr &p, DevScalars *sc, const SortedMap &map, long long max_groups,
                                cudaStream_t s);

// diagnostics (mpm_read_grid RHO_GRID / E_GRID, reading A18): num[i] = sum_k M a phi_i, den[i] = sum_k M phi_i with a = rho or E,
// then num[i] = num[i] / den[i] (0 where den = 0).  num, den: zeroed by the caller.  map.groups == NULL: particles 0 .. n-1.
void launch_grid_diagnostic(const GridDesc &gd, const PArr &p, const double *field, double *num, double *den, long long n,
                            const SortedMap &map, long long max_groups, cudaStream_t s);

// node kernels -- mpm_kernels_grid.cu
void launch_grid_clear(const GridDesc &gd, const GArr &g, cudaStream_t s);
// zero_mv2: also reset mv2 for l.8 (false when the kernel only replays l.4-5 for mpm_read_grid)
void launch_node1(const GridDesc &gd, const GArr &g, const DevScalars *sc, cudaStream_t s, bool zero_mv2 = true);
void launch_node2(const GridDesc &gd, const GArr &g, cudaStream_t s);

// time loop scalars -- mpm_kernels_grid.cu
void launch_begin_step(DevScalars *sc, double h, bool have_particles, cudaStream_t s);
void launch_end_step(DevScalars *sc, double h, cudaStream_t s);
void launch_initial_cfl(const GridDesc &gd, const PArr &p, DevScalars *sc, long long n, cudaStream_t s);
void launch_stats_reduce(const GridDesc &gd, const PArr &p, DevScalars *sc, long long n, cudaStream_t s);

// re-ordering: cell key, histogram + rank, exclusive scan, permutation -- mpm_sort.cu
void launch_iota(int *id, long long n, cudaStream_t s);
void launch_key_rank(const GridDesc &gd, const PArr &p, int *key, int *rank, int *count, long long n, cudaStream_t s);
void launch_exclusive_scan(int *data, long long n, int *aux, cudaStream_t s);   // in place, aux >= n/4096 + 2 ints
// out = exclusive scan of in (round_even: of in rounded up to even); in == out allowed
void launch_exclusive_scan_from(const int *in, int *out, long long n, int *aux, bool round_even, cudaStream_t s);
void launch_permute(const GridDesc &gd, const PArr &src, const PArr &dst, const int *key, const int *rank,
                    const int *offset, long long n, cudaStream_t s);
void launch_gather_by_id(const double *src, const int *id, double *dst, long long n, cudaStream_t s);

}  // namespace mpm
