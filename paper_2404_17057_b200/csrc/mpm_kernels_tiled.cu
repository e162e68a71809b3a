// mpm_kernels_tiled.cu -- TILED kernel family: the SORTED family's lane groups (one cell per group, butterfly
// reductions, fused re-ordering) re-organised around shared-memory grid tiles.
//
//   * cell keys are tile-major (TileGeo: 8 x 8 x 4 cells in 3D, 16 x 16 in 2D), so the particles of one tile are one
//     contiguous run of the cell-sorted order (the grid-to-particle connectivity of PAPER.md:745-748, per tile);
//   * every cell's slot range starts at an EVEN slot (an odd cell leaves one unused slot), so that lane l of a group
//     owns the two consecutive particles first + 2l, first + 2l + 1 and fetches each field with ONE aligned 128-bit load;
//   * a thread block works on a chunk of consecutive groups, cut into segments at tile boundaries.  Per segment:
//       gathers (Alg. 1 l.6, l.10): the tile's (T+1)^d node values are loaded once into shared memory and every lane
//         reads its 2^d corners from there (no per-group staging, no redundant global node loads);
//       scatters (l.3, l.8): group totals go into a shared-memory accumulator tile with fp64 atomicAdd (a CAS loop on
//         sm_100a, measured 6 clk per conflict-free warp operation against 20 clk for a global RED), and the tile is
//         flushed with ONE global fp64 reduction per touched node and channel: ~1.5 RED per particle instead of 7 + 3.
//   * Alg. 1 l.12 is fused as in the SORTED family: the gather kernel ranks every particle in its new cell, a scan of
//     the (even-rounded) counts gives the new slot offsets, the update kernel writes straight to the sorted slot.
#include "mpm_lane_groups.cuh"

#ifndef MPM_SCATTER_GLOBAL
#define MPM_SCATTER_GLOBAL 0   // 1: group totals go straight to global memory (REDG), no shared accumulator tile
#endif
#ifndef MPM_MINB
#define MPM_MINB 2   // resident blocks per SM the particle kernels are compiled for (register budget)
#endif

namespace mpm {

namespace {

using namespace lg;

template <int DIM>
struct TK {
    using TG = TileGeo<DIM>;
    static constexpr int NB = 1 << DIM, LG = NB / 2, GPB = kBlock / LG;
    static constexpr int CG = 8 * GPB;                      // groups per chunk (a multiple of the groups per iteration)
    static constexpr int NA = 2 * DIM;                      // doubles per node in the (vbar, acc) tile
    static constexpr int NBS = (DIM == 3) ? 4 : 2;          // doubles per node in the v2 tile (padded to 16 bytes)
    static constexpr int NN = TG::NN;
};

template <int DIM>
__device__ __forceinline__ void tile_origin(const GridDesc &gd, int tile, int o[DIM])
{
    using TG = TileGeo<DIM>;
    o[0] = (tile % gd.ntile[0]) << TG::LT0;
    o[1] = ((tile / gd.ntile[0]) % gd.ntile[1]) << TG::LT1;
    if (DIM == 3) o[DIM - 1] = (tile / (gd.ntile[0] * gd.ntile[1])) << TG::LT2;
}

// global node index of local node ln of the tile with origin o; -1 if the node lies outside the grid (partial tile).
// Periodic axes: node n == node 0 (A11).
template <int DIM>
__device__ __forceinline__ int tile_global_node(const GridDesc &gd, const int o[DIM], int ln)
{
    using TG = TileGeo<DIM>;
    int i[3] = { ln % TG::N0, (ln / TG::N0) % TG::N1, ln / (TG::N0 * TG::N1) };
    int idx = 0, stride = 1;
    bool ok = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int gi = o[a] + i[a];
        if (gi > gd.nc[a]) ok = false;
        if (gd.per[a] && gi == gd.nc[a]) gi = 0;
        idx += stride * gi;
        stride *= gd.nn[a];
    }
    return ok ? idx : -1;
}

// local node index of corner 0 of the cell with coordinates c (the tile origin is a multiple of the tile size)
template <int DIM>
__device__ __forceinline__ int tile_local_base(const int c[DIM])
{
    using TG = TileGeo<DIM>;
    int ln = (c[0] & (TG::T0 - 1)) + TG::N0 * (c[1] & (TG::T1 - 1));
    if (DIM == 3) ln += TG::N0 * TG::N1 * (c[DIM - 1] & (TG::T2 - 1));
    return ln;
}

// first group index past the segment that starts at group seg_begin: the end of its tile or of the chunk
template <int DIM>
__device__ __forceinline__ int segment_end(const SortedMap &map, int seg_begin, int g_end, int &tile)
{
    using TG = TileGeo<DIM>;
    const int key0 = __ldg(&map.groups[seg_begin].z);
    tile = key0 >> TG::LTC;
    return min(g_end, __ldg(&map.goff[(tile + 1) << TG::LTC]));
}

__device__ __forceinline__ double2 ld2(const double *__restrict__ p, long long k, bool ok)
{
    return ok ? __ldg(reinterpret_cast<const double2 *>(p + k)) : make_double2(0.0, 0.0);
}

template <int DIM>
__device__ __forceinline__ int tiled_key_of_position(const GridDesc &gd, const double X[DIM])
{
    int c[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double xi;
        cell_1d(X[a], gd.inv_h, gd.nc[a], c[a], xi);
    }
    return tiled_key_of_cell<DIM>(gd, c);
}

// flush one accumulator channel of the tile: one global fp64 reduction per touched node (the data race
// of P2G is closed with atomics; here once per tile and node instead of once per particle and node)
template <int DIM>
__device__ __forceinline__ void flush_channel(const GridDesc &gd, const int o[DIM], const double *s_ch, double *__restrict__ dst)
{
    for (int ln = threadIdx.x; ln < TK<DIM>::NN; ln += kBlock) {
        const double v = s_ch[ln];
        if (v != 0.0) {
            const int gn = tile_global_node<DIM>(gd, o, ln);
            if (gn >= 0) atomicAdd(dst + gn, v);
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.3
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_p2g1_tiled(GridDesc gd, PArr p, const double *__restrict__ Sarr, GArr g, SortedMap map)
{
    using K = TK<DIM>;
    constexpr int NB = K::NB, LG = K::LG, GPB = K::GPB, NN = K::NN, NCH = 1 + 2 * DIM;
    __shared__ double s_acc[NCH * NN];
    const int n_groups = *map.n_groups;
    const int l = threadIdx.x % LG;
    for (int chunk = blockIdx.x; (long long)chunk * K::CG < n_groups; chunk += gridDim.x) {
        const int g_begin = chunk * K::CG, g_end = min(g_begin + K::CG, n_groups);
        int seg_begin = g_begin;
        while (seg_begin < g_end) {
            int tile;
            const int seg_end = segment_end<DIM>(map, seg_begin, g_end, tile);
            int o[DIM];
            tile_origin<DIM>(gd, tile, o);
#if !MPM_SCATTER_GLOBAL
            for (int i = threadIdx.x; i < NCH * NN; i += kBlock) s_acc[i] = 0.0;
            __syncthreads();
#endif
            int gidx = seg_begin + threadIdx.x / LG;
            Group next = fetch_group(map.groups, gidx, seg_end);
            for (int gb = seg_begin; gb < seg_end; gb += GPB, gidx += GPB) {
                const Group grp = next;
                next = fetch_group(map.groups, (long long)gidx + GPB, seg_end);
                int c[DIM];
                unpack_coords<DIM>(grp.cpack, c);
                const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
                const long long k0 = (long long)grp.first + 2 * l;
                double X[2][DIM], V[2][DIM], M[2], S[2];
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    const double2 tx = ld2(p.x[a], k0, valid[0]), tv = ld2(p.v[a], k0, valid[0]);
                    X[0][a] = tx.x; X[1][a] = valid[1] ? tx.y : 0.0;
                    V[0][a] = tv.x; V[1][a] = valid[1] ? tv.y : 0.0;
                }
                {
                    const double2 tm = ld2(p.m, k0, valid[0]), ts = ld2(Sarr, k0, valid[0]);
                    M[0] = tm.x; M[1] = valid[1] ? tm.y : 0.0;
                    S[0] = ts.x; S[1] = valid[1] ? ts.y : 0.0;
                }
                double w[2][NB];
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    double xi[DIM];
                    const bool fast = valid[i] && local_coords<DIM>(gd, X[i], c, xi);
                    if (valid[i] && !fast) { slow_p2g1<DIM>(gd, g, X[i], V[i], M[i], S[i]); M[i] = 0.0; S[i] = 0.0; }
                    if (fast) swizzled_weights<DIM>(xi, l, w[i]);
                    else {
#pragma unroll
                        for (int r = 0; r < NB; ++r) w[i][r] = 0.0;
                    }
                }
                // lane totals per corner, then group totals: channels M, M V_a, S (see mpm_kernels_sorted.cu)
                double tot[DIM + 2][2];
#pragma unroll
                for (int ch = 0; ch < DIM + 2; ++ch) {
                    double pay[2];
#pragma unroll
                    for (int i = 0; i < 2; ++i) pay[i] = (ch == 0) ? M[i] : (ch == DIM + 1) ? S[i] : M[i] * V[i][ch - 1];
                    double v[NB];
#pragma unroll
                    for (int r = 0; r < NB; ++r) v[r] = fma(pay[1], w[1][r], pay[0] * w[0][r]);
                    butterfly<DIM>(v);
                    tot[ch][0] = v[0];
                    tot[ch][1] = v[LG];
                }
                double F[DIM][2];
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        double other;
                        if ((1 << a) < LG) other = shfl_xor_d(tot[DIM + 1][q], 1 << a);
                        else other = tot[DIM + 1][q ^ 1];
                        const int b = l + q * LG;
                        const double pair = (tot[DIM + 1][q] + other) * gd.inv_h;
                        F[a][q] = ((b >> a) & 1) ? pair : -pair;
                    }
                }
                if (grp.cnt > 0) {
#if MPM_SCATTER_GLOBAL
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const int node = corner_node_i<DIM>(gd, c, l + q * LG);
                        atomicAdd(&g.m[node], tot[0][q]);
#pragma unroll
                        for (int a = 0; a < DIM; ++a) {
                            atomicAdd(&g.mv[a][node], tot[1 + a][q]);
                            atomicAdd(&g.f[a][node], F[a][q]);
                        }
                    }
#else
                    const int base = tile_local_base<DIM>(c);
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        const int b = l + q * LG;
                        const int ln = base + (b & 1) + TileGeo<DIM>::N0 * ((b >> 1) & 1) +
                                       ((DIM == 3) ? TileGeo<DIM>::N0 * TileGeo<DIM>::N1 * ((b >> 2) & 1) : 0);
                        atomicAdd(&s_acc[ln], tot[0][q]);
#pragma unroll
                        for (int a = 0; a < DIM; ++a) {
                            atomicAdd(&s_acc[(1 + a) * NN + ln], tot[1 + a][q]);
                            atomicAdd(&s_acc[(1 + DIM + a) * NN + ln], F[a][q]);
                        }
                    }
#endif
                }
            }
#if !MPM_SCATTER_GLOBAL
            __syncthreads();
            flush_channel<DIM>(gd, o, s_acc, g.m);
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                flush_channel<DIM>(gd, o, s_acc + (1 + a) * NN, g.mv[a]);
                flush_channel<DIM>(gd, o, s_acc + (1 + DIM + a) * NN, g.f[a]);
            }
            __syncthreads();
#endif
            seg_begin = seg_end;
        }
    }
}

// load the (vbar, acc) node values of a tile: node-major global array na[node][2 DIM] -> s_a[local node][2 DIM]
template <int DIM>
__device__ __forceinline__ void load_tile_a(const GridDesc &gd, const int o[DIM], const double *__restrict__ na, double *s_a)
{
    constexpr int NN = TK<DIM>::NN, U = DIM;    // double2 units per node
    for (int i = threadIdx.x; i < NN * U; i += kBlock) {
        const int ln = i / U, j = i % U;
        const int gn = tile_global_node<DIM>(gd, o, ln);
        double2 t = make_double2(0.0, 0.0);
        if (gn >= 0) t = __ldg(reinterpret_cast<const double2 *>(na + (long long)gn * (2 * DIM)) + j);
        reinterpret_cast<double2 *>(s_a)[i] = t;
    }
}

// v2 = mv2/m of a tile: nb[node][DIM] -> s_b[local node][NBS]
template <int DIM>
__device__ __forceinline__ void load_tile_b(const GridDesc &gd, const int o[DIM], const double *__restrict__ nb, double *s_b)
{
    constexpr int NN = TK<DIM>::NN, NBS = TK<DIM>::NBS;
    for (int ln = threadIdx.x; ln < NN; ln += kBlock) {
        const int gn = tile_global_node<DIM>(gd, o, ln);
#pragma unroll
        for (int a = 0; a < NBS; ++a) s_b[ln * NBS + a] = (gn >= 0 && a < DIM) ? __ldg(nb + (long long)gn * DIM + a) : 0.0;
    }
}

// phi-weighted gather of vbar, acc from the shared tile
template <int DIM>
__device__ __forceinline__ void gather_tile_a(const double *s_a, int base, const double w[1 << DIM], double Vb[DIM], double A[DIM])
{
    using TG = TileGeo<DIM>;
    double out[2 * DIM];
#pragma unroll
    for (int cc = 0; cc < 2 * DIM; ++cc) out[cc] = 0.0;
#pragma unroll
    for (int b = 0; b < (1 << DIM); ++b) {
        const int ln = base + (b & 1) + TG::N0 * ((b >> 1) & 1) + ((DIM == 3) ? TG::N0 * TG::N1 * ((b >> 2) & 1) : 0);
        const double2 *row = reinterpret_cast<const double2 *>(s_a + ln * (2 * DIM));
#pragma unroll
        for (int j = 0; j < DIM; ++j) {
            const double2 t = row[j];
            out[2 * j] = fma(w[b], t.x, out[2 * j]);
            out[2 * j + 1] = fma(w[b], t.y, out[2 * j + 1]);
        }
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) { Vb[a] = out[a]; A[a] = out[DIM + a]; }
}

// D = sum_b sum_a v2_a(b) d_a phi_b (eq. 19, trace only: PAPER.md:362-364) from the shared v2 tile
template <int DIM>
__device__ __forceinline__ double gather_divergence(const double *s_b, int base, const double xi[DIM], double inv_h)
{
    using TG = TileGeo<DIM>;
    constexpr int NBS = TK<DIM>::NBS;
    double wa[DIM][2];
#pragma unroll
    for (int a = 0; a < DIM; ++a) { wa[a][0] = 1.0 - xi[a]; wa[a][1] = xi[a]; }
    double Da[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) Da[a] = 0.0;
#pragma unroll
    for (int b = 0; b < (1 << DIM); ++b) {
        const int ln = base + (b & 1) + TG::N0 * ((b >> 1) & 1) + ((DIM == 3) ? TG::N0 * TG::N1 * ((b >> 2) & 1) : 0);
        double v2[DIM];
        const double2 t = *reinterpret_cast<const double2 *>(s_b + ln * NBS);
        v2[0] = t.x; v2[1] = t.y;
        if (DIM == 3) v2[DIM - 1] = s_b[ln * NBS + 2];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            double q = 1.0;
#pragma unroll
            for (int a2 = 0; a2 < DIM; ++a2)
                if (a2 != a) q *= wa[a2][(b >> a2) & 1];
            Da[a] = ((b >> a) & 1) ? fma(q, v2[a], Da[a]) : fma(-q, v2[a], Da[a]);
        }
    }
    double D = 0.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) D += Da[a];
    return D * inv_h;
}

// Alg. 1 l.11 for one particle (see lg::move_particle); the persistent id is only needed by the recycling generator
// (A8), so it is fetched only when a particle actually leaves through an OUTFLOW face.
template <int DIM>
__device__ __forceinline__ void move_particle_lazy_id(const GridDesc &gd, const double X[DIM], const double Vb[DIM], double dt,
                                                      const int *__restrict__ idarr, long long k, long long step, double Xn[DIM])
{
    bool leaves = false;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const double x = fma(dt, Vb[a], X[a]);
        if (!gd.per[a]) {
            if (x < 0.0 && gd.bc[a][0] == MPM_BC_OUTFLOW) leaves = true;
            if (x > gd.L[a] && gd.bc[a][1] == MPM_BC_OUTFLOW) leaves = true;
        }
    }
    const long long id = (leaves && gd.in_axis >= 0) ? (long long)idarr[k] : 0;
    bool recycled;
    int nclamp;
    move_particle<DIM>(gd, X, Vb, dt, id, step, Xn, recycled, nclamp);
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.6-8 (+ l.11-12 bookkeeping)
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_g2p_p2g2_tiled(GridDesc gd, PArr p, GArr g, const double *__restrict__ na,
                                                           const DevScalars *__restrict__ sc, SortedMap map,
                                                           int *__restrict__ count, unsigned long long *__restrict__ dest)
{
    using K = TK<DIM>;
    using TG = TileGeo<DIM>;
    constexpr int NB = K::NB, LG = K::LG, GPB = K::GPB, NN = K::NN;
    __shared__ __align__(16) double s_a[NN * K::NA];
    __shared__ double s_acc[DIM * NN];
    const int n_groups = *map.n_groups;
    const double dt = sc->dt;
    const long long step = sc->step;
    const int l = threadIdx.x % LG;
    for (int chunk = blockIdx.x; (long long)chunk * K::CG < n_groups; chunk += gridDim.x) {
        const int g_begin = chunk * K::CG, g_end = min(g_begin + K::CG, n_groups);
        int seg_begin = g_begin;
        while (seg_begin < g_end) {
            int tile;
            const int seg_end = segment_end<DIM>(map, seg_begin, g_end, tile);
            int o[DIM];
            tile_origin<DIM>(gd, tile, o);
            load_tile_a<DIM>(gd, o, na, s_a);
#if !MPM_SCATTER_GLOBAL
            for (int i = threadIdx.x; i < DIM * NN; i += kBlock) s_acc[i] = 0.0;
#endif
            __syncthreads();
            int gidx = seg_begin + threadIdx.x / LG;
            Group next = fetch_group(map.groups, gidx, seg_end);
            for (int gb = seg_begin; gb < seg_end; gb += GPB, gidx += GPB) {
                const Group grp = next;
                next = fetch_group(map.groups, (long long)gidx + GPB, seg_end);
                int c[DIM];
                unpack_coords<DIM>(grp.cpack, c);
                const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
                const long long k0 = (long long)grp.first + 2 * l;
                double X[2][DIM], V[2][DIM], M[2];
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    const double2 tx = ld2(p.x[a], k0, valid[0]), tv = ld2(p.v[a], k0, valid[0]);
                    X[0][a] = tx.x; X[1][a] = valid[1] ? tx.y : 0.0;
                    V[0][a] = tv.x; V[1][a] = valid[1] ? tv.y : 0.0;
                }
                {
                    const double2 tm = ld2(p.m, k0, valid[0]);
                    M[0] = tm.x; M[1] = valid[1] ? tm.y : 0.0;
                }
                const int base = tile_local_base<DIM>(c);
                double ws[2][NB], MV[2][DIM];
                unsigned long long dk[2] = { 0ull, 0ull };
#pragma unroll
                for (int i = 0; i < 2; ++i) {
#pragma unroll
                    for (int r = 0; r < NB; ++r) ws[i][r] = 0.0;
#pragma unroll
                    for (int a = 0; a < DIM; ++a) MV[i][a] = 0.0;
                    if (valid[i]) {
                        double xi[DIM], Vb[DIM], A[DIM];
                        const bool fast = local_coords<DIM>(gd, X[i], c, xi);
                        if (fast) {
                            double w[NB];
                            natural_weights<DIM>(xi, w);
                            gather_tile_a<DIM>(s_a, base, w, Vb, A);
                            swizzled_weights<DIM>(xi, l, ws[i]);
                        } else {
                            slow_gather<DIM>(gd, na, nullptr, X[i], Vb, A, nullptr);
                        }
#pragma unroll
                        for (int a = 0; a < DIM; ++a) MV[i][a] = M[i] * fma(dt, A[a], V[i][a]);   // M V'
                        if (!fast) {
                            slow_p2g2<DIM>(gd, g, X[i], MV[i]);
#pragma unroll
                            for (int a = 0; a < DIM; ++a) MV[i][a] = 0.0;
                        }
                        double Xn[DIM];
                        move_particle_lazy_id<DIM>(gd, X[i], Vb, dt, p.id, k0 + i, step, Xn);
                        const int key = tiled_key_of_position<DIM>(gd, Xn);
                        const int rank = atomicAdd(&count[key], 1);
                        dk[i] = ((unsigned long long)(unsigned)key << 32) | (unsigned)rank;
                    }
                }
                if (valid[1]) *reinterpret_cast<ulonglong2 *>(dest + k0) = make_ulonglong2(dk[0], dk[1]);
                else if (valid[0]) dest[k0] = dk[0];
                double tot[DIM][2];
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    double v[NB];
#pragma unroll
                    for (int r = 0; r < NB; ++r) v[r] = fma(MV[1][a], ws[1][r], MV[0][a] * ws[0][r]);
                    butterfly<DIM>(v);
                    tot[a][0] = v[0];
                    tot[a][1] = v[LG];
                }
                if (grp.cnt > 0) {
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
#if MPM_SCATTER_GLOBAL
                        const int node = corner_node_i<DIM>(gd, c, l + q * LG);
#pragma unroll
                        for (int a = 0; a < DIM; ++a) atomicAdd(&g.mv2[a][node], tot[a][q]);
#else
                        const int b = l + q * LG;
                        const int ln = base + (b & 1) + TG::N0 * ((b >> 1) & 1) + ((DIM == 3) ? TG::N0 * TG::N1 * ((b >> 2) & 1) : 0);
#pragma unroll
                        for (int a = 0; a < DIM; ++a) atomicAdd(&s_acc[a * NN + ln], tot[a][q]);
#endif
                    }
                }
            }
            __syncthreads();
#if !MPM_SCATTER_GLOBAL
#pragma unroll
            for (int a = 0; a < DIM; ++a) flush_channel<DIM>(gd, o, s_acc + a * NN, g.mv2[a]);
            __syncthreads();
#endif
            seg_begin = seg_end;
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.10-13
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_update_tiled(GridDesc gd, PArr p, PArr q, const double *__restrict__ na,
                                                         const double *__restrict__ nb, DevScalars *sc, SortedMap map,
                                                         const int *__restrict__ off_new,
                                                         const unsigned long long *__restrict__ dest, double *__restrict__ S_out)
{
    using K = TK<DIM>;
    constexpr int NB = K::NB, LG = K::LG, GPB = K::GPB, NN = K::NN;
    __shared__ __align__(16) double s_a[NN * K::NA];
    __shared__ __align__(16) double s_b[NN * K::NBS];
    __shared__ double s_v[kBlock / 32], s_c[kBlock / 32];
    const int n_groups = *map.n_groups;
    const double dt = sc->dt;
    const long long step = sc->step;
    const int l = threadIdx.x % LG;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double vloc = 0.0, cloc = 0.0;
    int n_rec = 0, n_clamp = 0, n_neg = 0, n_nonfin = 0;
    const double gm1 = gd.gamma - 1.0;
    for (int chunk = blockIdx.x; (long long)chunk * K::CG < n_groups; chunk += gridDim.x) {
        const int g_begin = chunk * K::CG, g_end = min(g_begin + K::CG, n_groups);
        int seg_begin = g_begin;
        while (seg_begin < g_end) {
            int tile;
            const int seg_end = segment_end<DIM>(map, seg_begin, g_end, tile);
            int o[DIM];
            tile_origin<DIM>(gd, tile, o);
            load_tile_a<DIM>(gd, o, na, s_a);
            load_tile_b<DIM>(gd, o, nb, s_b);
            __syncthreads();
            int gidx = seg_begin + threadIdx.x / LG;
            Group next = fetch_group(map.groups, gidx, seg_end);
            for (int gb = seg_begin; gb < seg_end; gb += GPB, gidx += GPB) {
                const Group grp = next;
                next = fetch_group(map.groups, (long long)gidx + GPB, seg_end);
                int c[DIM];
                unpack_coords<DIM>(grp.cpack, c);
                const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
                const long long k0 = (long long)grp.first + 2 * l;
                double X[2][DIM], V[2][DIM], M[2], rho[2], E[2];
                int id[2];
                unsigned long long dk[2];
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    const double2 tx = ld2(p.x[a], k0, valid[0]), tv = ld2(p.v[a], k0, valid[0]);
                    X[0][a] = tx.x; X[1][a] = valid[1] ? tx.y : 0.0;
                    V[0][a] = tv.x; V[1][a] = valid[1] ? tv.y : 0.0;
                }
                {
                    const double2 tm = ld2(p.m, k0, valid[0]), tr = ld2(p.rho, k0, valid[0]), te = ld2(p.e, k0, valid[0]);
                    M[0] = tm.x; M[1] = valid[1] ? tm.y : 0.0;
                    rho[0] = valid[0] ? tr.x : 1.0; rho[1] = valid[1] ? tr.y : 1.0;
                    E[0] = te.x; E[1] = valid[1] ? te.y : 0.0;
                    int2 ti = make_int2(0, 0);
                    ulonglong2 td = make_ulonglong2(0ull, 0ull);
                    if (valid[0]) {
                        ti = __ldg(reinterpret_cast<const int2 *>(p.id + k0));
                        td = __ldg(reinterpret_cast<const ulonglong2 *>(dest + k0));
                    }
                    id[0] = ti.x; id[1] = ti.y;
                    dk[0] = td.x; dk[1] = td.y;
                }
                const int base = tile_local_base<DIM>(c);
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    if (valid[i]) {
                        double xi[DIM], Vb[DIM], A[DIM], D;
                        if (local_coords<DIM>(gd, X[i], c, xi)) {
                            double w[NB];
                            natural_weights<DIM>(xi, w);
                            gather_tile_a<DIM>(s_a, base, w, Vb, A);
                            D = gather_divergence<DIM>(s_b, base, xi, gd.inv_h);
                        } else {
                            slow_gather<DIM>(gd, na, nb, X[i], Vb, A, &D);
                        }
                        double Vn[DIM];
#pragma unroll
                        for (int a = 0; a < DIM; ++a) Vn[a] = fma(dt, A[a], V[i][a]);   // V'
                        // particle thermodynamics (eq. 4 with this step's D: reading A2)
                        const double r = rho[i], e0 = E[i];
                        double Q = 0.0, Q_over_rho = 0.0;
                        if (D < 0.0) {
                            const double cs0 = sqrt(gd.gamma * gm1 * e0);
                            if (gd.visc_form == MPM_VISC_STANDARD) {
                                Q_over_rho = gd.c0 * gd.h * gd.h * D * D - gd.c1 * gd.h * cs0 * D;
                                Q = r * Q_over_rho;
                            } else {
                                Q = gd.c0 * (r * gd.h * D) * (r * gd.h * D) - gd.c1 * gd.h * cs0 * D;
                                Q_over_rho = Q / r;
                            }
                        }
                        double En = e0 - dt * (gm1 * e0 + Q_over_rho) * D;
                        const double jac = fma(dt, D, 1.0);
                        if (jac <= 0.0) n_neg++;
                        double rhon = r / jac;
                        const double cs = sqrt(gd.gamma * gm1 * En);
                        if (!isfinite(En) || !isfinite(rhon)) n_nonfin++;
                        double vv = 0.0, vb2 = 0.0;
#pragma unroll
                        for (int a = 0; a < DIM; ++a) { vv = fma(Vn[a], Vn[a], vv); vb2 = fma(Vb[a], Vb[a], vb2); }
                        vloc = fmax(vloc, fmax(vv, vb2));      // squared; the root is taken once at the end
                        cloc = fmax(cloc, cs);
                        double Xn[DIM];
                        bool recycled;
                        int nclamp;
                        move_particle<DIM>(gd, X[i], Vb, dt, (long long)id[i], step, Xn, recycled, nclamp);
                        n_clamp += nclamp;
                        double Mn = M[i];
                        if (recycled) {
#pragma unroll
                            for (int a = 0; a < DIM; ++a) Vn[a] = gd.inflow_v[a];
                            rhon = gd.inflow_rho; En = gd.inflow_e; Q = 0.0; Mn = gd.inflow_mass;
                            n_rec++;
                        }
                        const long long dst = (long long)off_new[(int)(dk[i] >> 32)] + (long long)(unsigned)(dk[i] & 0xffffffffull);
#pragma unroll
                        for (int a = 0; a < DIM; ++a) { q.x[a][dst] = Xn[a]; q.v[a][dst] = Vn[a]; }
                        q.m[dst] = Mn;
                        q.rho[dst] = rhon;
                        q.e[dst] = En;
                        q.q[dst] = Q;
                        q.id[dst] = id[i];
                        S_out[dst] = (gm1 * rhon * En + Q) * Mn / rhon;     // eq. (13) payload of the next step
                    }
                }
            }
            __syncthreads();      // the tiles are reloaded by the next segment
            seg_begin = seg_end;
        }
    }
    vloc = warp_max_nonneg(sqrt(vloc));
    cloc = warp_max_nonneg(cloc >= 0.0 ? cloc : 0.0);
    if (lane == 0) { s_v[warp] = vloc; s_c[warp] = cloc; }
    const int rec_sum = __reduce_add_sync(kFull, n_rec), neg_sum = __reduce_add_sync(kFull, n_neg),
              nf_sum = __reduce_add_sync(kFull, n_nonfin), clamp_sum = __reduce_add_sync(kFull, n_clamp);
    if (lane == 0) {
        if (rec_sum) atomicAdd(&sc->n_recycled, (unsigned long long)rec_sum);
        if (neg_sum) atomicAdd(&sc->n_negjac, (unsigned long long)neg_sum);
        if (nf_sum) atomicAdd(&sc->n_nonfinite, (unsigned long long)nf_sum);
        if (clamp_sum) atomicAdd(&sc->n_clamped, (unsigned long long)clamp_sum);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = s_v[0], cc = s_c[0];
#pragma unroll
        for (int w = 1; w < kBlock / 32; ++w) { v = fmax(v, s_v[w]); cc = fmax(cc, s_c[w]); }
        if (v > 0.0) atomic_max_nonneg(&sc->vmax_bits, v);
        if (cc > 0.0) atomic_max_nonneg(&sc->cmax_bits, cc);
    }
}

// ------------------------------------------------------------------------------------------------ bookkeeping kernels

__global__ void __launch_bounds__(kBlock) k_force_payload_slots(double gamma, const double *m, const double *rho, const double *e,
                                                                const double *q, double *S, long long n)
{
    const long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k < n) S[k] = ((gamma - 1.0) * rho[k] * e[k] + q[k]) * m[k] / rho[k];    // unused slots hold zeros -> NaN, never read
}

__global__ void __launch_bounds__(kBlock) k_group_counts_tiled(const int *count, int *gcount, int nkeys, int cap)
{
    const int c = blockIdx.x * kBlock + threadIdx.x;
    if (c < nkeys) gcount[c] = (count[c] + cap - 1) / cap;
    else if (c == nkeys) gcount[c] = 0;
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_group_fill_tiled(GridDesc gd, const int *count, const int *off, const int *goff,
                                                             int4 *groups, int *n_groups, int nkeys)
{
    constexpr int CAP = 1 << DIM;
    const int key = blockIdx.x * kBlock + threadIdx.x;
    if (key == 0) *n_groups = goff[nkeys];
    if (key >= nkeys) return;
    const int g0 = goff[key], g1 = goff[key + 1];
    if (g0 == g1) return;
    int c[DIM];
    tiled_cell_of_key<DIM>(gd, key, c);
    const int cpack = (DIM == 3) ? (c[0] | (c[1] << 10) | (c[DIM - 1] << 20)) : (c[0] | (c[1] << 16));
    int first = off[key];
    const int end = first + count[key];
    for (int gq = g0; gq < g1; ++gq, first += CAP) groups[gq] = make_int4(first, min(CAP, end - first), key, cpack);
}

// dst[id] = src[slot] for every occupied slot (one thread per group); coff != NULL: dst[compact storage index] instead
__global__ void __launch_bounds__(kBlock) k_gather_by_id_groups(const double *src, const int *id, double *dst, SortedMap map,
                                                                const int *coff, const int *off)
{
    const int n_groups = *map.n_groups;
    for (long long gq = (long long)blockIdx.x * kBlock + threadIdx.x; gq < n_groups; gq += (long long)gridDim.x * kBlock) {
        const int4 r = map.groups[gq];
        for (int j = 0; j < r.y; ++j) {
            const long long k = (long long)r.x + j;
            const long long d = coff ? (long long)coff[r.z] + (k - off[r.z]) : (long long)id[k];
            dst[d] = src[k];
        }
    }
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_stats_reduce_groups(PArr p, DevScalars *sc, SortedMap map)
{
    __shared__ double s[kBlock / 32][5];
    double acc[5] = { 0, 0, 0, 0, 0 };
    const int n_groups = *map.n_groups;
    for (long long gq = (long long)blockIdx.x * kBlock + threadIdx.x; gq < n_groups; gq += (long long)gridDim.x * kBlock) {
        const int4 r = map.groups[gq];
        for (int j = 0; j < r.y; ++j) {
            const long long k = (long long)r.x + j;
            const double M = p.m[k];
            double v2 = 0.0;
            acc[0] += M;
#pragma unroll
            for (int a = 0; a < DIM; ++a) { const double v = p.v[a][k]; acc[1 + a] += M * v; v2 += v * v; }
            acc[4] += M * (p.e[k] + 0.5 * v2);
        }
    }
#pragma unroll
    for (int j = 0; j < 5; ++j)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc[j] += __shfl_xor_sync(0xffffffffu, acc[j], o);
    if ((threadIdx.x & 31) == 0)
        for (int j = 0; j < 5; ++j) s[threadIdx.x >> 5][j] = acc[j];
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int w = 0; w < kBlock / 32; ++w) t += s[w][threadIdx.x];
        double *dst = (threadIdx.x == 0) ? &sc->sum_mass : (threadIdx.x == 4) ? &sc->sum_energy : &sc->sum_mom[threadIdx.x - 1];
        atomicAdd(dst, t);
    }
}

__global__ void k_stats_clear_t(DevScalars *sc)
{
    sc->sum_mass = 0.0; sc->sum_energy = 0.0;
    sc->sum_mom[0] = sc->sum_mom[1] = sc->sum_mom[2] = 0.0;
}

inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

// persistent launch: as many blocks as are resident at once (occupancy query), never more than there are chunks
template <typename Kernel>
inline unsigned persistent_blocks(long long max_groups, int groups_per_chunk, Kernel kernel)
{
    int dev = 0, sms = 148, per_sm = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kBlock, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
    const long long want = (long long)sms * per_sm;
    const long long need = (max_groups + groups_per_chunk - 1) / groups_per_chunk;
    return (unsigned)(need < want ? (need > 0 ? need : 1) : want);
}

}  // namespace

void launch_force_payload_slots(const GridDesc &gd, const PArr &p, double *S, long long nslots, cudaStream_t s)
{
    if (nslots > 0) k_force_payload_slots<<<blocks_for(nslots, kBlock), kBlock, 0, s>>>(gd.gamma, p.m, p.rho, p.e, p.q, S, nslots);
}

void launch_build_groups_tiled(const GridDesc &gd, const int *count, const int *off, int *goff, int *scan_aux, int4 *groups,
                               int *n_groups, cudaStream_t s)
{
    const int cap = 1 << gd.dim;
    const int nkeys = (int)gd.Nkeys;
    k_group_counts_tiled<<<blocks_for(nkeys + 1, kBlock), kBlock, 0, s>>>(count, goff, nkeys, cap);
    launch_exclusive_scan(goff, nkeys + 1, scan_aux, s);
    if (gd.dim == 2) k_group_fill_tiled<2><<<blocks_for(nkeys, kBlock), kBlock, 0, s>>>(gd, count, off, goff, groups, n_groups, nkeys);
    else k_group_fill_tiled<3><<<blocks_for(nkeys, kBlock), kBlock, 0, s>>>(gd, count, off, goff, groups, n_groups, nkeys);
}

void launch_p2g1_tiled(const GridDesc &gd, const PArr &p, const double *S, const GArr &g, const SortedMap &map,
                       long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2) k_p2g1_tiled<2><<<persistent_blocks(max_groups, TK<2>::CG, k_p2g1_tiled<2>), kBlock, 0, s>>>(gd, p, S, g, map);
    else k_p2g1_tiled<3><<<persistent_blocks(max_groups, TK<3>::CG, k_p2g1_tiled<3>), kBlock, 0, s>>>(gd, p, S, g, map);
}

void launch_g2p_p2g2_tiled(const GridDesc &gd, const PArr &p, const GArr &g, const double *na, const DevScalars *sc,
                           const SortedMap &map, int *count, unsigned long long *dest, long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_g2p_p2g2_tiled<2><<<persistent_blocks(max_groups, TK<2>::CG, k_g2p_p2g2_tiled<2>), kBlock, 0, s>>>(gd, p, g, na, sc, map, count, dest);
    else
        k_g2p_p2g2_tiled<3><<<persistent_blocks(max_groups, TK<3>::CG, k_g2p_p2g2_tiled<3>), kBlock, 0, s>>>(gd, p, g, na, sc, map, count, dest);
}

void launch_update_tiled(const GridDesc &gd, const PArr &p, const PArr &q, const double *na, const double *nb, DevScalars *sc,
                         const SortedMap &map, const int *off_new, const unsigned long long *dest, double *S_out,
                         long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_update_tiled<2><<<persistent_blocks(max_groups, TK<2>::CG, k_update_tiled<2>), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map, off_new, dest, S_out);
    else
        k_update_tiled<3><<<persistent_blocks(max_groups, TK<3>::CG, k_update_tiled<3>), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map, off_new, dest, S_out);
}

void launch_gather_by_id_groups(const double *src, const int *id, double *dst, const SortedMap &map, long long max_groups,
                                const int *coff, const int *off, cudaStream_t s)
{
    if (max_groups <= 0) return;
    const unsigned blocks = (unsigned)((max_groups + kBlock - 1) / kBlock < 148 * 16 ? (max_groups + kBlock - 1) / kBlock : 148 * 16);
    k_gather_by_id_groups<<<blocks, kBlock, 0, s>>>(src, id, dst, map, coff, off);
}

void launch_stats_reduce_groups(const GridDesc &gd, const PArr &p, DevScalars *sc, const SortedMap &map, long long max_groups,
                                cudaStream_t s)
{
    k_stats_clear_t<<<1, 1, 0, s>>>(sc);
    if (max_groups <= 0) return;
    const unsigned blocks = (unsigned)((max_groups + kBlock - 1) / kBlock < 148 * 8 ? (max_groups + kBlock - 1) / kBlock : 148 * 8);
    if (gd.dim == 2) k_stats_reduce_groups<2><<<blocks, kBlock, 0, s>>>(p, sc, map);
    else k_stats_reduce_groups<3><<<blocks, kBlock, 0, s>>>(p, sc, map);
}

}  // namespace mpm
