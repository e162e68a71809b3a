// mpm_kernels_sorted.cu -- SORTED kernel family: particles are kept EXACTLY cell-sorted every step and processed in
// aligned lane groups, one cell per group, one particle per lane (GS = 2^d lanes: 8 in 3D, 4 in 2D).
//
// What this buys over the paper's one-thread-per-particle + atomicAdd design:
//   * scatters (Alg. 1 l.3 and l.8): every lane computes its particle's contribution to the 2^d corners of the cell,
//     the group sums them with a transposed XOR butterfly (2^d - 1 shuffles per channel) after which lane j owns the
//     total of corner j, and issues ONE global fp64 reduction per channel: 2^d x fewer REDs, spread over 2^d nodes.
//     (Shared-memory fp64 atomicAdd is a CAS loop on sm_100a -- ATOMS.CAST.SPIN.64 -- so it is never used.)
//   * gathers (l.6, l.10, l.11): lane j fetches the node values of corner j once per group (16-byte loads from
//     node-major arrays), parks them in shared memory, and every lane reads all corners back as conflict-free
//     128-bit broadcasts: 2^d x fewer global gathers.
//   * gradient channels are folded into phi-weighted channels using sum_{b_a} w_a(b_a) = 1:
//       f_a(b) = +-(1/h) sum_{b_a} T_S(b),  T_S(b) = sum_k S_k phi_b(X_k)             (P2G#1: 1+d+1 channels, not 1+2d)
//       D_k    = sum_b phi_b(X_k) sum_a (v2_a(b | a) - v2_a(b & ~a))/h                (G2PD  : 1 channel, not d)
//   * the re-ordering (l.12) is fused into the sweeps: the gather kernel of l.6-8 computes each particle's new cell
//     and its rank in it (one returning integer atomic), a scan of the per-cell counts gives the new cell offsets, and
//     the update kernel of l.10-11 writes every particle straight to its sorted slot in the other buffer: no
//     separate permutation pass.
// A particle whose true cell differs from its group's cell (never the case when the invariant holds; cheap to test)
// takes a slow path with direct global reductions / gathers, so correctness never depends on the ordering.
#include "mpm_internal.cuh"

namespace mpm {

namespace {

constexpr int kBlock = 256;
constexpr unsigned kFull = 0xffffffffu;

template <int DIM>
struct Geo {
    static constexpr int GS = 1 << DIM;            // lanes per group = corners per cell
    static constexpr int NG = 32 / GS;             // groups per warp
    static constexpr int GPB = kBlock / GS;        // groups per block
    // shared staging of corner node values: [group][corner][channel]; strides chosen so that the 16-byte broadcast
    // reads of the NG groups of a warp fall into distinct banks
    static constexpr int CH = (DIM == 3) ? 8 : 6;                       // doubles per corner (vbar, acc, dsum, pad)
    static constexpr int CORNER_STRIDE = CH;                            // doubles
    static constexpr int GROUP_STRIDE = (DIM == 3) ? 68 : 26;           // doubles: 544 B / 208 B
    static constexpr int WARP_DOUBLES = NG * GROUP_STRIDE;
};

__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(kFull, v, m); }

// after the call v[0] holds the group-wide sum for corner j = lane-in-group (see header comment)
template <int DIM>
__device__ __forceinline__ void butterfly(double v[1 << DIM])
{
    if (DIM == 3) {
#pragma unroll
        for (int r = 0; r < 4; ++r) v[r] += shfl_xor_d(v[r + 4], 4);
    }
#pragma unroll
    for (int r = 0; r < 2; ++r) v[r] += shfl_xor_d(v[r + 2], 2);
    v[0] += shfl_xor_d(v[1], 1);
}

struct Group {
    int cell;      // linear cell index of the group
    int first;     // first particle of the group
    int cnt;       // particles in the group (<= GS), 0 = idle group
};

template <int DIM>
__device__ __forceinline__ Group load_group(const int *grp_cell, const int *grp_first, const int *off, const int *n_groups,
                                            int &j)
{
    constexpr int GS = Geo<DIM>::GS;
    const long long gidx = (long long)blockIdx.x * Geo<DIM>::GPB + threadIdx.x / GS;
    j = threadIdx.x % GS;
    Group g{ 0, 0, 0 };
    if (gidx < (long long)*n_groups) {
        g.cell = grp_cell[gidx];
        g.first = grp_first[gidx];
        g.cnt = min(GS, off[g.cell + 1] - g.first);
    }
    return g;
}

template <int DIM>
__device__ __forceinline__ void cell_coords(const GridDesc &gd, int cell, int c[DIM])
{
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        c[a] = cell % gd.nc[a];
        cell /= gd.nc[a];
    }
}

// local coordinates w.r.t. the GROUP's cell; returns false if the particle's own cell (A6, A19) is a different one
template <int DIM>
__device__ __forceinline__ bool local_coords(const GridDesc &gd, const double X[DIM], const int c[DIM], double xi[DIM])
{
    bool same = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int ci;
        cell_1d(X[a], gd.inv_h, gd.nc[a], ci, xi[a]);
        same = same && (ci == c[a]);
    }
    return same;
}

// weights in natural corner order (gathers) ...
template <int DIM>
__device__ __forceinline__ void natural_weights(const double xi[DIM], double w[1 << DIM])
{
#pragma unroll
    for (int b = 0; b < (1 << DIM); ++b) w[b] = corner_phi<DIM>(xi, b);
}
// ... and in butterfly order (scatters): register r of lane j holds the weight of corner r ^ j
template <int DIM>
__device__ __forceinline__ void swizzled_weights(const double xi[DIM], int j, double w[1 << DIM])
{
    double p[DIM][2];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const bool hi = (j >> a) & 1;
        p[a][0] = hi ? xi[a] : 1.0 - xi[a];
        p[a][1] = hi ? 1.0 - xi[a] : xi[a];
    }
#pragma unroll
    for (int r = 0; r < (1 << DIM); ++r) {
        double q = 1.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) q *= p[a][(r >> a) & 1];
        w[r] = q;
    }
}

// ---------------------------------------------------------------------------------------------- slow paths
template <int DIM>
__device__ __forceinline__ void slow_p2g1(const GridDesc &gd, const GArr &g, const double X[DIM], const double V[DIM],
                                       double M, double S)
{
    int c[DIM];
    double xi[DIM];
    particle_cell<DIM>(gd, X, c, xi);
#pragma unroll 1
    for (int ib = 0; ib < (1 << DIM); ++ib) {
        const long long i = corner_node<DIM>(gd, c, ib);
        const double phi = corner_phi<DIM>(xi, ib);
        atomicAdd(&g.m[i], M * phi);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            atomicAdd(&g.mv[a][i], M * V[a] * phi);
            atomicAdd(&g.f[a][i], S * corner_dphi<DIM>(xi, ib, a, gd.inv_h));
        }
    }
}

template <int DIM>
__device__ __forceinline__ void slow_gather(const GridDesc &gd, const double *na, const double *nb, const double X[DIM],
                                         double Vb[DIM], double A[DIM], double *D)
{
    int c[DIM];
    double xi[DIM];
    particle_cell<DIM>(gd, X, c, xi);
    double d = 0.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) { Vb[a] = 0.0; A[a] = 0.0; }
#pragma unroll 1
    for (int ib = 0; ib < (1 << DIM); ++ib) {
        const long long i = corner_node<DIM>(gd, c, ib);
        const double phi = corner_phi<DIM>(xi, ib);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            Vb[a] += phi * na[i * (2 * DIM) + a];
            A[a] += phi * na[i * (2 * DIM) + DIM + a];
            if (nb) d += nb[i * DIM + a] * corner_dphi<DIM>(xi, ib, a, gd.inv_h);
        }
    }
    if (D) *D = d;
}

template <int DIM>
__device__ __forceinline__ void slow_p2g2(const GridDesc &gd, const GArr &g, const double X[DIM], const double MV[DIM])
{
    int c[DIM];
    double xi[DIM];
    particle_cell<DIM>(gd, X, c, xi);
#pragma unroll 1
    for (int ib = 0; ib < (1 << DIM); ++ib) {
        const long long i = corner_node<DIM>(gd, c, ib);
        const double phi = corner_phi<DIM>(xi, ib);
#pragma unroll
        for (int a = 0; a < DIM; ++a) atomicAdd(&g.mv2[a][i], MV[a] * phi);
    }
}

// ---------------------------------------------------------------------------------------------- shared pieces

// Alg. 1 l.11 for one particle: X' = X + dt Vbar, periodic wrap (A11), outflow detection, recycling position (A8),
// clamp.  Used by BOTH the gather kernel (to find the new cell) and the update kernel (to write X'), so the two agree.
template <int DIM>
__device__ __forceinline__ void move_particle(const GridDesc &gd, const double X[DIM], const double Vb[DIM], double dt,
                                              long long id, long long step, double Xn[DIM], bool &recycled, int &nclamp)
{
    bool recycle = false;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double x = fma(dt, Vb[a], X[a]);
        if (gd.per[a]) {
            x = x - gd.L[a] * floor(x / gd.L[a]);
            if (x >= gd.L[a]) x = 0.0;
        } else {
            if (x < 0.0 && gd.bc[a][0] == MPM_BC_OUTFLOW) recycle = true;
            if (x > gd.L[a] && gd.bc[a][1] == MPM_BC_OUTFLOW) recycle = true;
        }
        Xn[a] = x;
    }
    recycled = recycle && gd.in_axis >= 0;
    if (recycled) {
        int jj = 0;
        const double u0 = recycle_uniform(gd.recycle_seed, id, step, jj++);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            if (a == gd.in_axis) {
                Xn[a] = (gd.in_side == 0) ? u0 * gd.h : gd.L[a] - u0 * gd.h;
            } else {
                const double u1 = recycle_uniform(gd.recycle_seed, id, step, jj++);
                const double u2 = recycle_uniform(gd.recycle_seed, id, step, jj++);
                int cell = (int)floor(u1 * (double)gd.nc[a]);
                cell = min(cell, gd.nc[a] - 1);
                Xn[a] = ((double)cell + u2) * gd.h;
            }
        }
    }
    nclamp = 0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (!gd.per[a]) {
            if (Xn[a] < 0.0) { Xn[a] = 0.0; nclamp++; }
            if (Xn[a] > gd.L[a]) { Xn[a] = gd.L[a]; nclamp++; }
        }
    }
}

template <int DIM>
__device__ __forceinline__ int cell_key(const GridDesc &gd, const double X[DIM])
{
    int key = 0, stride = 1;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int c;
        double xi;
        cell_1d(X[a], gd.inv_h, gd.nc[a], c, xi);
        key += stride * c;
        stride *= gd.nc[a];
    }
    return key;
}

// node index of corner j of cell c (periodic wrap: node n == node 0)
template <int DIM>
__device__ __forceinline__ int group_node(const GridDesc &gd, const int c[DIM], int j)
{
    return (int)corner_node<DIM>(gd, c, j);
}

// lane j stages vbar, acc of corner j (node-major array na[node][2 DIM]) into shared memory; returns nothing
template <int DIM>
__device__ __forceinline__ void stage_na(const double *__restrict__ na, int node, double *s_corner)
{
    const double2 *src = reinterpret_cast<const double2 *>(na + (long long)node * (2 * DIM));
    double2 *dst = reinterpret_cast<double2 *>(s_corner);
#pragma unroll
    for (int q = 0; q < DIM; ++q) dst[q] = __ldg(src + q);
}

// phi-weighted gather of the staged channels: out[c] = sum_b w[b] vals[b][c], c < 2*NP2 (pairs of doubles)
template <int DIM, int NPAIR>
__device__ __forceinline__ void gather_pairs(const double *s_group, const double w[1 << DIM], double out[2 * NPAIR])
{
#pragma unroll
    for (int c = 0; c < 2 * NPAIR; ++c) out[c] = 0.0;
#pragma unroll
    for (int b = 0; b < (1 << DIM); ++b) {
        const double2 *row = reinterpret_cast<const double2 *>(s_group + b * Geo<DIM>::CORNER_STRIDE);
#pragma unroll
        for (int q = 0; q < NPAIR; ++q) {
            const double2 t = row[q];
            out[2 * q] = fma(w[b], t.x, out[2 * q]);
            out[2 * q + 1] = fma(w[b], t.y, out[2 * q + 1]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.3
// m, mv from phi-weighted channels (M, M V); f from the phi-weighted channel S = (P+Q) M / rho
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_p2g1_sorted(GridDesc gd, PArr p, const double *__restrict__ Sarr, GArr g,
                                                        const int *__restrict__ grp_cell, const int *__restrict__ grp_first,
                                                        const int *__restrict__ off, const int *__restrict__ n_groups)
{
    constexpr int NB = 1 << DIM;
    int j;
    const Group grp = load_group<DIM>(grp_cell, grp_first, off, n_groups, j);
    int c[DIM];
    cell_coords<DIM>(gd, grp.cell, c);
    double w[NB];
#pragma unroll
    for (int r = 0; r < NB; ++r) w[r] = 0.0;
    double M = 0.0, S = 0.0, MV[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) MV[a] = 0.0;
    if (j < grp.cnt) {
        const long long k = grp.first + j;
        double X[DIM], V[DIM], xi[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) { X[a] = p.x[a][k]; V[a] = p.v[a][k]; }
        M = p.m[k];
        S = Sarr[k];
        if (local_coords<DIM>(gd, X, c, xi)) {
            swizzled_weights<DIM>(xi, j, w);
#pragma unroll
            for (int a = 0; a < DIM; ++a) MV[a] = M * V[a];
        } else {
            slow_p2g1<DIM>(gd, g, X, V, M, S);
            M = 0.0; S = 0.0;
        }
    }
    // group sums per corner: channels M, M V_a, S
    double v[NB];
    double tot[DIM + 2];
#pragma unroll
    for (int ch = 0; ch < DIM + 2; ++ch) {
        const double pay = (ch == 0) ? M : (ch == DIM + 1) ? S : MV[ch - 1];
#pragma unroll
        for (int r = 0; r < NB; ++r) v[r] = pay * w[r];
        butterfly<DIM>(v);
        tot[ch] = v[0];
    }
    // force of corner j: f_a = +-(1/h) (T_S(j) + T_S(j ^ bit_a)), sign + where the corner is on the high side of axis a
    double F[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const double pair = tot[DIM + 1] + shfl_xor_d(tot[DIM + 1], 1 << a);
        F[a] = ((j >> a) & 1) ? pair * gd.inv_h : -(pair * gd.inv_h);
    }
    if (grp.cnt > 0) {
        const int node = group_node<DIM>(gd, c, j);
        atomicAdd(&g.m[node], tot[0]);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            atomicAdd(&g.mv[a][node], tot[1 + a]);
            atomicAdd(&g.f[a][node], F[a]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.6-8 (+ l.11-12 bookkeeping)
// A = G2P(f/m), Vbar = G2P(mv'/m); V' = V + dt A; mv2 += M V' phi.  Also: the particle's cell after the
// move of l.11 and its rank inside that cell, for the fused re-ordering.  V' is NOT stored: the update kernel recomputes it.
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_g2p_p2g2_sorted(GridDesc gd, PArr p, GArr g, const double *__restrict__ na,
                                                            const DevScalars *__restrict__ sc,
                                                            const int *__restrict__ grp_cell, const int *__restrict__ grp_first,
                                                            const int *__restrict__ off, const int *__restrict__ n_groups,
                                                            int *__restrict__ count, unsigned long long *__restrict__ dest)
{
    constexpr int NB = 1 << DIM;
    __shared__ __align__(16) double s_vals[(kBlock / 32) * Geo<DIM>::WARP_DOUBLES];
    int j;
    const Group grp = load_group<DIM>(grp_cell, grp_first, off, n_groups, j);
    int c[DIM];
    cell_coords<DIM>(gd, grp.cell, c);
    const int warp = threadIdx.x >> 5, gi = (threadIdx.x & 31) / Geo<DIM>::GS;
    double *s_group = s_vals + warp * Geo<DIM>::WARP_DOUBLES + gi * Geo<DIM>::GROUP_STRIDE;
    const int node = group_node<DIM>(gd, c, j);
    if (grp.cnt > 0) stage_na<DIM>(na, node, s_group + j * Geo<DIM>::CORNER_STRIDE);
    __syncwarp();
    const double dt = sc->dt;
    double ws[NB];
#pragma unroll
    for (int r = 0; r < NB; ++r) ws[r] = 0.0;
    double MV[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) MV[a] = 0.0;
    if (j < grp.cnt) {
        const long long k = grp.first + j;
        double X[DIM], V[DIM], xi[DIM], Vb[DIM], A[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) { X[a] = p.x[a][k]; V[a] = p.v[a][k]; }
        const double M = p.m[k];
        const bool fast = local_coords<DIM>(gd, X, c, xi);
        if (fast) {
            double w[NB], out[2 * DIM];
            natural_weights<DIM>(xi, w);
            gather_pairs<DIM, DIM>(s_group, w, out);
#pragma unroll
            for (int a = 0; a < DIM; ++a) { Vb[a] = out[a]; A[a] = out[DIM + a]; }
            swizzled_weights<DIM>(xi, j, ws);
        } else {
            slow_gather<DIM>(gd, na, nullptr, X, Vb, A, nullptr);
        }
#pragma unroll
        for (int a = 0; a < DIM; ++a) MV[a] = M * fma(dt, A[a], V[a]);   // M V'
        if (!fast) {
            slow_p2g2<DIM>(gd, g, X, MV);
#pragma unroll
            for (int a = 0; a < DIM; ++a) MV[a] = 0.0;
        }
        // where the particle will be after l.11, and its rank among the particles that end up in that cell
        double Xn[DIM];
        bool recycled;
        int nclamp;
        move_particle<DIM>(gd, X, Vb, dt, (long long)p.id[k], sc->step, Xn, recycled, nclamp);
        const int key = cell_key<DIM>(gd, Xn);
        const int rank = atomicAdd(&count[key], 1);
        dest[k] = ((unsigned long long)(unsigned)key << 32) | (unsigned)rank;
    }
    double v[NB];
    double tot[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
#pragma unroll
        for (int r = 0; r < NB; ++r) v[r] = MV[a] * ws[r];
        butterfly<DIM>(v);
        tot[a] = v[0];
    }
    if (grp.cnt > 0) {
#pragma unroll
        for (int a = 0; a < DIM; ++a) atomicAdd(&g.mv2[a][node], tot[a]);
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.10-13
// D = trace G2PD(mv2/m); Q (eq. 4), E', rho'; V' = V + dt A again; CFL maxima;
// X' = X + dt Vbar; the particle is written to its cell-sorted slot of the OTHER buffer (l.12),
// together with next step's force payload S' = (P'+Q') M / rho' (eq. 13).
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_update_sorted(GridDesc gd, PArr p, PArr q, const double *__restrict__ na,
                                                          const double *__restrict__ nb, DevScalars *sc,
                                                          const int *__restrict__ grp_cell, const int *__restrict__ grp_first,
                                                          const int *__restrict__ off, const int *__restrict__ n_groups,
                                                          const int *__restrict__ off_new,
                                                          const unsigned long long *__restrict__ dest, double *__restrict__ S_out)
{
    constexpr int NB = 1 << DIM;
    constexpr int NPAIR = (DIM == 3) ? 4 : 3;
    __shared__ __align__(16) double s_vals[(kBlock / 32) * Geo<DIM>::WARP_DOUBLES];
    __shared__ double s_v[kBlock / 32], s_c[kBlock / 32];
    int j;
    const Group grp = load_group<DIM>(grp_cell, grp_first, off, n_groups, j);
    int c[DIM];
    cell_coords<DIM>(gd, grp.cell, c);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gi = lane / Geo<DIM>::GS;
    double *s_group = s_vals + warp * Geo<DIM>::WARP_DOUBLES + gi * Geo<DIM>::GROUP_STRIDE;
    const int node = group_node<DIM>(gd, c, j);
    // stage vbar, acc of corner j, and dsum_j = sum_a (v2_a(high corner) - v2_a(low corner)) / h
    double v2[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) v2[a] = (grp.cnt > 0) ? __ldg(nb + (long long)node * DIM + a) : 0.0;
    double dsum = 0.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const double other = shfl_xor_d(v2[a], 1 << a);
        dsum += ((j >> a) & 1) ? (v2[a] - other) : (other - v2[a]);
    }
    if (grp.cnt > 0) {
        stage_na<DIM>(na, node, s_group + j * Geo<DIM>::CORNER_STRIDE);
        s_group[j * Geo<DIM>::CORNER_STRIDE + 2 * DIM] = dsum * gd.inv_h;
        if (DIM == 3) s_group[j * Geo<DIM>::CORNER_STRIDE + 7] = 0.0; else s_group[j * Geo<DIM>::CORNER_STRIDE + 5] = 0.0;
    }
    __syncwarp();
    double vloc = 0.0, cloc = 0.0;
    int n_rec = 0, n_clamp = 0, n_neg = 0, n_nonfin = 0;
    if (j < grp.cnt) {
        const long long k = grp.first + j;
        const double dt = sc->dt;
        double X[DIM], V[DIM], xi[DIM], Vb[DIM], A[DIM], D;
#pragma unroll
        for (int a = 0; a < DIM; ++a) { X[a] = p.x[a][k]; V[a] = p.v[a][k]; }
        double M = p.m[k], rho = p.rho[k], E = p.e[k];
        const int id = p.id[k];
        const unsigned long long dk = dest[k];
        if (local_coords<DIM>(gd, X, c, xi)) {
            double w[NB], out[2 * NPAIR];
            natural_weights<DIM>(xi, w);
            gather_pairs<DIM, NPAIR>(s_group, w, out);
#pragma unroll
            for (int a = 0; a < DIM; ++a) { Vb[a] = out[a]; A[a] = out[DIM + a]; }
            D = out[2 * DIM];
        } else {
            slow_gather<DIM>(gd, na, nb, X, Vb, A, &D);
        }
#pragma unroll
        for (int a = 0; a < DIM; ++a) V[a] = fma(dt, A[a], V[a]);   // V'
        // particle thermodynamics (eq. 4 with this step's D: reading A2)
        const double P = (gd.gamma - 1.0) * rho * E;
        double Q = 0.0;
        if (D < 0.0) {
            const double cs0 = sqrt(gd.gamma * P / rho);
            if (gd.visc_form == MPM_VISC_STANDARD)
                Q = rho * (gd.c0 * gd.h * gd.h * D * D - gd.c1 * gd.h * cs0 * D);
            else
                Q = gd.c0 * (rho * gd.h * D) * (rho * gd.h * D) - gd.c1 * gd.h * cs0 * D;
        }
        double En = E + dt * (-(P + Q) / rho) * D;
        const double jac = 1.0 + dt * D;
        if (jac <= 0.0) n_neg = 1;
        double rhon = rho / jac;
        const double Pn = (gd.gamma - 1.0) * rhon * En;
        const double cs = sqrt(gd.gamma * Pn / rhon);
        if (!isfinite(En) || !isfinite(rhon)) n_nonfin = 1;
        double vv = 0.0, vb2 = 0.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) { vv += V[a] * V[a]; vb2 += Vb[a] * Vb[a]; }
        vloc = fmax(sqrt(vv), sqrt(vb2));
        cloc = cs;
        double Xn[DIM];
        bool recycled;
        move_particle<DIM>(gd, X, Vb, dt, (long long)id, sc->step, Xn, recycled, n_clamp);
        if (recycled) {
#pragma unroll
            for (int a = 0; a < DIM; ++a) V[a] = gd.inflow_v[a];
            rhon = gd.inflow_rho; En = gd.inflow_e; Q = 0.0; M = gd.inflow_mass;
            n_rec = 1;
        }
        const long long dst = (long long)off_new[(int)(dk >> 32)] + (long long)(unsigned)(dk & 0xffffffffull);
#pragma unroll
        for (int a = 0; a < DIM; ++a) { q.x[a][dst] = Xn[a]; q.v[a][dst] = V[a]; }
        q.m[dst] = M;
        q.rho[dst] = rhon;
        q.e[dst] = En;
        q.q[dst] = Q;
        q.id[dst] = id;
        S_out[dst] = ((gd.gamma - 1.0) * rhon * En + Q) * M / rhon;     // eq. (13) payload of the next step
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        vloc = fmax(vloc, __shfl_xor_sync(kFull, vloc, o));
        cloc = fmax(cloc, __shfl_xor_sync(kFull, cloc, o));
    }
    if (lane == 0) { s_v[warp] = vloc; s_c[warp] = cloc; }
    const unsigned any_rec = __ballot_sync(kFull, n_rec), any_neg = __ballot_sync(kFull, n_neg),
                   any_nf = __ballot_sync(kFull, n_nonfin);
    int clamp_sum = n_clamp;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) clamp_sum += __shfl_xor_sync(kFull, clamp_sum, o);
    if (lane == 0) {
        if (any_rec) atomicAdd(&sc->n_recycled, (unsigned long long)__popc(any_rec));
        if (any_neg) atomicAdd(&sc->n_negjac, (unsigned long long)__popc(any_neg));
        if (any_nf) atomicAdd(&sc->n_nonfinite, (unsigned long long)__popc(any_nf));
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

// S = (P+Q) M / rho for a freshly loaded / permuted particle set (eq. 13)
__global__ void __launch_bounds__(kBlock) k_force_payload(double gamma, const double *m, const double *rho, const double *e,
                                                          const double *q, double *S, long long n)
{
    const long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k < n) S[k] = ((gamma - 1.0) * rho[k] * e[k] + q[k]) * m[k] / rho[k];
}

// groups per cell = ceil(count / GS), from the cell offsets
__global__ void __launch_bounds__(kBlock) k_group_counts(const int *off, int *gcount, int ncell, int gs)
{
    const int c = blockIdx.x * kBlock + threadIdx.x;
    if (c < ncell) gcount[c] = (off[c + 1] - off[c] + gs - 1) / gs;
    else if (c == ncell) gcount[c] = 0;
}

// fill the group map from the scanned group offsets; goff[ncell] = total number of groups
__global__ void __launch_bounds__(kBlock) k_group_fill(const int *off, const int *goff, int *grp_cell, int *grp_first,
                                                       int *n_groups, int ncell, int gs)
{
    const int c = blockIdx.x * kBlock + threadIdx.x;
    if (c == 0) *n_groups = goff[ncell];
    if (c >= ncell) return;
    const int g0 = goff[c], g1 = goff[c + 1];
    int first = off[c];
    for (int g = g0; g < g1; ++g, first += gs) { grp_cell[g] = c; grp_first[g] = first; }
}

inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

}  // namespace

void launch_force_payload(const GridDesc &gd, const PArr &p, double *S, long long n, cudaStream_t s)
{
    if (n > 0) k_force_payload<<<blocks_for(n, kBlock), kBlock, 0, s>>>(gd.gamma, p.m, p.rho, p.e, p.q, S, n);
}

void launch_build_groups(const GridDesc &gd, const int *off, int *gcount_goff, int *scan_aux, int *grp_cell, int *grp_first,
                         int *n_groups, cudaStream_t s)
{
    const int gs = 1 << gd.dim;
    const int ncell = (int)gd.Nc;
    k_group_counts<<<blocks_for(ncell + 1, kBlock), kBlock, 0, s>>>(off, gcount_goff, ncell, gs);
    launch_exclusive_scan(gcount_goff, ncell + 1, scan_aux, s);
    k_group_fill<<<blocks_for(ncell, kBlock), kBlock, 0, s>>>(off, gcount_goff, grp_cell, grp_first, n_groups, ncell, gs);
}

void launch_p2g1_sorted(const GridDesc &gd, const PArr &p, const double *S, const GArr &g, const SortedMap &map,
                        long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_p2g1_sorted<2><<<blocks_for(max_groups, Geo<2>::GPB), kBlock, 0, s>>>(gd, p, S, g, map.grp_cell, map.grp_first, map.off, map.n_groups);
    else
        k_p2g1_sorted<3><<<blocks_for(max_groups, Geo<3>::GPB), kBlock, 0, s>>>(gd, p, S, g, map.grp_cell, map.grp_first, map.off, map.n_groups);
}

void launch_g2p_p2g2_sorted(const GridDesc &gd, const PArr &p, const GArr &g, const double *na, const DevScalars *sc,
                            const SortedMap &map, int *count, unsigned long long *dest, long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_g2p_p2g2_sorted<2><<<blocks_for(max_groups, Geo<2>::GPB), kBlock, 0, s>>>(gd, p, g, na, sc, map.grp_cell, map.grp_first, map.off, map.n_groups, count, dest);
    else
        k_g2p_p2g2_sorted<3><<<blocks_for(max_groups, Geo<3>::GPB), kBlock, 0, s>>>(gd, p, g, na, sc, map.grp_cell, map.grp_first, map.off, map.n_groups, count, dest);
}

void launch_update_sorted(const GridDesc &gd, const PArr &p, const PArr &q, const double *na, const double *nb, DevScalars *sc,
                          const SortedMap &map, const int *off_new, const unsigned long long *dest, double *S_out,
                          long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_update_sorted<2><<<blocks_for(max_groups, Geo<2>::GPB), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map.grp_cell, map.grp_first, map.off, map.n_groups, off_new, dest, S_out);
    else
        k_update_sorted<3><<<blocks_for(max_groups, Geo<3>::GPB), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map.grp_cell, map.grp_first, map.off, map.n_groups, off_new, dest, S_out);
}

}  // namespace mpm
