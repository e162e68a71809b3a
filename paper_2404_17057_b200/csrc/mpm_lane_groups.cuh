// mpm_lane_groups.cuh -- device helpers of the TILED kernel family: lane-group geometry, the transposed butterfly
// reduction, corner weights in butterfly order, the P2G#1 of a particle whose cell is not its group's cell (after a load
// only), and the particle move of Alg. 1 l.11.
#pragma once
#include "mpm_internal.cuh"

namespace mpm {
namespace lg {

constexpr int kBlock = 256;
constexpr unsigned kFull = 0xffffffffu;

template <int DIM>
struct Geo {
    static constexpr int NB = 1 << DIM;            // corners per cell = particles per group
    static constexpr int LG = NB / 2;              // lanes per group
    static constexpr int NG = 32 / LG;             // groups per warp
    static constexpr int GPB = kBlock / LG;        // groups per block and iteration
};

__device__ __forceinline__ double shfl_xor_d(double v, int m) { return __shfl_xor_sync(kFull, v, m); }

// Transposed butterfly over the LG lanes of a group.  Before: register r of lane l holds the lane's contribution to
// corner r ^ l.  After: registers r = q * LG (q = 0, 1) hold the group totals of corners l + q * LG.
template <int DIM>
__device__ __forceinline__ void butterfly(double v[1 << DIM])
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG;
#pragma unroll
    for (int m = LG / 2; m >= 1; m >>= 1) {
#pragma unroll
        for (int r = 0; r < NB; ++r)
            if ((r & m) == 0 && (r & (LG - 1) & ~(2 * m - 1)) == 0) v[r] += shfl_xor_d(v[r | m], m);
    }
}

struct Group {
    int first;     // first particle of the group
    int cnt;       // particles in the group (<= 2^d), 0 = idle
    int cell;      // cell key
    int cpack;     // packed cell coordinates (3D: 10 bits each, 2D: 16 bits each)
    int multi;     // the cell has more than one group (more than 2^d particles)
};

__device__ __forceinline__ Group fetch_group(const int4 *__restrict__ groups, long long gidx, int n_groups)
{
    Group g{ 0, 0, 0, 0, 0 };
    if (gidx < (long long)n_groups) {
        const int4 r = __ldg(groups + gidx);      // {first slot, count | multi << 8, key, packed coordinates}
        g.first = r.x; g.cnt = r.y & 0xff; g.multi = r.y >> 8; g.cell = r.z; g.cpack = r.w;
    }
    return g;
}

template <int DIM>
__device__ __forceinline__ void unpack_coords(int cpack, int c[DIM])
{
    if (DIM == 3) { c[0] = cpack & 1023; c[1] = (cpack >> 10) & 1023; c[DIM - 1] = (cpack >> 20) & 1023; }
    else { c[0] = cpack & 65535; c[1] = (cpack >> 16) & 65535; }
}

// node index of corner b of cell c (periodic wrap: node n == node 0, A11)
template <int DIM>
__device__ __forceinline__ int corner_node_i(const GridDesc &gd, const int c[DIM], int b)
{
    int idx = 0, stride = 1;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int i = c[a] + ((b >> a) & 1);
        if (gd.per[a] && i == gd.nc[a]) i = 0;
        idx += stride * i;
        stride *= gd.nn[a];
    }
    return idx;
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

// corner weights in butterfly order (scatters): register r of lane l holds the weight of corner r ^ l (l < LG)
template <int DIM>
__device__ __forceinline__ void swizzled_weights(const double xi[DIM], int l, double w[1 << DIM])
{
    double p[DIM][2];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const bool hi = (l >> a) & 1;       // l < LG: only the low axes are ever swapped
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

// max over the warp of a NON-NEGATIVE double with two integer REDUX ops (bit patterns order like the values)
__device__ __forceinline__ double warp_max_nonneg(double v)
{
    const unsigned hi = (unsigned)__double2hiint(v), lo = (unsigned)__double2loint(v);
    const unsigned mhi = __reduce_max_sync(kFull, hi);
    const unsigned mlo = __reduce_max_sync(kFull, hi == mhi ? lo : 0u);
    return __hiloint2double((int)mhi, (int)mlo);
}

// ---------------------------------------------------------------------------------------------- slow paths
template <int DIM, bool ACC32 = false>
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
        if (ACC32) {      // fp32 grid accumulation (TILED family only): node-major float nm[N_n][8] = { m, mv[3], f[3], - }
            float *nm = reinterpret_cast<float *>(g.m) + 8 * i;
            atomicAdd(nm, (float)(M * phi));
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                atomicAdd(nm + 1 + a, (float)(M * V[a] * phi));
                atomicAdd(nm + 4 + a, (float)(S * corner_dphi<DIM>(xi, ib, a, gd.inv_h)));
            }
            continue;
        }
        atomicAdd(&g.m[i], M * phi);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            atomicAdd(&g.mv[a][i], M * V[a] * phi);
            atomicAdd(&g.f[a][i], S * corner_dphi<DIM>(xi, ib, a, gd.inv_h));
        }
    }
}

// ---------------------------------------------------------------------------------------------- shared pieces

// Alg. 1 l.11 for one particle: X' = X + dt Vbar, periodic wrap (A11), outflow detection, recycling position (A8),
// clamp.  Used by BOTH the gather kernel (to find the new cell) and the update kernel (to write X'): every rounding is
// explicit (fma / __dmul_rn / __dsub_rn), so that both kernels get the same X' bit for bit from the same inputs.
template <int DIM>
__device__ __forceinline__ void move_particle(const GridDesc &gd, const double X[DIM], const double Vb[DIM], double dt,
                                              long long id, long long step, double Xn[DIM], bool &recycled, int &nclamp,
                                              bool *left_slab = nullptr)
{
    bool recycle = false;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double x = fma(dt, Vb[a], X[a]);
        if (gd.per[a]) {
            if (x < 0.0 || x >= gd.L[a]) {
                x = __dsub_rn(x, __dmul_rn(gd.L[a], floor(x / gd.L[a])));
                if (x >= gd.L[a]) x = 0.0;
            }
        } else {
            if (x < 0.0 && gd.bc[a][0] == MPM_BC_OUTFLOW) recycle = true;
            if (x > gd.L[a] && gd.bc[a][1] == MPM_BC_OUTFLOW) recycle = true;
        }
        Xn[a] = x;
    }
    recycled = recycle && gd.in_axis >= 0;
    if (recycled) {
        // j = 0: offset normal to the inflow face; every other axis, in order, takes the next two numbers (cell, offset).
        // Written as selects on a compile-time axis: an indexed store Xn[in_axis] would put Xn into local memory.
        const double off = __dmul_rn(recycle_uniform(gd.recycle_seed, id, step, 0), gd.h);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const int jb = 1 + 2 * (a - (a > gd.in_axis ? 1 : 0));
            const double u1 = recycle_uniform(gd.recycle_seed, id, step, jb);
            const double u2 = recycle_uniform(gd.recycle_seed, id, step, jb + 1);
            // a slab of a larger domain (last axis): the inflow face is the GLOBAL one, the cell index is made slab-local
            const bool slab = gd.slab_global_n > 0 && a == DIM - 1;
            const int na = slab ? gd.slab_global_n : gd.nc[a];
            int cell = (int)floor(u1 * (double)na);
            cell = min(cell, na - 1) - (slab ? gd.slab_offset : 0);
            const double x_face = (gd.in_side == 0) ? off : __dsub_rn(gd.L[a], off);
            const double x_other = ((double)cell + u2) * gd.h;
            Xn[a] = (a == gd.in_axis) ? x_face : x_other;
        }
    }
    nclamp = 0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (!gd.per[a]) {      // an OPEN face is an interface to the neighbouring slab: the particle leaves, unclamped
            if (Xn[a] < 0.0) { if (gd.bc[a][0] != MPM_BC_OPEN) { Xn[a] = 0.0; nclamp++; } else if (left_slab) *left_slab = true; }
            if (Xn[a] >= gd.L[a]) {
                if (gd.bc[a][1] == MPM_BC_OPEN) { if (left_slab) *left_slab = true; }
                else if (Xn[a] > gd.L[a]) { Xn[a] = gd.L[a]; nclamp++; }
            }
        }
    }
}

}  // namespace lg
}  // namespace mpm
