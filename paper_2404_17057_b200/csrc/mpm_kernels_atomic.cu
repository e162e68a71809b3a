// mpm_kernels_atomic.cu -- ATOMIC kernel family: one thread per particle, global fp64 reductions (REDG.ADD.F64).
//
// This is the paper's own parallelisation (one thread per particle for P2G and G2P, atomicAdd for the P2G data
// race) with the per-quantity launches fused: one scatter kernel for m, mv, f
// (Alg. 1 l.3), one gather+scatter kernel for l.6-8, one gather+update kernel for l.10-11 and the CFL maxima.
// It works for ANY particle order, so it serves the shuffled runs of config 2 and is the parity cross-check
// of the TILED family.
//
// The kernels are written over a tensor-product SUPPORT of NS nodes per axis: NS = 2 is the paper's Q1 hat basis
// (PAPER.md:254), NS = 3 the quadratic B-spline basis it names as the next one (mpm_config.basis =
// MPM_BASIS_QUADRATIC, periodic grids only: reading A20).  Everything else of Algorithm 1 is the same code.
#include "mpm_internal.cuh"

namespace mpm {

namespace {

constexpr int kBlock = 256;

template <int DIM>
__device__ __forceinline__ void load_vec(double *const arr[3], long long k, double out[DIM])
{
#pragma unroll
    for (int a = 0; a < DIM; ++a) out[a] = arr[a][k];
}

// 1D weights and slopes of the NS^d nodes a particle sees, and the index of the first one per axis.
//   NS = 2 (Q1, A6, A19): base = cell c, w = (1 - xi, xi), slopes (-1/h, +1/h);
//   NS = 3 (quadratic B-spline N(u) = 3/4 - u^2 for |u| < 1/2, (3/2 - |u|)^2 / 2 for 1/2 <= |u| < 3/2):
//          base = floor(X/h - 1/2) (may be -1: periodic wrap), f = X/h - base in [1/2, 3/2),
//          w = ((3/2 - f)^2 / 2, 3/4 - (f - 1)^2, (f - 1/2)^2 / 2), slopes (-(3/2 - f), -2 (f - 1), f - 1/2) / h.
template <int DIM, int NS>
struct Support {
    int base[DIM];
    double w[DIM][NS], g[DIM][NS];
    static constexpr int NODES = (NS == 2) ? (1 << DIM) : (DIM == 2 ? 9 : 27);

    __device__ __forceinline__ void at(const GridDesc &gd, const double X[DIM])
    {
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            if (NS == 2) {
                double xi;
                cell_1d(X[a], gd.inv_h, gd.nc[a], base[a], xi);
                w[a][0] = 1.0 - xi; w[a][1] = xi;
                g[a][0] = -gd.inv_h; g[a][1] = gd.inv_h;
            } else {
                const double s = __dmul_rn(X[a], gd.inv_h);
                const int b = (int)floor(s - 0.5);
                const double f = s - (double)b;
                base[a] = b;
                w[a][0] = 0.5 * (1.5 - f) * (1.5 - f);
                w[a][1] = 0.75 - (f - 1.0) * (f - 1.0);
                w[a][NS - 1] = 0.5 * (f - 0.5) * (f - 0.5);
                g[a][0] = -(1.5 - f) * gd.inv_h;
                g[a][1] = -2.0 * (f - 1.0) * gd.inv_h;
                g[a][NS - 1] = (f - 0.5) * gd.inv_h;
            }
        }
    }
    // position of node q (x fastest) inside the support along axis a
    __device__ __forceinline__ static constexpr int j_of(int q, int a) { return a == 0 ? q % NS : a == 1 ? (q / NS) % NS : q / (NS * NS); }
    // global node index (periodic: node n == node 0, A11; the quadratic support wraps on both sides)
    __device__ __forceinline__ long long node(const GridDesc &gd, int q) const
    {
        long long idx = 0, stride = 1;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            int i = base[a] + j_of(q, a);
            if (NS == 2) { if (gd.per[a] && i == gd.nc[a]) i = 0; }
            else { if (i < 0) i += gd.nc[a]; else if (i >= gd.nc[a]) i -= gd.nc[a]; }
            idx += stride * (long long)i;
            stride *= (long long)gd.nn[a];
        }
        return idx;
    }
    __device__ __forceinline__ double phi(int q) const
    {
        double v = 1.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) v *= w[a][j_of(q, a)];
        return v;
    }
    __device__ __forceinline__ double dphi(int q, int a) const
    {
        double v = g[a][j_of(q, a)];
#pragma unroll
        for (int a2 = 0; a2 < DIM; ++a2)
            if (a2 != a) v *= w[a2][j_of(q, a2)];
        return v;
    }
};

// ------------------------------------------------------------------------------------------------ Alg. 1 l.3
// m_i += M phi, mv_i += M V phi, f_i += (P+Q)(M/rho) grad phi  (eqs. 13, 14, 16, 18)
template <int DIM, int NS>
__global__ void __launch_bounds__(kBlock) k_p2g1_atomic(GridDesc gd, PArr p, GArr g, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k >= n) return;
    double X[DIM], V[DIM];
    load_vec<DIM>(p.x, k, X);
    load_vec<DIM>(p.v, k, V);
    const double M = p.m[k], rho = p.rho[k], E = p.e[k], Q = p.q[k];
    Support<DIM, NS> sp;
    sp.at(gd, X);
    const double P = (gd.gamma - 1.0) * rho * E;   // eq. (3)
    const double S = (P + Q) * M / rho;            // eq. (13)
#pragma unroll
    for (int ib = 0; ib < Support<DIM, NS>::NODES; ++ib) {
        const long long i = sp.node(gd, ib);
        const double phi = sp.phi(ib);
        atomicAdd(&g.m[i], M * phi);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            atomicAdd(&g.mv[a][i], M * V[a] * phi);
            atomicAdd(&g.f[a][i], S * sp.dphi(ib, a));
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.6-8
// A = G2P(f/m); V' = V + dt A; mv2_i += M V' phi at the same weights.
// Vbar = G2P(mv'/m) is not needed here: it is gathered again, from the same node field, where it is used (l.11).
template <int DIM, int NS>
__global__ void __launch_bounds__(kBlock) k_g2p_p2g2_atomic(GridDesc gd, PArr p, GArr g, const DevScalars *sc, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k >= n) return;
    const double dt = sc->dt;
    double X[DIM], V[DIM];
    load_vec<DIM>(p.x, k, X);
    load_vec<DIM>(p.v, k, V);
    const double M = p.m[k];
    constexpr int NODES = Support<DIM, NS>::NODES;
    Support<DIM, NS> sp;
    sp.at(gd, X);
    long long node[NODES];
    double phi[NODES];
    double A[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) A[a] = 0.0;
#pragma unroll
    for (int ib = 0; ib < NODES; ++ib) {
        node[ib] = sp.node(gd, ib);
        phi[ib] = sp.phi(ib);
#pragma unroll
        for (int a = 0; a < DIM; ++a) A[a] += phi[ib] * g.acc[a][node[ib]];
    }
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        V[a] = V[a] + dt * A[a];
        p.v[a][k] = V[a];
    }
#pragma unroll
    for (int ib = 0; ib < NODES; ++ib)
#pragma unroll
        for (int a = 0; a < DIM; ++a) atomicAdd(&g.mv2[a][node[ib]], M * V[a] * phi[ib]);
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.10-13
// D = trace G2PD(mv2/m); E, rho, Q update (eq. 4); Vbar = G2P(mv'/m);
// CFL maxima over |V'|, |Vbar|, c_s (A12); X' = X + dt Vbar, wrap / recycle / clamp (PAPER.md:372-376,
// :548-554; A8, A11).
template <int DIM, int NS>
__global__ void __launch_bounds__(kBlock) k_update_atomic(GridDesc gd, PArr p, GArr g, DevScalars *sc, long long n)
{
    __shared__ double s_v[kBlock / 32], s_c[kBlock / 32];
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    const bool live = k < n;
    double vloc = 0.0, cloc = 0.0;
    int n_rec = 0, n_clamp = 0, n_neg = 0, n_nonfin = 0;
    if (live) {
        const double dt = sc->dt;
        double X[DIM], V[DIM];
        load_vec<DIM>(p.x, k, X);
        load_vec<DIM>(p.v, k, V);
        double rho = p.rho[k], E = p.e[k], Q;
        Support<DIM, NS> sp;
        sp.at(gd, X);
        double D = 0.0, Vb[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) Vb[a] = 0.0;
#pragma unroll
        for (int ib = 0; ib < Support<DIM, NS>::NODES; ++ib) {
            const long long i = sp.node(gd, ib);
            const double phi = sp.phi(ib);
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                D += g.v2[a][i] * sp.dphi(ib, a);
                Vb[a] += phi * g.vbar[a][i];
            }
        }
        // particle thermodynamics, exactly the printed formulas; Q from eq. (4) with the D just gathered and the
        // un-primed rho, P (eqs. 5a/5b use one div v for q and for the energy equation; reading A2)
        const double P = (gd.gamma - 1.0) * rho * E;
        double Qn = 0.0;
        if (D < 0.0) {
            const double cs0 = sqrt(gd.gamma * P / rho);
            if (gd.visc_form == MPM_VISC_STANDARD)
                Qn = rho * (gd.c0 * gd.h * gd.h * D * D - gd.c1 * gd.h * cs0 * D);
            else
                Qn = gd.c0 * (rho * gd.h * D) * (rho * gd.h * D) - gd.c1 * gd.h * cs0 * D;
        }
        const double En = E + dt * (-(P + Qn) / rho) * D;
        const double jac = 1.0 + dt * D;
        if (jac <= 0.0) n_neg = 1;
        const double rhon = rho / jac;
        const double Pn = (gd.gamma - 1.0) * rhon * En;
        const double cs = sqrt(gd.gamma * Pn / rhon);
        if (!isfinite(En) || !isfinite(rhon)) n_nonfin = 1;
        // CFL maxima on V', Vbar, rho', E' before recycling (A12)
        double v2 = 0.0, vb2 = 0.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            v2 += V[a] * V[a];
            vb2 += Vb[a] * Vb[a];
        }
        vloc = fmax(sqrt(v2), sqrt(vb2));
        cloc = cs;
        // advection
        bool recycle = false;
        double Xn[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            double x = X[a] + dt * Vb[a];
            if (gd.per[a]) {
                x = x - gd.L[a] * floor(x / gd.L[a]);
                if (x >= gd.L[a]) x = 0.0;
            } else {
                if (x < 0.0 && gd.bc[a][0] == MPM_BC_OUTFLOW) recycle = true;
                if (x > gd.L[a] && gd.bc[a][1] == MPM_BC_OUTFLOW) recycle = true;
            }
            Xn[a] = x;
        }
        double Mn = 0.0;
        bool rewrite = false;
        if (recycle && gd.in_axis >= 0) {
            const long long id = p.id[k];
            const long long step = sc->step;
            int j = 0;
            const double u0 = recycle_uniform(gd.recycle_seed, id, step, j++);
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                if (a == gd.in_axis) {
                    Xn[a] = (gd.in_side == 0) ? u0 * gd.h : gd.L[a] - u0 * gd.h;
                } else {
                    const double u1 = recycle_uniform(gd.recycle_seed, id, step, j++);
                    const double u2 = recycle_uniform(gd.recycle_seed, id, step, j++);
                    const bool slab = gd.slab_global_n > 0 && a == DIM - 1;      // see lg::move_particle
                    const int na = slab ? gd.slab_global_n : gd.nc[a];
                    int cell = (int)floor(u1 * (double)na);
                    cell = min(cell, na - 1) - (slab ? gd.slab_offset : 0);
                    Xn[a] = ((double)cell + u2) * gd.h;
                }
                V[a] = gd.inflow_v[a];
            }
            rho = gd.inflow_rho;
            E = gd.inflow_e;
            Q = 0.0;
            Mn = gd.inflow_mass;
            rewrite = true;
            n_rec = 1;
        } else {
            rho = rhon;
            E = En;
            Q = Qn;
        }
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            if (!gd.per[a]) {
                if (Xn[a] < 0.0 && gd.bc[a][0] != MPM_BC_OPEN) { Xn[a] = 0.0; n_clamp++; }
                if (Xn[a] > gd.L[a] && gd.bc[a][1] != MPM_BC_OPEN) { Xn[a] = gd.L[a]; n_clamp++; }
            }
            p.x[a][k] = Xn[a];
        }
        p.rho[k] = rho;
        p.e[k] = E;
        p.q[k] = Q;
        if (rewrite) {
            p.m[k] = Mn;
#pragma unroll
            for (int a = 0; a < DIM; ++a) p.v[a][k] = V[a];
        }
    }
    // block maxima -> one atomicMax per block (max is order-free, so this is exact)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        vloc = fmax(vloc, __shfl_xor_sync(0xffffffffu, vloc, o));
        cloc = fmax(cloc, __shfl_xor_sync(0xffffffffu, cloc, o));
    }
    // NaN must not be lost by fmax: flag it through the counters instead (n_nonfinite)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) { s_v[warp] = vloc; s_c[warp] = cloc; }
    const unsigned any_rec = __ballot_sync(0xffffffffu, n_rec), any_neg = __ballot_sync(0xffffffffu, n_neg),
                   any_nf = __ballot_sync(0xffffffffu, n_nonfin);
    int clamp_sum = n_clamp;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) clamp_sum += __shfl_xor_sync(0xffffffffu, clamp_sum, o);
    if (lane == 0) {
        if (any_rec) atomicAdd(&sc->n_recycled, (unsigned long long)__popc(any_rec));
        if (any_neg) atomicAdd(&sc->n_negjac, (unsigned long long)__popc(any_neg));
        if (any_nf) atomicAdd(&sc->n_nonfinite, (unsigned long long)__popc(any_nf));
        if (clamp_sum) atomicAdd(&sc->n_clamped, (unsigned long long)clamp_sum);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = s_v[0], c = s_c[0];
#pragma unroll
        for (int w = 1; w < kBlock / 32; ++w) { v = fmax(v, s_v[w]); c = fmax(c, s_c[w]); }
        atomic_max_nonneg(&sc->vmax_bits, v);
        atomic_max_nonneg(&sc->cmax_bits, c);
    }
}

inline unsigned grid_for(long long n) { return (unsigned)((n + kBlock - 1) / kBlock); }

}  // namespace

void launch_p2g1_atomic(const GridDesc &gd, const PArr &p, const GArr &g, long long n, cudaStream_t s)
{
    if (n <= 0) return;
    if (gd.quadratic) {
        if (gd.dim == 2) k_p2g1_atomic<2, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, n);
        else k_p2g1_atomic<3, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, n);
    } else if (gd.dim == 2) k_p2g1_atomic<2, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, n);
    else k_p2g1_atomic<3, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, n);
}

void launch_g2p_p2g2_atomic(const GridDesc &gd, const PArr &p, const GArr &g, const DevScalars *sc, long long n,
                            cudaStream_t s)
{
    if (n <= 0) return;
    if (gd.quadratic) {
        if (gd.dim == 2) k_g2p_p2g2_atomic<2, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
        else k_g2p_p2g2_atomic<3, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
    } else if (gd.dim == 2) k_g2p_p2g2_atomic<2, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
    else k_g2p_p2g2_atomic<3, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
}

void launch_update_atomic(const GridDesc &gd, const PArr &p, const GArr &g, DevScalars *sc, long long n, cudaStream_t s)
{
    if (n <= 0) return;
    if (gd.quadratic) {
        if (gd.dim == 2) k_update_atomic<2, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
        else k_update_atomic<3, 3><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
    } else if (gd.dim == 2) k_update_atomic<2, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
    else k_update_atomic<3, 2><<<grid_for(n), kBlock, 0, s>>>(gd, p, g, sc, n);
}

}  // namespace mpm
