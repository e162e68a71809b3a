// mpm_kernels_grid.cu -- node kernels (one thread per node) and the device-resident time-loop scalars.
//
//   node1 : Alg. 1 l.4-5  BC + obstacle on (mv, f) (eqs. 21, 22, 30), mv' = mv + dt f,
//           plus the node velocities the gathers read: vbar = mv'/m, acc = f/m (theta of PAPER.md:295; ratio := 0 where
//           m = 0, reading A5) and the reset of mv2 for l.8.
//   node2 : Alg. 1 l.9    BC on mv2, v2 = mv2/m.
//   begin/end_step : dt from the CFL reduction (eq. 25/29), t += dt -- no host round trip.
#include "mpm_node_bc.cuh"

namespace mpm {

namespace {

constexpr int kBlock = 256;

template <int DIM>
__device__ __forceinline__ void node_coords(const GridDesc &gd, long long i, int idx[DIM])
{
    long long r = i;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        idx[a] = (int)(r % gd.nn[a]);
        r /= gd.nn[a];
    }
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_node1(GridDesc gd, GArr g, const DevScalars *sc, bool zero_mv2)
{
    const long long i = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (i >= gd.Nn) return;
    const double dt = sc->dt;
    int idx[DIM];
    node_coords<DIM>(gd, i, idx);
    const double m = g.m[i];
    double mv[DIM], f[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) { mv[a] = g.mv[a][i]; f[a] = g.f[a][i]; }
    apply_bc<DIM, true>(gd, g, i, idx, m, mv, f);
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        const double mvp = mv[a] + dt * f[a];
        g.mv[a][i] = mvp;
        g.f[a][i] = f[a];
        const double vb = (m != 0.0) ? mvp / m : 0.0;
        const double ac = (m != 0.0) ? f[a] / m : 0.0;
        if (g.vbar[a]) {
            g.vbar[a][i] = vb;
            g.acc[a][i] = ac;
        }
        if (zero_mv2) g.mv2[a][i] = 0.0;
    }
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_node2(GridDesc gd, GArr g)
{
    const long long i = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (i >= gd.Nn) return;
    int idx[DIM];
    node_coords<DIM>(gd, i, idx);
    const double m = g.m[i];
    double mv[DIM], f[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) { mv[a] = g.mv2[a][i]; f[a] = 0.0; }
    apply_bc<DIM, false>(gd, g, i, idx, m, mv, f);
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        g.mv2[a][i] = mv[a];
        const double v2 = (m != 0.0) ? mv[a] / m : 0.0;
        if (g.v2[a]) g.v2[a][i] = v2;
    }
}

// dt of the step (eq. 25/29).  A state with v_max + c_max = 0 (cold gas at rest) or a non-finite
// maximum has no CFL step: dt := 0 for this step (nothing moves, nothing becomes NaN) and the event is counted; mpm_step
// reports it as MPM_E_NONFINITE when the caller asks for dt_last, mpm_get_stats shows the counter.
__global__ void k_begin_step(DevScalars *sc, double h, int have_particles)
{
    double dt = sc->dt_fixed;
    if (!(dt > 0.0)) {
        dt = sc->alpha * h / (sc->vmax + sc->cmax);
        if (!(dt > 0.0) || !isfinite(dt)) {
            dt = 0.0;
            if (have_particles) sc->n_bad_dt += 1ull;
        }
    }
    sc->dt = dt;
    sc->vmax_bits = 0ull;
    sc->cmax_bits = 0ull;
}

__global__ void k_end_step(DevScalars *sc, double h)
{
    sc->vmax = __longlong_as_double((long long)sc->vmax_bits);
    sc->cmax = __longlong_as_double((long long)sc->cmax_bits);
    const double dtn = sc->alpha * h / (sc->vmax + sc->cmax);
    sc->dt_next = (dtn > 0.0 && isfinite(dtn)) ? dtn : 0.0;
    sc->t += sc->dt;
    sc->step += 1;
}

// first CFL reduction from the loaded state: |V| and c_s = sqrt(gamma P / rho) (reading A13)
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_initial_cfl(GridDesc gd, PArr p, DevScalars *sc, long long n)
{
    __shared__ double s_v[kBlock / 32], s_c[kBlock / 32];
    double vloc = 0.0, cloc = 0.0;
    for (long long k = (long long)blockIdx.x * kBlock + threadIdx.x; k < n; k += (long long)gridDim.x * kBlock) {
        double v2 = 0.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) { const double v = p.v[a][k]; v2 += v * v; }
        const double rho = p.rho[k];
        const double P = (gd.gamma - 1.0) * rho * p.e[k];
        vloc = fmax(vloc, sqrt(v2));
        cloc = fmax(cloc, sqrt(gd.gamma * P / rho));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        vloc = fmax(vloc, __shfl_xor_sync(0xffffffffu, vloc, o));
        cloc = fmax(cloc, __shfl_xor_sync(0xffffffffu, cloc, o));
    }
    if ((threadIdx.x & 31) == 0) { s_v[threadIdx.x >> 5] = vloc; s_c[threadIdx.x >> 5] = cloc; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kBlock / 32; ++w) { vloc = fmax(vloc, s_v[w]); cloc = fmax(cloc, s_c[w]); }
        atomic_max_nonneg(&sc->vmax_bits, fmax(vloc, s_v[0]));
        atomic_max_nonneg(&sc->cmax_bits, fmax(cloc, s_c[0]));
    }
}

__global__ void k_finish_initial_cfl(DevScalars *sc)
{
    sc->vmax = __longlong_as_double((long long)sc->vmax_bits);
    sc->cmax = __longlong_as_double((long long)sc->cmax_bits);
}

// diagnostics on demand: sum M, sum M V, sum M (E + |V|^2 / 2)
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_stats_reduce(PArr p, DevScalars *sc, long long n)
{
    __shared__ double s[kBlock / 32][5];
    double acc[5] = { 0, 0, 0, 0, 0 };
    for (long long k = (long long)blockIdx.x * kBlock + threadIdx.x; k < n; k += (long long)gridDim.x * kBlock) {
        const double M = p.m[k];
        double v2 = 0.0;
        acc[0] += M;
#pragma unroll
        for (int a = 0; a < DIM; ++a) { const double v = p.v[a][k]; acc[1 + a] += M * v; v2 += v * v; }
        acc[4] += M * (p.e[k] + 0.5 * v2);
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

__global__ void k_stats_clear(DevScalars *sc)
{
    sc->sum_mass = 0.0; sc->sum_energy = 0.0;
    sc->sum_mom[0] = sc->sum_mom[1] = sc->sum_mom[2] = 0.0;
}

// diagnostics, off the hot path: one thread per particle (ATOMIC layout) or per group record (TILED layout)
template <int DIM>
__device__ __forceinline__ void diag_scatter(const GridDesc &gd, const PArr &p, const double *field, double *num, double *den, long long k)
{
    double X[DIM], xi[DIM];
    int c[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) X[a] = p.x[a][k];
    particle_cell<DIM>(gd, X, c, xi);
    const double M = p.m[k], a = field[k];
#pragma unroll
    for (int ib = 0; ib < (1 << DIM); ++ib) {
        const long long i = corner_node<DIM>(gd, c, ib);
        const double phi = corner_phi<DIM>(xi, ib);
        atomicAdd(&num[i], M * a * phi);
        atomicAdd(&den[i], M * phi);
    }
}
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_grid_diagnostic(GridDesc gd, PArr p, const double *field, double *num, double *den,
                                                            long long n, SortedMap map)
{
    if (map.groups) {
        const int n_groups = *map.n_groups;
        for (long long gq = (long long)blockIdx.x * kBlock + threadIdx.x; gq < n_groups; gq += (long long)gridDim.x * kBlock) {
            const int4 r = map.groups[gq];
            for (int j = 0; j < (r.y & 0xff); ++j) diag_scatter<DIM>(gd, p, field, num, den, (long long)r.x + j);
        }
    } else {
        for (long long k = (long long)blockIdx.x * kBlock + threadIdx.x; k < n; k += (long long)gridDim.x * kBlock)
            diag_scatter<DIM>(gd, p, field, num, den, k);
    }
}
__global__ void __launch_bounds__(kBlock) k_safe_quotient(double *num, const double *den, long long n)
{
    for (long long i = (long long)blockIdx.x * kBlock + threadIdx.x; i < n; i += (long long)gridDim.x * kBlock)
        num[i] = (den[i] != 0.0) ? num[i] / den[i] : 0.0;
}

inline unsigned grid_for(long long n) { return (unsigned)((n + kBlock - 1) / kBlock); }

}  // namespace

void launch_grid_diagnostic(const GridDesc &gd, const PArr &p, const double *field, double *num, double *den, long long n,
                            const SortedMap &map, long long max_groups, cudaStream_t s)
{
    const long long work = map.groups ? max_groups : n;
    if (work > 0) {
        const unsigned blocks = (unsigned)((work + kBlock - 1) / kBlock < 148 * 16 ? (work + kBlock - 1) / kBlock : 148 * 16);
        if (gd.dim == 2) k_grid_diagnostic<2><<<blocks, kBlock, 0, s>>>(gd, p, field, num, den, n, map);
        else k_grid_diagnostic<3><<<blocks, kBlock, 0, s>>>(gd, p, field, num, den, n, map);
    }
    k_safe_quotient<<<148 * 4, kBlock, 0, s>>>(num, den, gd.Nn);
}

void launch_grid_clear(const GridDesc &gd, const GArr &g, cudaStream_t s)
{
    // Alg. 1 l.2 grid reset; flags and normals are static
    cudaMemsetAsync(g.m, 0, sizeof(double) * (size_t)gd.Nn, s);
    for (int a = 0; a < gd.dim; ++a) {
        cudaMemsetAsync(g.mv[a], 0, sizeof(double) * (size_t)gd.Nn, s);
        cudaMemsetAsync(g.f[a], 0, sizeof(double) * (size_t)gd.Nn, s);
    }
}

void launch_node1(const GridDesc &gd, const GArr &g, const DevScalars *sc, cudaStream_t s, bool zero_mv2)
{
    if (gd.dim == 2) k_node1<2><<<grid_for(gd.Nn), kBlock, 0, s>>>(gd, g, sc, zero_mv2);
    else k_node1<3><<<grid_for(gd.Nn), kBlock, 0, s>>>(gd, g, sc, zero_mv2);
}

void launch_node2(const GridDesc &gd, const GArr &g, cudaStream_t s)
{
    if (gd.dim == 2) k_node2<2><<<grid_for(gd.Nn), kBlock, 0, s>>>(gd, g);
    else k_node2<3><<<grid_for(gd.Nn), kBlock, 0, s>>>(gd, g);
}

void launch_begin_step(DevScalars *sc, double h, bool have_particles, cudaStream_t s) { k_begin_step<<<1, 1, 0, s>>>(sc, h, have_particles ? 1 : 0); }
void launch_end_step(DevScalars *sc, double h, cudaStream_t s) { k_end_step<<<1, 1, 0, s>>>(sc, h); }

void launch_initial_cfl(const GridDesc &gd, const PArr &p, DevScalars *sc, long long n, cudaStream_t s)
{
    const unsigned blocks = (unsigned)((n + kBlock - 1) / kBlock < 148 * 8 ? (n + kBlock - 1) / kBlock : 148 * 8);
    if (n > 0) {
        if (gd.dim == 2) k_initial_cfl<2><<<blocks, kBlock, 0, s>>>(gd, p, sc, n);
        else k_initial_cfl<3><<<blocks, kBlock, 0, s>>>(gd, p, sc, n);
    }
    k_finish_initial_cfl<<<1, 1, 0, s>>>(sc);
}

void launch_stats_reduce(const GridDesc &gd, const PArr &p, DevScalars *sc, long long n, cudaStream_t s)
{
    k_stats_clear<<<1, 1, 0, s>>>(sc);
    if (n <= 0) return;
    const unsigned blocks = (unsigned)((n + kBlock - 1) / kBlock < 148 * 8 ? (n + kBlock - 1) / kBlock : 148 * 8);
    if (gd.dim == 2) k_stats_reduce<2><<<blocks, kBlock, 0, s>>>(p, sc, n);
    else k_stats_reduce<3><<<blocks, kBlock, 0, s>>>(p, sc, n);
}

}  // namespace mpm
