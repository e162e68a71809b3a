// mpm_kernels_sorted.cu -- SORTED kernel family: particles are kept EXACTLY cell-sorted every step and processed in
// aligned lane groups, one cell per group.  A group has LG = 2^d / 2 lanes (4 in 3D, 2 in 2D) and holds up to 2^d
// particles of one cell, two per lane (lane l takes particles first + l and first + LG + l).
//
// What this buys over the paper's one-thread-per-particle + atomicAdd design:
//   * scatters (Alg. 1 l.3 and l.8): a lane adds up the contributions of its two particles to the 2^d corners of the
//     cell in registers, the group sums them with a transposed XOR butterfly (2^d - 2 shuffles per channel) after which
//     lane l owns the totals of corners l and l + LG, and issues ONE global fp64 reduction per corner and channel:
//     2^d x fewer REDs than one atomicAdd per particle, corner and channel.
//     (Shared-memory fp64 atomicAdd is a CAS loop on sm_100a -- ATOMS.CAST.SPIN.64 -- so it is never used.)
//   * gathers (l.6, l.10, l.11): lane l fetches the node values of corners l and l + LG once per group (16-byte loads
//     from node-major arrays), parks them in shared memory, and every lane reads all corners back as conflict-free
//     128-bit broadcasts: 2^d x fewer global gathers.
//   * gradient channels are folded into phi-weighted channels using sum_{b_a} w_a(b_a) = 1:
//       f_a(b) = +-(1/h) sum_{b_a} T_S(b),  T_S(b) = sum_k S_k phi_b(X_k)             (P2G#1: 1+d+1 channels, not 1+2d)
//       D_k    = sum_b phi_b(X_k) sum_a (v2_a(b | a) - v2_a(b & ~a))/h                (G2PD  : 1 channel, not d)
//   * the re-ordering (l.12) is fused into the sweeps: the gather kernel of l.6-8 computes each particle's new cell
//     and its rank in it (one returning integer atomic), a scan of the per-cell counts gives the new cell offsets, and
//     the update kernel of l.10-11 writes every particle straight to its sorted slot in the other buffer: no
//     separate permutation pass.
//   * kernels are persistent (grid = a multiple of the SM count, grid-stride loop over 16-byte group records, the
//     next record prefetched while the current group is processed), so the dependent chain in front of the particle
//     loads is one load deep.
// A particle whose true cell differs from its group's cell (never the case when the invariant holds; cheap to test)
// takes a slow path with direct global reductions / gathers, so correctness never depends on the ordering.
#include "mpm_lane_groups.cuh"

#ifndef MPM_MINB
#define MPM_MINB 2   // resident blocks per SM the particle kernels are compiled for (register budget)
#endif

namespace mpm {

namespace {

using namespace lg;

// ------------------------------------------------------------------------------------------------ Alg. 1 l.3
// m, mv from phi-weighted channels (M, M V); f from the phi-weighted channel S = (P+Q) M / rho
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_p2g1_sorted(GridDesc gd, PArr p, const double *__restrict__ Sarr, GArr g,
                                                        const int4 *__restrict__ groups, const int *__restrict__ n_groups_p)
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = Geo<DIM>::GPB;
    const int n_groups = *n_groups_p;
    const int l = threadIdx.x % LG;
    const long long stride = (long long)gridDim.x * GPB;
    long long gidx = (long long)blockIdx.x * GPB + threadIdx.x / LG;
    Group next = fetch_group(groups, gidx, n_groups);
    for (long long g0 = (long long)blockIdx.x * GPB; g0 < n_groups; g0 += stride, gidx += stride) {
        const Group grp = next;
        next = fetch_group(groups, gidx + stride, n_groups);
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        // issue all particle loads first
        double X[2][DIM], V[2][DIM], M[2], S[2];
        bool valid[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            valid[i] = (l + LG * i) < grp.cnt;
            const long long k = valid[i] ? (long long)grp.first + l + LG * i : 0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) { X[i][a] = valid[i] ? p.x[a][k] : 0.0; V[i][a] = valid[i] ? p.v[a][k] : 0.0; }
            M[i] = valid[i] ? p.m[k] : 0.0;
            S[i] = valid[i] ? Sarr[k] : 0.0;
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
        // lane totals per corner, then group totals: channels M, M V_a, S
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
        // forces of corners b_q = l + q LG: f_a = +-(1/h) (T_S(b) + T_S(b ^ bit_a)), + on the high side of axis a
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
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.6-8 (+ l.11-12 bookkeeping)
// A = G2P(f/m), Vbar = G2P(mv'/m); V' = V + dt A; mv2 += M V' phi.  Also: the particle's cell after the
// move of l.11 and its rank inside that cell, for the fused re-ordering.  V' is NOT stored: the update kernel recomputes it.
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_g2p_p2g2_sorted(GridDesc gd, PArr p, GArr g, const double *__restrict__ na,
                                                            const DevScalars *__restrict__ sc,
                                                            const int4 *__restrict__ groups, const int *__restrict__ n_groups_p,
                                                            int *__restrict__ count, unsigned long long *__restrict__ dest)
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = Geo<DIM>::GPB;
    __shared__ __align__(16) double s_vals[(kBlock / 32) * Geo<DIM>::WARP_DOUBLES];
    const int n_groups = *n_groups_p;
    const double dt = sc->dt;
    const long long step = sc->step;
    const int l = threadIdx.x % LG;
    const int warp = threadIdx.x >> 5, gi = (threadIdx.x & 31) / LG;
    double *s_group = s_vals + warp * Geo<DIM>::WARP_DOUBLES + gi * Geo<DIM>::GROUP_STRIDE;
    const long long stride = (long long)gridDim.x * GPB;
    long long gidx = (long long)blockIdx.x * GPB + threadIdx.x / LG;
    Group next = fetch_group(groups, gidx, n_groups);
    for (long long g0 = (long long)blockIdx.x * GPB; g0 < n_groups; g0 += stride, gidx += stride) {
        const Group grp = next;
        next = fetch_group(groups, gidx + stride, n_groups);
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        double X[2][DIM], V[2][DIM], M[2];
        int id[2];
        bool valid[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            valid[i] = (l + LG * i) < grp.cnt;
            const long long k = valid[i] ? (long long)grp.first + l + LG * i : 0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) { X[i][a] = valid[i] ? p.x[a][k] : 0.0; V[i][a] = valid[i] ? p.v[a][k] : 0.0; }
            M[i] = valid[i] ? p.m[k] : 0.0;
            id[i] = valid[i] ? p.id[k] : 0;
        }
        int node[2];
#pragma unroll
        for (int q = 0; q < 2; ++q) node[q] = corner_node_i<DIM>(gd, c, l + q * LG);
        if (grp.cnt > 0) {
#pragma unroll
            for (int q = 0; q < 2; ++q) stage_na<DIM>(na, node[q], s_group + (l + q * LG) * Geo<DIM>::CH);
        }
        __syncwarp();
        double ws[2][NB], MV[2][DIM];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
#pragma unroll
            for (int r = 0; r < NB; ++r) ws[i][r] = 0.0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) MV[i][a] = 0.0;
            if (valid[i]) {
                const long long k = (long long)grp.first + l + LG * i;
                double xi[DIM], Vb[DIM], A[DIM];
                const bool fast = local_coords<DIM>(gd, X[i], c, xi);
                if (fast) {
                    double w[NB], out[2 * DIM];
                    natural_weights<DIM>(xi, w);
                    gather_pairs<DIM, DIM>(s_group, w, out);
#pragma unroll
                    for (int a = 0; a < DIM; ++a) { Vb[a] = out[a]; A[a] = out[DIM + a]; }
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
                // where the particle will be after l.11, and its rank among the particles that end up in that cell
                double Xn[DIM];
                bool recycled;
                int nclamp;
                move_particle<DIM>(gd, X[i], Vb, dt, (long long)id[i], step, Xn, recycled, nclamp);
                const int key = cell_key<DIM>(gd, Xn);
                const int rank = atomicAdd(&count[key], 1);
                dest[k] = ((unsigned long long)(unsigned)key << 32) | (unsigned)rank;
            }
        }
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
            for (int q = 0; q < 2; ++q)
#pragma unroll
                for (int a = 0; a < DIM; ++a) atomicAdd(&g.mv2[a][node[q]], tot[a][q]);
        }
        __syncwarp();      // the staging area is rewritten by the next iteration
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.10-13
// D = trace G2PD(mv2/m); Q (eq. 4), E', rho'; V' = V + dt A again; CFL maxima;
// X' = X + dt Vbar; the particle is written to its cell-sorted slot of the OTHER buffer (l.12),
// together with next step's force payload S' = (P'+Q') M / rho' (eq. 13).
template <int DIM>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_update_sorted(GridDesc gd, PArr p, PArr q, const double *__restrict__ na,
                                                          const double *__restrict__ nb, DevScalars *sc,
                                                          const int4 *__restrict__ groups, const int *__restrict__ n_groups_p,
                                                          const int *__restrict__ off_new,
                                                          const unsigned long long *__restrict__ dest, double *__restrict__ S_out)
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = Geo<DIM>::GPB;
    constexpr int NPAIR = (DIM == 3) ? 4 : 3;
    __shared__ __align__(16) double s_vals[(kBlock / 32) * Geo<DIM>::WARP_DOUBLES];
    __shared__ double s_v[kBlock / 32], s_c[kBlock / 32];
    const int n_groups = *n_groups_p;
    const double dt = sc->dt;
    const long long step = sc->step;
    const int l = threadIdx.x % LG;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, gi = lane / LG;
    double *s_group = s_vals + warp * Geo<DIM>::WARP_DOUBLES + gi * Geo<DIM>::GROUP_STRIDE;
    const long long stride = (long long)gridDim.x * GPB;
    long long gidx = (long long)blockIdx.x * GPB + threadIdx.x / LG;
    Group next = fetch_group(groups, gidx, n_groups);
    double vloc = 0.0, cloc = 0.0;
    int n_rec = 0, n_clamp = 0, n_neg = 0, n_nonfin = 0;
    const double gm1 = gd.gamma - 1.0;
    for (long long g0 = (long long)blockIdx.x * GPB; g0 < n_groups; g0 += stride, gidx += stride) {
        const Group grp = next;
        next = fetch_group(groups, gidx + stride, n_groups);
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        double X[2][DIM], V[2][DIM], M[2], rho[2], E[2];
        int id[2];
        unsigned long long dk[2];
        bool valid[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            valid[i] = (l + LG * i) < grp.cnt;
            const long long k = valid[i] ? (long long)grp.first + l + LG * i : 0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) { X[i][a] = valid[i] ? p.x[a][k] : 0.0; V[i][a] = valid[i] ? p.v[a][k] : 0.0; }
            M[i] = valid[i] ? p.m[k] : 0.0;
            rho[i] = valid[i] ? p.rho[k] : 1.0;
            E[i] = valid[i] ? p.e[k] : 0.0;
            id[i] = valid[i] ? p.id[k] : 0;
            dk[i] = valid[i] ? dest[k] : 0ull;
        }
        // stage vbar, acc of corners l, l + LG, and dsum_b = sum_a (v2_a(high corner) - v2_a(low corner)) / h
        double v2[2][DIM];
        int node[2];
#pragma unroll
        for (int qq = 0; qq < 2; ++qq) {
            node[qq] = corner_node_i<DIM>(gd, c, l + qq * LG);
#pragma unroll
            for (int a = 0; a < DIM; ++a) v2[qq][a] = (grp.cnt > 0) ? __ldg(nb + (long long)node[qq] * DIM + a) : 0.0;
        }
        double dsum[2] = { 0.0, 0.0 };
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                double other;
                if ((1 << a) < LG) other = shfl_xor_d(v2[qq][a], 1 << a);
                else other = v2[qq ^ 1][a];
                const int b = l + qq * LG;
                dsum[qq] += ((b >> a) & 1) ? (v2[qq][a] - other) : (other - v2[qq][a]);
            }
        }
        if (grp.cnt > 0) {
#pragma unroll
            for (int qq = 0; qq < 2; ++qq) {
                double *s_corner = s_group + (l + qq * LG) * Geo<DIM>::CH;
                stage_na<DIM>(na, node[qq], s_corner);
                *reinterpret_cast<double2 *>(s_corner + 2 * DIM) = make_double2(dsum[qq] * gd.inv_h, 0.0);
            }
        }
        __syncwarp();
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            if (valid[i]) {
                double xi[DIM], Vb[DIM], A[DIM], D;
                if (local_coords<DIM>(gd, X[i], c, xi)) {
                    double w[NB], out[2 * NPAIR];
                    natural_weights<DIM>(xi, w);
                    gather_pairs<DIM, NPAIR>(s_group, w, out);
#pragma unroll
                    for (int a = 0; a < DIM; ++a) { Vb[a] = out[a]; A[a] = out[DIM + a]; }
                    D = out[2 * DIM];
                } else {
                    slow_gather<DIM>(gd, na, nb, X[i], Vb, A, &D);
                }
                double Vn[DIM];
#pragma unroll
                for (int a = 0; a < DIM; ++a) Vn[a] = fma(dt, A[a], V[i][a]);   // V'
                // particle thermodynamics (eq. 4 with this step's D: reading A2).  P/rho = (gamma-1) E
                // and gamma P/rho = gamma (gamma-1) E are used in place of the quotients (one rounding apart).
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
        __syncwarp();      // the staging area is rewritten by the next iteration
    }
    // block maxima -> one atomicMax per block (max is order-free, so this is exact)
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

// S = (P+Q) M / rho for a freshly loaded / permuted particle set (eq. 13)
__global__ void __launch_bounds__(kBlock) k_force_payload(double gamma, const double *m, const double *rho, const double *e,
                                                          const double *q, double *S, long long n)
{
    const long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k < n) S[k] = ((gamma - 1.0) * rho[k] * e[k] + q[k]) * m[k] / rho[k];
}

// groups per cell = ceil(count / capacity), from the cell offsets
__global__ void __launch_bounds__(kBlock) k_group_counts(const int *off, int *gcount, int ncell, int cap)
{
    const int c = blockIdx.x * kBlock + threadIdx.x;
    if (c < ncell) gcount[c] = (off[c + 1] - off[c] + cap - 1) / cap;
    else if (c == ncell) gcount[c] = 0;
}

// fill the group records from the scanned group offsets; goff[ncell] = total number of groups
template <int DIM>
__global__ void __launch_bounds__(kBlock) k_group_fill(GridDesc gd, const int *off, const int *goff, int4 *groups,
                                                       int *n_groups, int ncell)
{
    constexpr int CAP = 1 << DIM;
    const int c = blockIdx.x * kBlock + threadIdx.x;
    if (c == 0) *n_groups = goff[ncell];
    if (c >= ncell) return;
    const int g0 = goff[c], g1 = goff[c + 1];
    if (g0 == g1) return;
    int cpack;
    if (DIM == 3) {
        const int cx = c % gd.nc[0], cy = (c / gd.nc[0]) % gd.nc[1], cz = c / (gd.nc[0] * gd.nc[1]);
        cpack = cx | (cy << 10) | (cz << 20);
    } else {
        cpack = (c % gd.nc[0]) | ((c / gd.nc[0]) << 16);
    }
    int first = off[c];
    const int end = off[c + 1];
    for (int gq = g0; gq < g1; ++gq, first += CAP) groups[gq] = make_int4(first, min(CAP, end - first), c, cpack);
}

inline unsigned blocks_for(long long n, int per) { return (unsigned)((n + per - 1) / per); }

// persistent launch: enough blocks to fill the 148 SMs a few times over, never more than the work needs
inline unsigned persistent_blocks(long long max_groups, int gpb, int per_sm)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const long long want = (long long)sms * per_sm;
    const long long need = (max_groups + gpb - 1) / gpb;
    return (unsigned)(need < want ? (need > 0 ? need : 1) : want);
}

}  // namespace

void launch_force_payload(const GridDesc &gd, const PArr &p, double *S, long long n, cudaStream_t s)
{
    if (n > 0) k_force_payload<<<blocks_for(n, kBlock), kBlock, 0, s>>>(gd.gamma, p.m, p.rho, p.e, p.q, S, n);
}

void launch_build_groups(const GridDesc &gd, const int *off, int *gcount_goff, int *scan_aux, int4 *groups, int *n_groups,
                         cudaStream_t s)
{
    const int cap = 1 << gd.dim;
    const int ncell = (int)gd.Nc;
    k_group_counts<<<blocks_for(ncell + 1, kBlock), kBlock, 0, s>>>(off, gcount_goff, ncell, cap);
    launch_exclusive_scan(gcount_goff, ncell + 1, scan_aux, s);
    if (gd.dim == 2) k_group_fill<2><<<blocks_for(ncell, kBlock), kBlock, 0, s>>>(gd, off, gcount_goff, groups, n_groups, ncell);
    else k_group_fill<3><<<blocks_for(ncell, kBlock), kBlock, 0, s>>>(gd, off, gcount_goff, groups, n_groups, ncell);
}

void launch_p2g1_sorted(const GridDesc &gd, const PArr &p, const double *S, const GArr &g, const SortedMap &map,
                        long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_p2g1_sorted<2><<<persistent_blocks(max_groups, Geo<2>::GPB, 8), kBlock, 0, s>>>(gd, p, S, g, map.groups, map.n_groups);
    else
        k_p2g1_sorted<3><<<persistent_blocks(max_groups, Geo<3>::GPB, 8), kBlock, 0, s>>>(gd, p, S, g, map.groups, map.n_groups);
}

void launch_g2p_p2g2_sorted(const GridDesc &gd, const PArr &p, const GArr &g, const double *na, const DevScalars *sc,
                            const SortedMap &map, int *count, unsigned long long *dest, long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_g2p_p2g2_sorted<2><<<persistent_blocks(max_groups, Geo<2>::GPB, 8), kBlock, 0, s>>>(gd, p, g, na, sc, map.groups, map.n_groups, count, dest);
    else
        k_g2p_p2g2_sorted<3><<<persistent_blocks(max_groups, Geo<3>::GPB, 8), kBlock, 0, s>>>(gd, p, g, na, sc, map.groups, map.n_groups, count, dest);
}

void launch_update_sorted(const GridDesc &gd, const PArr &p, const PArr &q, const double *na, const double *nb, DevScalars *sc,
                          const SortedMap &map, const int *off_new, const unsigned long long *dest, double *S_out,
                          long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    if (gd.dim == 2)
        k_update_sorted<2><<<persistent_blocks(max_groups, Geo<2>::GPB, 8), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map.groups, map.n_groups, off_new, dest, S_out);
    else
        k_update_sorted<3><<<persistent_blocks(max_groups, Geo<3>::GPB, 8), kBlock, 0, s>>>(gd, p, q, na, nb, sc, map.groups, map.n_groups, off_new, dest, S_out);
}

}  // namespace mpm
