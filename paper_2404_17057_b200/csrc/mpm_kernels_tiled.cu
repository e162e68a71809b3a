// mpm_kernels_tiled.cu -- TILED kernel family: lane groups (one cell per group of 2^d / 2 lanes, two particles per lane,
// butterfly reductions, fused re-ordering: mpm_lane_groups.cuh) with
//
//   * tile-major cell keys (TileGeo: 8 x 8 x 4 cells in 3D, 16 x 16 in 2D): the particles of one tile are one contiguous
//     run of the cell-sorted order (the grid-to-particle connectivity of PAPER.md:745-748, per tile).  One thread block
//     works on one tile (or a chunk of a dense tile): the tile's (T+1)^d node velocities are staged ONCE in shared memory
//     and every particle of the tile gathers from there (no per-group staging, each corner read once per lane);
//   * even-aligned cell slots: every cell's slot range starts at an EVEN slot (an odd cell leaves one unused slot), so
//     that lane l of a group owns the two consecutive particles first + 2l, first + 2l + 1 and fetches each field with
//     ONE aligned 128-bit load (half the load instructions of the SORTED family);
//   * TWO particle sweeps per step instead of three: P2G#1 of step n+1 (Alg. 1 l.3) has no dt in it and
//     only needs the state the update of step n has just produced, so it is fused into the update kernel (l.10-12):
//     a particle that stays in its cell (the common case, CFL <= 0.5: PAPER.md:526) joins the group's butterfly with
//     weights taken at its NEW position, a particle that changes cell adds its 2^d x (1 + 2d) contributions directly.
//     The force payload S = (P+Q) M / rho never goes to memory.  Node accumulators m, mv, f are double-buffered.
//
// Shared-memory accumulator tiles with fp64 atomicAdd were measured and dropped (git history: CAS loops stall the
// 16 resident warps; a global RED is asynchronous): scatters use global fp64 reductions.
#include "mpm_lane_groups.cuh"
#include "mpm_node_bc.cuh"

#ifndef MPM_MINB
#define MPM_MINB 2   // resident blocks per SM the particle kernels are compiled for (register budget)
#endif

namespace mpm {

namespace {

using namespace lg;

#if defined(MPM_CHECKED) && MPM_CHECKED
// bounds of the checked build, set by the launchers before every launch (one handle at a time per process in that build)
__device__ long long g_checked_nodes = 0, g_checked_slots = 0;
#endif

__device__ __forceinline__ double2 ld2(const double *__restrict__ p, long long k, bool ok)
{
    MPM_CHECK(!ok || (k >= 0 && k + 1 < g_checked_slots && (k & 1) == 0));
    return ok ? __ldg(reinterpret_cast<const double2 *>(p + k)) : make_double2(0.0, 0.0);
}
__device__ __forceinline__ void st2(double *p, long long k, double a, double b)
{
    MPM_CHECK(k >= 0 && k + 1 < g_checked_slots && (k & 1) == 0);
    *reinterpret_cast<double2 *>(p + k) = make_double2(a, b);
}

// ------------------------------------------------------------------------------------------------ particle streams
// The particle fields of the NEXT pass are copied into shared memory while the current pass computes.  Two mechanisms,
// selected by the kernels' BULK template parameter (mpm_config.particle_stream):
//   BULK = false (default): per-thread cp.async (SASS LDGSTS), 16 bytes per lane and field = the lane's two particles,
//     tracked by commit groups;
//   BULK = true: the particles of a tile are ONE contiguous run of slots (tile-major cell order), and so are the particles
//     the 32 / LG groups of a warp work on in one pass: <= 64 slots.  Their fields come in with bulk asynchronous copies
//     (cp.async.bulk.shared::cluster.global, the non-tensor form of TMA: SASS UBLKCP), one per field and pass, issued by
//     lane 0 of the warp and tracked by an mbarrier (expect_tx / complete_tx); the lanes read their two particles from
//     the warp's window.  This takes the copies off the LSU / L1TEX path and replaces 32 address computations per field
//     by one.  Measured (profiles/r02_experiments.md sections 1 and 9): no faster than cp.async on config 4 and 2 % slower on config
//     5 (a one-lane issue sequence costs as many issue slots as a full-warp LDGSTS, and an mbarrier wait more than a
//     commit-group wait), hence not the default.
// Both use the same shared-memory layout, [warp][field][kWin slots]: cp.async lanes own slots 2 lane, 2 lane + 1.
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((unsigned)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
// all committed groups but the most recent one have landed
__device__ __forceinline__ void cp_async_wait_but_one() { asm volatile("cp.async.wait_group 1;" ::: "memory"); }
// all committed groups but the N most recent ones have landed
template <int N>
__device__ __forceinline__ void cp_async_wait_but() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of bulk copies to come (0 = none: the phase completes at once)
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MPM_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MPM_DONE_%=;\n"
        "bra MPM_WAIT_%=;\n"
        "MPM_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// bytes: a multiple of 16; smem and gmem 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *smem, const void *gmem, unsigned bytes, unsigned long long *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem)), "l"(gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// Window of slots [w0, w0 + wn) that holds the particles of the warp's groups in one pass, widened to multiples of 4 slots
// (16-byte alignment of the 4-byte id stream); wn = 0 for a warp without particles in this pass.  At most kWin slots.
constexpr int kWin = 2 * 32 + 4;
template <bool BULK>
__device__ __forceinline__ void warp_window(int first, int cnt, int &w0, int &wn)
{
    if (!BULK) { w0 = 0; wn = 0; return; }
    const int lo = __reduce_min_sync(0xffffffffu, cnt > 0 ? first : 0x7fffffff) & ~3;
    const int hi = (__reduce_max_sync(0xffffffffu, cnt > 0 ? first + ((cnt + 1) & ~1) : 0) + 3) & ~3;
    w0 = lo;
    wn = hi > lo ? hi - lo : 0;
}

// Node accumulators m, mv, f, mv2: fp64, component-major (default); or, with ACC32 (the fp32 grid-accumulation variant of
// BASELINE.json config 5: particle arithmetic stays fp64, the sums on the grid and the reductions that form them are fp32),
// fp32 and NODE-MAJOR: g.m points to float nm[N_n][8] = { m, mv_0, mv_1, mv_2, f_0, f_1, f_2, - } and g.mv2[0] to
// float v2[N_n][4] = { mv2_0, mv2_1, mv2_2, - } (unused components stay zero), so that a corner's channels go to the grid with
// TWO (one) vector reductions (red.global.add.v4.f32: SASS REDG.E.ADD.F32x4, sm_90+) instead of 1 + 2 d (d) scalar ones, and a
// tile node is staged with two (three) 16-byte loads.  fp64 has no vector reduction.
template <bool ACC32>
__device__ __forceinline__ void acc_add(double *arr, long long i, double v)
{
    static_assert(!ACC32, "the fp32 accumulators are node-major: acc32_add_nm / acc32_add_v2");
    MPM_CHECK(i >= 0 && i < g_checked_nodes);
    atomicAdd(arr + i, v);
}
template <bool ACC32>
__device__ __forceinline__ double acc_ld(const double *arr, long long i)
{
    static_assert(!ACC32, "the fp32 accumulators are node-major: acc32_ld");
    MPM_CHECK(i >= 0 && i < g_checked_nodes);
    return __ldg(arr + i);
}
__device__ __forceinline__ void red_add_f32x4(float *p, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
// m, mv, f of one node += (ACC32 layout)
template <int DIM>
__device__ __forceinline__ void acc32_add_nm(const GArr &g, long long node, double m, const double mv[DIM], const double f[DIM])
{
    MPM_CHECK(node >= 0 && node < g_checked_nodes);
    float *nm = reinterpret_cast<float *>(g.m) + 8 * node;
    red_add_f32x4(nm, (float)m, (float)mv[0], (float)mv[1], DIM == 3 ? (float)mv[DIM - 1] : 0.f);
    red_add_f32x4(nm + 4, (float)f[0], (float)f[1], DIM == 3 ? (float)f[DIM - 1] : 0.f, 0.f);
}
// mv2 of one node +=
template <int DIM>
__device__ __forceinline__ void acc32_add_v2(const GArr &g, long long node, const double v[DIM])
{
    MPM_CHECK(node >= 0 && node < g_checked_nodes);
    red_add_f32x4(reinterpret_cast<float *>(g.mv2[0]) + 4 * node, (float)v[0], (float)v[1], DIM == 3 ? (float)v[DIM - 1] : 0.f, 0.f);
}
// all sums of one node, widened
template <int DIM, bool WITH_V2>
__device__ __forceinline__ void acc32_ld(const GArr &g, long long node, double &m, double mv[DIM], double f[DIM], double mv2[DIM])
{
    MPM_CHECK(node >= 0 && node < g_checked_nodes);
    const float4 *nm = reinterpret_cast<const float4 *>(g.m) + 2 * node;
    const float4 a = __ldg(nm), b = __ldg(nm + 1);
    m = a.x;
    mv[0] = a.y; mv[1] = a.z; if (DIM == 3) mv[DIM - 1] = a.w;
    f[0] = b.x; f[1] = b.y; if (DIM == 3) f[DIM - 1] = b.z;
    if (WITH_V2) {
        const float4 c = __ldg(reinterpret_cast<const float4 *>(g.mv2[0]) + node);
        mv2[0] = c.x; mv2[1] = c.y; if (DIM == 3) mv2[DIM - 1] = c.z;
    }
}

// 1 / x to within about one unit in the last place for a finite x that is neither zero nor subnormal: the hardware
// approximation (relative error 2^-23) refined by two Newton steps, 5 instructions in place of the ~25 of an IEEE division
// (measured: profiles/r02_experiments.md section 8).  Used where the parity tolerance (1e-12) leaves room for the last bit:
// rho' = rho / (1 + dt D) and the node quotients by m.  x = 0 gives inf like the division; a subnormal x is flushed to 0.
#ifndef MPM_FAST_RCP
#define MPM_FAST_RCP 1
#endif
__device__ __forceinline__ double rcp_newton(double x)
{
#if MPM_FAST_RCP
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    y = fma(y, fma(-x, y, 1.0), y);
    y = fma(y, fma(-x, y, 1.0), y);
    return y;
#else
    return 1.0 / x;
#endif
}

template <int DIM, bool CM>
__device__ __forceinline__ int tiled_key_of_position(const GridDesc &gd, const double X[DIM])
{
    int c[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double xi;
        cell_1d(X[a], gd.inv_h, gd.nc[a], c[a], xi);
    }
    return tiled_key_of_cell<DIM>(gd, c, CM);
}

// A dense cell fills whole warps with its groups.  Then the groups' corner totals are added up across the warp first
// (xor shuffles over the group index) and the first group alone issues the reductions: 32 / LG times fewer fp64
// reductions on the same 2^d nodes.  Returns whether this lane's group still has to issue them.
template <int DIM, int NCH>
__device__ __forceinline__ bool fold_warp_one_cell(double tot[NCH][2], int lane, bool one_cell, bool any)
{
    if (!one_cell) return any;
#pragma unroll
    for (int m = Geo<DIM>::LG; m < 32; m <<= 1) {
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            tot[ch][0] += shfl_xor_d(tot[ch][0], m);
            tot[ch][1] += shfl_xor_d(tot[ch][1], m);
        }
    }
    return lane < Geo<DIM>::LG;      // lane 0's group is never idle unless the whole warp is (then every total is 0)
}

// warp-uniform: do all groups of this warp (idle ones aside) sit in the same cell?
__device__ __forceinline__ bool warp_one_cell(int cell, int cnt)
{
    const int first = __shfl_sync(kFull, cell, 0);
    return __all_sync(kFull, cnt == 0 || cell == first);
}

// Group totals of the P2G#1 channels (m, mv, f) from per-lane payloads and butterfly-order weights, reduced into the node
// accumulators g.m, g.mv, g.f with one global fp64 reduction per corner and channel:
//   pay[i] = { M, M V_a, S } of the lane's particle i, w[i][r] = weight of corner r ^ l (0 for a particle that is not
//   part of the group reduction).
// p2g1_group_totals leaves in out[ch][q], ch = 0 (m), 1 .. DIM (mv), DIM + 1 .. 2 DIM (f), the group's totals for the
// corners b_q = l + q LG and returns whether this lane's group has to add them to the grid at all.
template <int DIM>
__device__ __forceinline__ bool p2g1_group_totals(const GridDesc &gd, int l, bool any, const double pay[2][DIM + 2],
                                                  const double w[2][1 << DIM], bool one_cell, double out[2 * DIM + 1][2])
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG;
    double tot[DIM + 2][2];
#pragma unroll
    for (int ch = 0; ch < DIM + 2; ++ch) {
        double v[NB];
#pragma unroll
        for (int r = 0; r < NB; ++r) v[r] = fma(pay[1][ch], w[1][r], pay[0][ch] * w[0][r]);
        butterfly<DIM>(v);
        tot[ch][0] = v[0];
        tot[ch][1] = v[LG];
    }
    any = fold_warp_one_cell<DIM, DIM + 2>(tot, threadIdx.x & 31, one_cell, any);
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
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        out[0][q] = tot[0][q];
#pragma unroll
        for (int a = 0; a < DIM; ++a) { out[1 + a][q] = tot[1 + a][q]; out[1 + DIM + a][q] = F[a][q]; }
    }
    return any;
}

// ... added to the node accumulators with one global fp64 reduction per corner and channel
template <int DIM, bool ACC32>
__device__ __forceinline__ void p2g1_commit_global(const GridDesc &gd, const GArr &g, const int c[DIM], int l, const double tot[2 * DIM + 1][2])
{
    constexpr int LG = Geo<DIM>::LG;
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        const int node = corner_node_i<DIM>(gd, c, l + q * LG);
        if constexpr (ACC32) {
            double mv[DIM], f[DIM];
#pragma unroll
            for (int a = 0; a < DIM; ++a) { mv[a] = tot[1 + a][q]; f[a] = tot[1 + DIM + a][q]; }
            acc32_add_nm<DIM>(g, node, tot[0][q], mv, f);
        } else {
            acc_add<false>(g.m, node, tot[0][q]);
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                acc_add<false>(g.mv[a], node, tot[1 + a][q]);
                acc_add<false>(g.f[a], node, tot[1 + DIM + a][q]);
            }
        }
    }
}

template <int DIM, bool ACC32>
__device__ __forceinline__ void scatter_p2g1_group(const GridDesc &gd, const GArr &g, const int c[DIM], int l, bool any,
                                                   const double pay[2][DIM + 2], const double w[2][1 << DIM], bool one_cell = false)
{
    double tot[2 * DIM + 1][2];
    if (p2g1_group_totals<DIM>(gd, l, any, pay, w, one_cell, tot)) p2g1_commit_global<DIM, ACC32>(gd, g, c, l, tot);
}

// ------------------------------------------------------------------------------------------------ atomics-free tile accumulation
// The paper's proposal for a P2G without atomics: sort the particles by cell, colour the cells so that
// cells of one colour share no node, and process one colour at a time.  Here: the tile-local cell numbering is colour-major
// (TileGeo), so the groups a block works on in one pass belong to at most two consecutive colours in the common case.
// With COLOUR the group totals of a pass are added into a shared-memory accumulator tile with PLAIN read-modify-writes
// (no atomic of any kind): first the groups of the pass's first colour, after a block barrier those of its last colour.
// Groups of one colour in one pass are different cells, hence touch disjoint nodes.  Not eligible, and sent to the grid
// with global reductions as in the default path: groups of a cell that has more than one group (more than 2^d particles:
// the cell map flags them), groups of a third colour in a sparse pass, and particles that change cell.  The accumulator tile
// is flushed once per block with one global reduction per non-zero node value (neighbouring tiles and the ineligible
// groups add to the same nodes, so the flush cannot be a plain store).
template <int DIM>
__device__ __forceinline__ constexpr int corner_off(int b);

template <int DIM>
struct PassColours {
    int lo, hi;      // colours of the first and of the last group of the pass (block-uniform)
};

template <int DIM>
__device__ __forceinline__ PassColours<DIM> pass_colours(const int4 *__restrict__ groups, int g_first, int g_end, int gpb)
{
    using TG = TileGeo<DIM>;
    PassColours<DIM> pc{ 0, 0 };
    const int g_last = min(g_first + gpb, g_end) - 1;
    if (g_first <= g_last) {
        pc.lo = TG::colour_of(__ldg(&groups[g_first].z) & (TG::TC - 1));
        pc.hi = TG::colour_of(__ldg(&groups[g_last].z) & (TG::TC - 1));
    }
    return pc;
}

// phase in which this lane's group adds its totals to the shared accumulator tile: 0, 1, or -1 = not eligible
template <int DIM>
__device__ __forceinline__ int colour_phase(const PassColours<DIM> &pc, const Group &grp)
{
    if (grp.cnt == 0 || grp.multi) return -1;
    const int col = TileGeo<DIM>::colour_of(grp.cell & (TileGeo<DIM>::TC - 1));
    return col == pc.lo ? 0 : col == pc.hi ? 1 : -1;
}

// s_acc[node][NCH] += tot[ch][q] for the lane's two corners (plain additions: see above)
template <int DIM, int NCH>
__device__ __forceinline__ void tile_accumulate(double *s_acc, int j0, int l, const double tot[NCH][2])
{
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        double *dst = s_acc + (j0 + corner_off<DIM>(l + q * Geo<DIM>::LG)) * NCH;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) dst[ch] += tot[ch][q];
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.3 (after a load only)
// m, mv from phi-weighted channels (M, M V); f from the phi-weighted channel S = (P+Q) M / rho (eq. 13).
// Every later step gets its P2G#1 from the update kernel of the step before.
template <int DIM, bool ACC32>
__global__ void __launch_bounds__(kBlock, MPM_MINB) k_p2g1_tiled(GridDesc gd, PArr p, GArr g, SortedMap map)
{
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = Geo<DIM>::GPB;
    const int n_groups = *map.n_groups;
    const int l = threadIdx.x % LG;
    const double gm1 = gd.gamma - 1.0;
    const long long stride = (long long)gridDim.x * GPB;
    long long gidx = (long long)blockIdx.x * GPB + threadIdx.x / LG;
    for (long long g0 = (long long)blockIdx.x * GPB; g0 < n_groups; g0 += stride, gidx += stride) {
        const Group grp = fetch_group(map.groups, gidx, n_groups);
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
        const long long k0 = (long long)grp.first + 2 * l;
        double X[2][DIM], V[2][DIM], pay[2][DIM + 2], w[2][NB];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const double2 tx = ld2(p.x[a], k0, valid[0]), tv = ld2(p.v[a], k0, valid[0]);
            X[0][a] = tx.x; X[1][a] = valid[1] ? tx.y : 0.0;
            V[0][a] = tv.x; V[1][a] = valid[1] ? tv.y : 0.0;
        }
        const double2 tm = ld2(p.m, k0, valid[0]), tr = ld2(p.rho, k0, valid[0]), te = ld2(p.e, k0, valid[0]),
                      tq = ld2(p.q, k0, valid[0]);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double M = valid[i] ? (i ? tm.y : tm.x) : 0.0, rho = valid[i] ? (i ? tr.y : tr.x) : 1.0;
            const double E = i ? te.y : te.x, Q = i ? tq.y : tq.x;
            const double S = valid[i] ? (gm1 * rho * E + Q) * M / rho : 0.0;      // (P+Q) M / rho, P = (gamma-1) rho E (eq. 3)
            double xi[DIM];
            const bool fast = valid[i] && local_coords<DIM>(gd, X[i], c, xi);
            if (valid[i] && !fast) slow_p2g1<DIM, ACC32>(gd, g, X[i], V[i], M, S);
            pay[i][0] = fast ? M : 0.0;
            pay[i][DIM + 1] = fast ? S : 0.0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) pay[i][1 + a] = fast ? M * V[i][a] : 0.0;
            if (fast) swizzled_weights<DIM>(xi, l, w[i]);
            else {
#pragma unroll
                for (int r = 0; r < NB; ++r) w[i][r] = 0.0;
            }
        }
        scatter_p2g1_group<DIM, ACC32>(gd, g, c, l, grp.cnt > 0, pay, w);
    }
}

// ------------------------------------------------------------------------------------------------ tile work items
// A block works on one ITEM = up to Chunk<DIM>::GROUPS consecutive groups of ONE tile (a tile with more groups is cut into
// several items, so that a dense tile does not serialise on one block).  The item list is rebuilt every step from the
// per-key particle counts (k_cell_map_tiled).
#ifndef MPM_TB
#define MPM_TB 128
#endif
#ifndef MPM_TBMIN_G
#define MPM_TBMIN_G 4
#endif
#ifndef MPM_TBMIN_U
#define MPM_TBMIN_U 4
#endif
constexpr int kTB = MPM_TB;              // threads per block of the tile kernels
constexpr int kTBMinG = MPM_TBMIN_G;     // resident blocks per SM the gather kernel is compiled for (128 registers)
constexpr int kTBMinU = MPM_TBMIN_U;     // ... and the update kernel (128 registers, no spills)
#ifndef MPM_TBMIN_G2
#define MPM_TBMIN_G2 6
#endif
#ifndef MPM_TBMIN_U2
#define MPM_TBMIN_U2 4
#endif
// 2D: half the state per particle.  Measured on config 3 (profiles/r02_experiments.md): the gather kernel gains 14 % at 6 blocks
// per SM (80 registers, no spill); the update kernel spills below 128 registers and loses, so it stays at 4
constexpr int kTBMinG2 = MPM_TBMIN_G2, kTBMinU2 = MPM_TBMIN_U2;

template <int DIM>
struct Chunk {
    static constexpr int PASSES = 16;
    static constexpr int GROUPS = PASSES * (kTB / Geo<DIM>::LG);
};

// The group records of a block's item are copied into shared memory once, at the start of the block (one 16-byte cp.async
// per record: they are one contiguous run), and every pass reads its records from there.  ncu (profiles/r02_ncu_final.md section 3):
// fetching them with a global load inside the pass cost 6 - 9 % of both sweeps' stall samples -- the unpacking right behind
// the load, and shared-memory loads that waited on the scoreboard they shared with it.  STAGE = false (the COLOUR
// instantiations, whose static shared memory is full): records come from global memory as before.
template <int DIM, bool STAGE>
__device__ __forceinline__ void stage_groups(int4 *s_grp, const int4 *__restrict__ groups, int first, int n)
{
    if (STAGE) {
        for (int j = threadIdx.x; j < n; j += kTB) cp_async16(s_grp + j, groups + first + j);
        cp_async_commit();
    }
}
// record j of the item (j >= n: an idle group)
template <bool STAGE>
__device__ __forceinline__ Group item_group(const int4 *s_grp, const int4 *__restrict__ groups, int first, int j, int n)
{
    if (!STAGE) return fetch_group(groups, (long long)first + j, first + n);
    Group g{ 0, 0, 0, 0, 0 };
    if (j < n) {
        MPM_CHECK(j >= 0);
        const int4 r = s_grp[j];
        g.first = r.x; g.cnt = r.y & 0xff; g.multi = r.y >> 8; g.cell = r.z; g.cpack = r.w;
    }
    return g;
}
// ... or, without the staging: the raw record is loaded from global memory in the middle of a pass and only unpacked at the
// end of that pass, when it has had time to arrive (an all-zero record is an idle group)
__device__ __forceinline__ int4 raw_group(const int4 *__restrict__ groups, long long gidx, int n_groups)
{
    return gidx < (long long)n_groups ? __ldg(groups + gidx) : make_int4(0, 0, 0, 0);
}
__device__ __forceinline__ Group unpack_group(const int4 &r)
{
    Group g;
    g.first = r.x; g.cnt = r.y & 0xff; g.multi = r.y >> 8; g.cell = r.z; g.cpack = r.w;
    return g;
}

// tile-local node index j = lx + N0 (ly + N1 lz) of corner b of the cell with tile-local node index j0
template <int DIM>
__device__ __forceinline__ constexpr int corner_off(int b)
{
    using TG = TileGeo<DIM>;
    return (b & 1) + TG::N0 * ((b >> 1) & 1) + ((DIM == 3) ? TG::N0 * TG::N1 * ((b >> 2) & 1) : 0);
}

template <int DIM>
__device__ __forceinline__ void tile_origin(const GridDesc &gd, int tile, int org[DIM])
{
    using TG = TileGeo<DIM>;
    int t[3];
    tile_coords<DIM>(gd, tile, t);
    org[0] = t[0] << TG::LT0;
    org[1] = t[1] << TG::LT1;
    if (DIM == 3) org[DIM - 1] = t[2] << TG::LT2;
}

// global node index and node coordinates of tile-local node j (periodic wrap: node n == node 0, A11); -1 = outside the grid
template <int DIM>
__device__ __forceinline__ int tile_node_global(const GridDesc &gd, const int org[DIM], int j, int idx[DIM])
{
    using TG = TileGeo<DIM>;
    int ln[3];
    ln[0] = j % TG::N0;
    ln[1] = (j / TG::N0) % TG::N1;
    ln[2] = j / (TG::N0 * TG::N1);
    int node = 0, stride = 1;
    bool ok = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        int i = org[a] + ln[a];
        if (i > gd.nc[a]) ok = false;
        if (gd.per[a] && i == gd.nc[a]) i = 0;
        idx[a] = i;
        node += stride * i;
        stride *= gd.nn[a];
    }
    return ok ? node : -1;
}

// Stage the node velocities of one tile in shared memory, node-major with CH doubles per node, straight from the raw
// node accumulators m, mv, f (and mv2): Alg. 1 l.4 (BC + obstacle on mv, f: eqs. 21, 22, 30), l.5
// (mv' = mv + dt f) and the quotients the gathers read (theta of PAPER.md:295, ratio := 0 where m = 0,
// reading A5) are evaluated HERE, per tile node, instead of in a node kernel that writes them to memory first:
//   WITH_V2 = false (gather kernel): [0, DIM) vbar = mv'/m, [DIM, 2 DIM) acc = f/m;
//   WITH_V2 = true  (update kernel): [0, DIM) vbar = mv'/m, [DIM, 2 DIM) v2 = BC(mv2)/m (l.9); rest 0.
// One reciprocal per node (1 ulp from the true quotients of the node kernels, far inside the parity tolerance).
template <int DIM, int CH, bool WITH_V2, bool ACC32>
__device__ __forceinline__ void stage_tile(const GridDesc &gd, const int org[DIM], const GArr &g, double dt, double *s_tile)
{
    using TG = TileGeo<DIM>;
    constexpr int BATCH = WITH_V2 ? 2 : 4;              // measured: the update kernel has no registers to spare for 4
    constexpr int NALL = (TG::NN + kTB - 1) / kTB;      // nodes per thread
    constexpr int NIT = NALL < BATCH ? NALL : BATCH;    // ... loaded together
    for (int j0 = 0; j0 < TG::NN; j0 += NIT * kTB) {
    // the loads of NIT nodes are issued before the first one is used (fewer exposed memory latencies per tile)
    int node[NIT], idx[NIT][DIM];
    double m[NIT], mv[NIT][DIM], f[NIT][DIM], mv2[NIT][DIM];
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int j = j0 + threadIdx.x + it * kTB;
        node[it] = (j < TG::NN) ? tile_node_global<DIM>(gd, org, j, idx[it]) : -1;
        m[it] = 0.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) { mv[it][a] = 0.0; f[it][a] = 0.0; mv2[it][a] = 0.0; }
        if (node[it] >= 0) {
            if constexpr (ACC32) acc32_ld<DIM, WITH_V2>(g, node[it], m[it], mv[it], f[it], mv2[it]);
            else {
                m[it] = acc_ld<false>(g.m, node[it]);
#pragma unroll
                for (int a = 0; a < DIM; ++a) { mv[it][a] = acc_ld<false>(g.mv[a], node[it]); f[it][a] = acc_ld<false>(g.f[a], node[it]); }
                if (WITH_V2) {
#pragma unroll
                    for (int a = 0; a < DIM; ++a) mv2[it][a] = acc_ld<false>(g.mv2[a], node[it]);
                }
            }
        }
    }
#pragma unroll
    for (int it = 0; it < NIT; ++it) {
        const int j = j0 + threadIdx.x + it * kTB;
        if (j >= TG::NN) break;
        double v[CH];
#pragma unroll
        for (int q = 0; q < CH; ++q) v[q] = 0.0;
        if (node[it] >= 0) {
            apply_bc<DIM, true>(gd, g, node[it], idx[it], m[it], mv[it], f[it]);
            const double inv = (m[it] != 0.0) ? (fabs(m[it]) >= 1e-290 ? rcp_newton(m[it]) : 1.0 / m[it]) : 0.0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) v[a] = __dmul_rn(fma(dt, f[it][a], mv[it][a]), inv);      // every rounding explicit: both tile kernels stage the same vbar
            if (WITH_V2) {
                double none[DIM];
#pragma unroll
                for (int a = 0; a < DIM; ++a) none[a] = 0.0;
                apply_bc<DIM, false>(gd, g, node[it], idx[it], m[it], mv2[it], none);
#pragma unroll
                for (int a = 0; a < DIM; ++a) v[DIM + a] = mv2[it][a] * inv;
            } else {
#pragma unroll
                for (int a = 0; a < DIM; ++a) v[DIM + a] = f[it][a] * inv;
            }
        }
        double2 *dst = reinterpret_cast<double2 *>(s_tile + j * CH);
#pragma unroll
        for (int q = 0; q < CH / 2; ++q) dst[q] = make_double2(v[2 * q], v[2 * q + 1]);
    }
    }
}

// 1D weights of a particle w.r.t. the GROUP's cell c (the particle is in that cell: exact sort, see move_particle):
// W[a][0] = 1 - xi_a, W[a][1] = xi_a with xi = X / h - c (A19)
template <int DIM>
__device__ __forceinline__ void weights_1d(const GridDesc &gd, const double X[DIM], const int c[DIM], double xi[DIM], double W[DIM][2])
{
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        xi[a] = __dmul_rn(X[a], gd.inv_h) - (double)c[a];
        W[a][0] = 1.0 - xi[a];
        W[a][1] = xi[a];
    }
}

// Is a local coordinate vector inside the closed unit cell [0, 1]^d (1 included: a particle on the upper domain face,
// A6)?  Exact, on the integer pipe: a double in [0, 1] has a bit pattern <= that of 1.0 (sign clear, order-preserving).
template <int DIM>
__device__ __forceinline__ bool in_unit_cell(const double xi[DIM])
{
    bool in = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) in = in && ((unsigned long long)__double_as_longlong(xi[a]) <= 0x3FF0000000000000ull);
    return in;
}

// Does a particle of the group's cell c stay in that cell when it moves to Xn (Alg. 1 l.11-12)?  It does iff its local
// coordinate xin = Xn / h - c lies in [0, 1) on every axis: then floor(Xn / h) = c (the subtraction is exact next to c) and
// c needs no clamp, i.e. the general binning (cell_1d, readings A6, A19) returns c.  Exact, on the integer pipe: 0 <= xin < 1
// <=> the bit pattern is below that of 1.0 (a negative value has the sign bit set).  Everything else -- another cell, or the
// clamped cases on a domain face -- is binned by tiled_key_of_position.  Both tile kernels take this decision with this
// function on the same Xn (move_inside / move_particle), so they agree on it; xin is also what the P2G of the stayers needs.
template <int DIM>
__device__ __forceinline__ bool stays_in_cell(const GridDesc &gd, const double Xn[DIM], const int c[DIM], double xin[DIM])
{
    bool in = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        xin[a] = __dmul_rn(Xn[a], gd.inv_h) - (double)c[a];
        in = in && ((unsigned long long)__double_as_longlong(xin[a]) < 0x3FF0000000000000ull);
    }
    return in;
}

// phi-weighted gather of the staged tile for the TWO particles of a lane (each corner is read once for both):
//   out[i][ch] = sum_b phi_b(X_i) n_b[ch]  (eq. 17), ch < 2 DIM (Vbar, A) without WITH_D, ch < DIM (Vbar) with it;
//   with WITH_D also Dh[i] = h * sum_b sum_a v2_a(b) d_a phi_b(X_i), v2 = channels [DIM, 2 DIM)  (eq. 19, trace; the
//   factor 1/h is applied by the caller)
template <int DIM, int CH, bool WITH_D>
__device__ __forceinline__ void gather_tile(const double *s_cell, const double W[2][DIM][2], double out[2][2 * DIM], double Dh[2])
{
    constexpr int NPHI = WITH_D ? DIM : 2 * DIM;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        Dh[i] = 0.0;
#pragma unroll
        for (int ch = 0; ch < 2 * DIM; ++ch) out[i][ch] = 0.0;
    }
#pragma unroll
    for (int b = 0; b < (1 << DIM); ++b) {
        const double2 *row = reinterpret_cast<const double2 *>(s_cell + corner_off<DIM>(b) * CH);
        double val[CH];
#pragma unroll
        for (int q = 0; q < CH / 2; ++q) {
            const double2 t = row[q];
            val[2 * q] = t.x;
            val[2 * q + 1] = t.y;
        }
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            double phi = W[i][0][b & 1];
#pragma unroll
            for (int a = 1; a < DIM; ++a) phi *= W[i][a][(b >> a) & 1];
#pragma unroll
            for (int ch = 0; ch < NPHI; ++ch) out[i][ch] = fma(phi, val[ch], out[i][ch]);
            if (WITH_D) {
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    double q = 1.0;
#pragma unroll
                    for (int a2 = 0; a2 < DIM; ++a2)
                        if (a2 != a) q *= W[i][a2][(b >> a2) & 1];
                    const double sv = ((b >> a) & 1) ? val[DIM + a] : -val[DIM + a];
                    Dh[i] = fma(sv, q, Dh[i]);
                }
            }
        }
    }
}

// Fast path of Alg. 1 l.11: X' = X + dt Vbar.  When X' lies in [0, L) on every axis, neither the
// periodic wrap (A11), nor the outflow test (A8), nor the clamp of lg::move_particle changes it, so that function
// returns exactly this X'; the caller takes move_particle only when this returns false (rare: particles next to a
// domain face).  Both tile kernels use the same two functions on the same inputs, so they agree on X' bit for bit.
template <int DIM>
__device__ __forceinline__ bool move_inside(const GridDesc &gd, const double X[DIM], const double Vb[DIM], double dt, double Xn[DIM])
{
    bool in = true;
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        Xn[a] = fma(dt, Vb[a], X[a]);
        in = in && (Xn[a] >= 0.0) && (Xn[a] < gd.L[a]);
    }
    return in;
}

// P2G#1 (eqs. 13, 14, 16, 18) of the particles flagged in `mask` (one bit per lane), done by the WHOLE warp, 32 / 2^d
// particles per round: lane (slot = lane / 2^d, corner b = lane % 2^d) gets the data of the slot's particle by shuffle
// and adds its 1 + 2 d channels (m, mv_a, f_a) to corner b.  Used for particles that leave their group's cell (their
// contributions cannot join the group's butterfly).
template <int DIM, bool ACC32>
__device__ __forceinline__ void coop_p2g1(const GridDesc &gd, const GArr &gn, unsigned mask, const double Xn[DIM],
                                          const double Vn[DIM], double Mn, double Sn, int lane)
{
    constexpr int NB = 1 << DIM, SLOTS = 32 / NB;
    const int b = lane & (NB - 1), slot = lane / NB;
    while (mask) {
        int src = -1;
#pragma unroll
        for (int s = 0; s < SLOTS; ++s) {      // the slot's particle = the s-th flagged lane (mask is warp-uniform)
            const int f = mask ? __ffs(mask) - 1 : -1;
            if (s == slot) src = f;
            mask &= mask - 1u;
        }
        const int from = src < 0 ? 0 : src;
        double X[DIM], V[DIM];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            X[a] = __shfl_sync(kFull, Xn[a], from);
            V[a] = __shfl_sync(kFull, Vn[a], from);
        }
        const double M = __shfl_sync(kFull, Mn, from), S = __shfl_sync(kFull, Sn, from);
        if (src >= 0) {
            int c[DIM];
            double xi[DIM];
            particle_cell<DIM>(gd, X, c, xi);
            const long long node = corner_node<DIM>(gd, c, b);
            const double Mphi = M * corner_phi<DIM>(xi, b);
            if constexpr (ACC32) {
                double mv[DIM], f[DIM];
#pragma unroll
                for (int a = 0; a < DIM; ++a) { mv[a] = V[a] * Mphi; f[a] = S * corner_dphi<DIM>(xi, b, a, gd.inv_h); }
                acc32_add_nm<DIM>(gn, node, Mphi, mv, f);
            } else {
                acc_add<false>(gn.m, node, Mphi);
#pragma unroll
                for (int a = 0; a < DIM; ++a) {
                    acc_add<false>(gn.mv[a], node, V[a] * Mphi);
                    acc_add<false>(gn.f[a], node, S * corner_dphi<DIM>(xi, b, a, gd.inv_h));
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.6-8 (+ l.11-12 bookkeeping)
// One block (kTB threads) per item.  The tile's node velocities vbar = mv'/m, acc = f/m are staged once in shared memory;
// every lane gathers A = G2P(f/m), Vbar = G2P(mv'/m) for its two particles from there (eq. 17),
// V' = V + dt A, mv2 += M V' phi through the group butterfly.  Also: the particle's
// cell after the move of l.11 and its rank inside that cell, for the fused re-ordering (l.12): the particles of a group
// that stay in their cell take consecutive ranks from ONE atomic per group (ballot + popc), only the others pay one
// atomic each; the atomics are issued before the scatter and their results consumed after it.
// The particle fields of the NEXT pass are copied into shared memory while the current pass computes (see "particle
// streams" above).  V' overwrites V in place.
template <int DIM, bool ACC32, bool BULK, bool COLOUR, bool CM>
__global__ void __launch_bounds__(kTB, (DIM == 2 && !COLOUR) ? kTBMinG2 : kTBMinG) k_g2p_p2g2_tiled(GridDesc gd, PArr p, GArr g,
                                                                const DevScalars *__restrict__ sc, SortedMap map,
                                                                const int4 *__restrict__ items, const int *__restrict__ n_items,
                                                                int *__restrict__ count, unsigned *__restrict__ dest,
                                                                unsigned long long *__restrict__ n_cell_changes)
{
    static_assert(CM || !COLOUR, "accumulation by colour needs the colour-major cell numbering");
    using TG = TileGeo<DIM>;
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = kTB / LG, CH = 2 * DIM, NF = 2 * DIM + 1;
    __shared__ __align__(16) double s_tile[TG::NN * CH];
    __shared__ __align__(16) double s_pf[kTB / 32][NF][kWin];      // per warp: x[d], v[d], m of the pass's slot window
    __shared__ __align__(8) unsigned long long s_bar[kTB / 32][2];  // per warp: X copies / V, M copies
    __shared__ __align__(16) double s_acc[COLOUR ? TG::NN * DIM : 1];   // COLOUR: accumulator tile of mv2
    constexpr bool SG = !COLOUR;                                        // group records staged in shared memory
    __shared__ __align__(16) int4 s_grp[SG ? Chunk<DIM>::GROUPS : 1];
    __shared__ int s_moved;
    if (threadIdx.x == 0) s_moved = 0;
    if (COLOUR) for (int j = threadIdx.x; j < TG::NN * DIM; j += kTB) s_acc[j] = 0.0;
    int n_moved = 0;
    if ((int)blockIdx.x >= *n_items) return;
    const int4 item = __ldg(items + blockIdx.x);      // {tile, first group, groups, -}
    if (item.z == 0) return;                          // a tile without particles
    const int l = threadIdx.x % LG, lane = threadIdx.x & 31, sh = lane & ~(LG - 1);
    const int g_end = item.y + item.z;
    int gl = threadIdx.x / LG;
    MPM_CHECK(item.z <= Chunk<DIM>::GROUPS);
    stage_groups<DIM, SG>(s_grp, map.groups, item.y, item.z);      // the oldest copy group: complete before any later one
    Group grp = fetch_group(map.groups, (long long)item.y + gl, g_end);
    Group nxt = fetch_group(map.groups, (long long)item.y + gl + GPB, g_end);
    // two copy groups per pass: X (needed first, refilled as soon as it has been read: a whole pass of lead time) and V, M;
    // w0 = first slot of the warp's window of the pass being issued (returned for the reads)
    const int warp = threadIdx.x >> 5;
    if (BULK) {
        if (lane == 0) { mbar_init(&s_bar[warp][0], 1); mbar_init(&s_bar[warp][1], 1); mbar_fence_init(); }
        __syncwarp();
    }
    auto issue_x = [&](const Group &gr, int w0, int wn) {
        if (!BULK) {
            if (2 * l < gr.cnt) {
                const long long k0 = (long long)gr.first + 2 * l;
#pragma unroll
                for (int a = 0; a < DIM; ++a) cp_async16(&s_pf[warp][a][2 * lane], p.x[a] + k0);
            }
            cp_async_commit();
        } else if (lane == 0) {
            mbar_arrive_expect_tx(&s_bar[warp][0], (unsigned)(DIM * wn * 8));
            if (wn > 0) {
#pragma unroll
                for (int a = 0; a < DIM; ++a) bulk_g2s(&s_pf[warp][a][0], p.x[a] + w0, (unsigned)(wn * 8), &s_bar[warp][0]);
            }
        }
    };
    auto issue_vm = [&](const Group &gr, int w0, int wn) {
        if (!BULK) {
            if (2 * l < gr.cnt) {
                const long long k0 = (long long)gr.first + 2 * l;
#pragma unroll
                for (int a = 0; a < DIM; ++a) cp_async16(&s_pf[warp][DIM + a][2 * lane], p.v[a] + k0);
                if (!gd.uniform_mass) cp_async16(&s_pf[warp][2 * DIM][2 * lane], p.m + k0);
            }
            cp_async_commit();
        } else if (lane == 0) {
            const int nf = gd.uniform_mass ? DIM : DIM + 1;
            mbar_arrive_expect_tx(&s_bar[warp][1], (unsigned)(nf * wn * 8));
            if (wn > 0) {
#pragma unroll
                for (int a = 0; a < DIM; ++a) bulk_g2s(&s_pf[warp][DIM + a][0], p.v[a] + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
                if (!gd.uniform_mass) bulk_g2s(&s_pf[warp][2 * DIM][0], p.m + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
            }
        }
    };
    int w0, wn, w0n, wnn;
    warp_window<BULK>(grp.first, grp.cnt, w0, wn);
    warp_window<BULK>(nxt.first, nxt.cnt, w0n, wnn);
    issue_x(grp, w0, wn);
    issue_vm(grp, w0, wn);
    int org[DIM];
    tile_origin<DIM>(gd, item.x, org);
    const double dt = sc->dt;
    const long long step = sc->step;
    stage_tile<DIM, CH, false, ACC32>(gd, org, g, dt, s_tile);
    if (SG) { if (BULK) cp_async_wait_but<0>(); else cp_async_wait_but<2>(); }      // this thread's records have landed
    __syncthreads();
    unsigned parity = 0;
    PassColours<DIM> pc{ 0, 0 }, pcn{ 0, 0 };
    if (COLOUR) { pc = pass_colours<DIM>(map.groups, item.y, g_end, GPB); pcn = pass_colours<DIM>(map.groups, item.y + GPB, g_end, GPB); }
    for (int p0 = 0; p0 < item.z; p0 += GPB, gl += GPB, parity ^= 1u) {
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        const int local = grp.cell & (TG::TC - 1);      // grp.cell = tile-major key
        const int j0 = TG::node0_of(local, CM);
        const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
        const long long k0 = (long long)grp.first + 2 * l;
        double X[2][DIM], V[2][DIM], M[2];
        const int o = !BULK ? 2 * lane : valid[0] ? (int)(k0 - w0) : 0;      // the lane's two particles inside the warp's window
        MPM_CHECK(o >= 0 && o + 2 <= kWin && (o & 1) == 0 && j0 >= 0 && j0 + corner_off<DIM>(NB - 1) < TG::NN);
        MPM_CHECK(!valid[0] || (k0 >= 0 && k0 + 1 < gd.slots && grp.cell >= 0 && grp.cell < gd.Nkeys && (grp.cell >> TG::LTC) == item.x));
        if (BULK) mbar_wait(&s_bar[warp][0], parity); // this pass's X has landed (its V, M may still be in flight)
        else cp_async_wait_but_one();
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const double2 tx = *reinterpret_cast<const double2 *>(&s_pf[warp][a][o]);
            X[0][a] = valid[0] ? tx.x : 0.0; X[1][a] = valid[1] ? tx.y : 0.0;
        }
        if (BULK) __syncwarp();
        issue_x(nxt, w0n, wnn);                       // the window has been read: refill it for the next pass
        double W[2][DIM][2], xi[2][DIM], out[2][2 * DIM], Dh[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) weights_1d<DIM>(gd, X[i], c, xi[i], W[i]);
        gather_tile<DIM, CH, false>(s_tile + j0 * CH, W, out, Dh);
        if (BULK) mbar_wait(&s_bar[warp][1], parity); // this pass's V, M have landed (the next X may still be in flight)
        else cp_async_wait_but_one();
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const double2 tv = *reinterpret_cast<const double2 *>(&s_pf[warp][DIM + a][o]);
            V[0][a] = valid[0] ? tv.x : 0.0; V[1][a] = valid[1] ? tv.y : 0.0;
        }
        {
            const double2 tm = gd.uniform_mass ? make_double2(gd.um, gd.um) : *reinterpret_cast<const double2 *>(&s_pf[warp][2 * DIM][o]);
            M[0] = valid[0] ? tm.x : 0.0; M[1] = valid[1] ? tm.y : 0.0;
        }
        if (BULK) __syncwarp();
        issue_vm(nxt, w0n, wnn);
        double MV[2][DIM];
        int key[2];
        bool stay[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                V[i][a] = fma(dt, out[i][DIM + a], V[i][a]);      // V' = V + dt A
                MV[i][a] = M[i] * V[i][a];                        // M V'
            }
            // where the particle will be after l.11 (the persistent id is only needed by the recycling generator, A8)
            double Xn[DIM], xin[DIM];
            if (!move_inside<DIM>(gd, X[i], out[i], dt, Xn) && valid[i]) {
                bool recycled;
                int nclamp;
                move_particle<DIM>(gd, X[i], out[i], dt, gd.in_axis >= 0 ? (long long)p.id[k0 + i] : 0, step, Xn, recycled, nclamp);
            }
            // l.12: its cell there.  Still the group's cell (the common case at CFL < 1) or binned anew
            stay[i] = stays_in_cell<DIM>(gd, Xn, c, xin) && valid[i];
            key[i] = grp.cell;
            if (valid[i] && !stay[i]) key[i] = tiled_key_of_position<DIM, CM>(gd, Xn);
        }
        // V' replaces V in memory (the update kernel reads it back instead of gathering A again)
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            if (valid[1]) st2(p.v[a], k0, V[0][a], V[1][a]);
            else if (valid[0]) p.v[a][k0] = V[0][a];
        }
        // ranks among the particles that end up in the same cell (arrival order of the atomics, A17): issue the atomics
        MPM_CHECK((!valid[0] || (key[0] >= 0 && key[0] < gd.Nkeys)) && (!valid[1] || (key[1] >= 0 && key[1] < gd.Nkeys)));
        n_moved += (int)(valid[0] && !stay[0]) + (int)(valid[1] && !stay[1]);
        const unsigned gmask = (1u << LG) - 1u;
        const unsigned b0 = __ballot_sync(kFull, stay[0]), b1 = __ballot_sync(kFull, stay[1]);
        const unsigned g0 = (b0 >> sh) & gmask, g1 = (b1 >> sh) & gmask;
        const int nstay = __popc(g0) + __popc(g1);
        int base = 0, rank_m[2] = { 0, 0 };
        // a dense cell fills whole warps with its groups: then ONE atomic serves the warp (the groups' shares follow
        // from the ballots), instead of one per group on the same counter
        const bool one_cell = warp_one_cell(grp.cell, grp.cnt);
        if (one_cell) {
            if (lane == 0 && (b0 | b1)) base = atomicAdd(&count[grp.cell], __popc(b0) + __popc(b1));
        } else if (l == 0 && nstay > 0) base = atomicAdd(&count[grp.cell], nstay);
#pragma unroll
        for (int i = 0; i < 2; ++i)
            if (valid[i] && !stay[i]) rank_m[i] = atomicAdd(&count[key[i]], 1);
        // P2G#2: group totals of M V' phi per corner, one global reduction per corner and component
        {
            double ws[2][NB];
#pragma unroll
            for (int i = 0; i < 2; ++i) swizzled_weights<DIM>(xi[i], l, ws[i]);
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
            const bool issue = fold_warp_one_cell<DIM, DIM>(tot, lane, one_cell, grp.cnt > 0);
            int phase = -1;
            if (COLOUR) {      // eligible groups add into the shared accumulator tile, one colour at a time
                phase = colour_phase<DIM>(pc, grp);
                __syncthreads();                                   // the previous pass's additions are complete
                if (phase == 0 && issue) tile_accumulate<DIM, DIM>(s_acc, j0, l, tot);
                if (pc.hi != pc.lo) {
                    __syncthreads();
                    if (phase == 1 && issue) tile_accumulate<DIM, DIM>(s_acc, j0, l, tot);
                }
            }
            if (phase < 0 && issue) {
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    const int node = corner_node_i<DIM>(gd, c, l + q * LG);
                    if constexpr (ACC32) {
                        double v[DIM];
#pragma unroll
                        for (int a = 0; a < DIM; ++a) v[a] = tot[a][q];
                        acc32_add_v2<DIM>(g, node, v);
                    } else {
#pragma unroll
                        for (int a = 0; a < DIM; ++a) acc_add<false>(g.mv2[a], node, tot[a][q]);
                    }
                }
            }
        }
        // ... and only now use what they returned (consuming it one pass later instead was measured: neutral)
        if (one_cell) base = __shfl_sync(kFull, base, 0) + __popc(b0 & ((1u << sh) - 1u)) + __popc(b1 & ((1u << sh) - 1u));
        else base = __shfl_sync(kFull, base, sh);
        const unsigned lower = (1u << l) - 1u;
        const int pre = base + __popc(g0 & lower) + __popc(g1 & lower);
        const int rank0 = stay[0] ? pre : rank_m[0], rank1 = stay[1] ? pre + (int)((g0 >> l) & 1u) : rank_m[1];
        // the destination record is the rank alone: the update kernel finds the cell again from X' (stays_in_cell)
        // (bit 31: this kernel's stay / leave decision, which the update kernel checks against its own)
        const unsigned r0 = (unsigned)rank0 | (stay[0] ? 0x80000000u : 0u), r1 = (unsigned)rank1 | (stay[1] ? 0x80000000u : 0u);
        if (valid[1]) *reinterpret_cast<uint2 *>(dest + k0) = make_uint2(r0, r1);
        else if (valid[0]) dest[k0] = r0;
        grp = nxt;
        nxt = item_group<SG>(s_grp, map.groups, item.y, gl + 2 * GPB, item.z);
        w0 = w0n;
        wn = wnn;
        warp_window<BULK>(nxt.first, nxt.cnt, w0n, wnn);
        if (COLOUR) { pc = pcn; pcn = pass_colours<DIM>(map.groups, item.y + p0 + 2 * GPB, g_end, GPB); }
    }
    if (COLOUR) {      // flush the accumulator tile: one global reduction per non-zero node value
        __syncthreads();
        for (int j = threadIdx.x; j < TG::NN; j += kTB) {
            int idx[DIM];
            const int node = tile_node_global<DIM>(gd, org, j, idx);
            if (node < 0) continue;
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                const double v = s_acc[j * DIM + a];
                if (v != 0.0) acc_add<false>(g.mv2[a], node, v);      // COLOUR: fp64 accumulation only
            }
        }
    }
    // particles that changed cell in this step (mpm_stats.n_cell_changes): one atomic per block
    n_moved = __reduce_add_sync(kFull, n_moved);
    if (lane == 0 && n_moved) atomicAdd(&s_moved, n_moved);
    __syncthreads();
    if (threadIdx.x == 0 && s_moved) atomicAdd(n_cell_changes, (unsigned long long)s_moved);
}

// ------------------------------------------------------------------------------------------------ Alg. 1 l.10-13 + l.3 of the next step
// One block (kTB threads) per item; the tile's vbar and v2 = mv2/m are staged in shared memory.  D = trace
// G2PD(mv2/m) (eq. 19); Q (eq. 4), E', rho'; V' is read back from the gather kernel; CFL maxima;
// X' = X + dt Vbar; the particle is written to its cell-sorted slot of the OTHER buffer (l.12).  Then
// P2G#1 of the NEXT step at X' into the node accumulators `gn` (the other buffer of m, mv, f): a
// particle that stays in its cell joins the group's butterfly, the others are scattered by the whole warp (coop_p2g1).
// Particle fields of the next pass arrive in shared memory as in the gather kernel (cp.async or bulk copies).
template <int DIM>
struct UpdSmem {
    using TG = TileGeo<DIM>;
    static constexpr int CH = 2 * DIM;                      // doubles per staged node: vbar, v2
    static constexpr int NF = 2 * DIM + 3;                  // x[d], v[d], m, rho, e
    static constexpr int NW = kTB / 32;                     // warps: each has its own slot window of kWin slots per field
    static constexpr size_t TILE = sizeof(double) * TG::NN * CH;
    static constexpr size_t PF = sizeof(double) * NW * NF * kWin;
    static constexpr size_t DEST = sizeof(unsigned) * NW * kWin;      // destination records (ranks)
    static constexpr size_t ID = sizeof(int) * NW * kWin;
    static constexpr size_t BAR = sizeof(unsigned long long) * NW * 2;
    static constexpr size_t BYTES = TILE + PF + DEST + ID + BAR;
    static constexpr int NACC = 2 * DIM + 1;                // COLOUR: accumulator tile of m, mv, f behind the rest
    static constexpr size_t ACC = sizeof(double) * TG::NN * NACC;
    static_assert(TILE % 16 == 0 && PF % 16 == 0 && DEST % 16 == 0 && ID % 16 == 0 && BAR % 16 == 0, "16-byte aligned sections");
};

template <int DIM, bool ACC32, bool BULK, bool COLOUR, bool CM>
__global__ void __launch_bounds__(kTB, COLOUR ? 3 : DIM == 2 ? kTBMinU2 : kTBMinU) k_update_tiled(GridDesc gd, PArr p, PArr q, GArr g, DevScalars *sc, SortedMap map,
                                                              const int4 *__restrict__ items, const int *__restrict__ n_items,
                                                              const int *__restrict__ off_new,
                                                              const unsigned *__restrict__ dest, GArr gn, int store_q)
{
    using TG = TileGeo<DIM>;
    using SM = UpdSmem<DIM>;
    constexpr int NB = 1 << DIM, LG = Geo<DIM>::LG, GPB = kTB / LG, CH = SM::CH;
    extern __shared__ __align__(16) unsigned char s_raw[];
    double *s_tile = reinterpret_cast<double *>(s_raw);
    double (*s_pf)[SM::NF][kWin] = reinterpret_cast<double (*)[SM::NF][kWin]>(s_raw + SM::TILE);
    unsigned (*s_dest)[kWin] = reinterpret_cast<unsigned (*)[kWin]>(s_raw + SM::TILE + SM::PF);
    int (*s_id)[kWin] = reinterpret_cast<int (*)[kWin]>(s_raw + SM::TILE + SM::PF + SM::DEST);
    unsigned long long (*s_bar)[2] = reinterpret_cast<unsigned long long (*)[2]>(s_raw + SM::TILE + SM::PF + SM::DEST + SM::ID);
    double *s_acc = reinterpret_cast<double *>(s_raw + SM::BYTES);      // COLOUR only
    __shared__ double s_v[kTB / 32], s_c[kTB / 32];
    if ((int)blockIdx.x >= *n_items) return;
    const int4 item = __ldg(items + blockIdx.x);
    if (item.z == 0) return;
    const int l = threadIdx.x % LG, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int g_end = item.y + item.z;
    int gl = threadIdx.x / LG;
    Group grp = fetch_group(map.groups, (long long)item.y + gl, g_end);
    Group nxt = fetch_group(map.groups, (long long)item.y + gl + GPB, g_end);
    // two copy groups per pass: X and the destination record (needed first, refilled as soon as they have been read: a
    // whole pass of lead time) and the fields that are only needed after the gather
    if (BULK) {
        if (lane == 0) { mbar_init(&s_bar[warp][0], 1); mbar_init(&s_bar[warp][1], 1); mbar_fence_init(); }
        __syncwarp();
    }
    auto issue_x = [&](const Group &gr, int w0, int wn) {
        if (!BULK) {
            if (2 * l < gr.cnt) {
                const long long k0 = (long long)gr.first + 2 * l;
#pragma unroll
                for (int a = 0; a < DIM; ++a) cp_async16(&s_pf[warp][a][2 * lane], p.x[a] + k0);
                cp_async8(&s_dest[warp][2 * lane], dest + k0);
            }
            cp_async_commit();
        } else if (lane == 0) {
            mbar_arrive_expect_tx(&s_bar[warp][0], (unsigned)(DIM * wn * 8 + wn * 4));
            if (wn > 0) {
#pragma unroll
                for (int a = 0; a < DIM; ++a) bulk_g2s(&s_pf[warp][a][0], p.x[a] + w0, (unsigned)(wn * 8), &s_bar[warp][0]);
                bulk_g2s(&s_dest[warp][0], dest + w0, (unsigned)(wn * 4), &s_bar[warp][0]);
            }
        }
    };
    const bool ids = gd.track_ids != 0;      // the persistent ids travel with the particles (else the id arrays are not touched)
    auto issue_rest = [&](const Group &gr, int w0, int wn) {
        if (!BULK) {
            if (2 * l < gr.cnt) {
                const long long k0 = (long long)gr.first + 2 * l;
#pragma unroll
                for (int a = 0; a < DIM; ++a) cp_async16(&s_pf[warp][DIM + a][2 * lane], p.v[a] + k0);
                if (!gd.uniform_mass) cp_async16(&s_pf[warp][2 * DIM][2 * lane], p.m + k0);
                cp_async16(&s_pf[warp][2 * DIM + 1][2 * lane], p.rho + k0);
                cp_async16(&s_pf[warp][2 * DIM + 2][2 * lane], p.e + k0);
                if (ids) cp_async8(&s_id[warp][2 * lane], p.id + k0);
            }
            cp_async_commit();
        } else if (lane == 0) {
            const int nf = gd.uniform_mass ? DIM + 2 : DIM + 3;
            mbar_arrive_expect_tx(&s_bar[warp][1], (unsigned)(nf * wn * 8 + (ids ? wn * 4 : 0)));
            if (wn > 0) {
#pragma unroll
                for (int a = 0; a < DIM; ++a) bulk_g2s(&s_pf[warp][DIM + a][0], p.v[a] + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
                if (!gd.uniform_mass) bulk_g2s(&s_pf[warp][2 * DIM][0], p.m + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
                bulk_g2s(&s_pf[warp][2 * DIM + 1][0], p.rho + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
                bulk_g2s(&s_pf[warp][2 * DIM + 2][0], p.e + w0, (unsigned)(wn * 8), &s_bar[warp][1]);
                if (ids) bulk_g2s(&s_id[warp][0], p.id + w0, (unsigned)(wn * 4), &s_bar[warp][1]);
            }
        }
    };
    int w0, wn, w0n, wnn;
    warp_window<BULK>(grp.first, grp.cnt, w0, wn);
    warp_window<BULK>(nxt.first, nxt.cnt, w0n, wnn);
    issue_x(grp, w0, wn);
    issue_rest(grp, w0, wn);
    int org[DIM];
    tile_origin<DIM>(gd, item.x, org);
    const double dt = sc->dt;
    const long long step = sc->step;
    stage_tile<DIM, CH, true, ACC32>(gd, org, g, dt, s_tile);
    if (COLOUR) for (int j = threadIdx.x; j < TG::NN * SM::NACC; j += kTB) s_acc[j] = 0.0;
    PassColours<DIM> pc{ 0, 0 }, pcn{ 0, 0 };
    if (COLOUR) { pc = pass_colours<DIM>(map.groups, item.y, g_end, GPB); pcn = pass_colours<DIM>(map.groups, item.y + GPB, g_end, GPB); }
    __syncthreads();
    double vloc = 0.0, cloc = 0.0;
    // per-thread event counters of the block's <= 16 passes x 2 particles, packed into one register: recycled (bits 0-5),
    // clamped coordinates (6-12, <= 3 per particle), 1 + dt D <= 0 (13-18), non-finite (19-24), out of cell (25-30)
    unsigned events = 0u;
    int n_left = 0;      // particles that ended beyond an OPEN face (slab interfaces only)
    static_assert(Chunk<DIM>::PASSES * 2 <= 32, "event counters are 6 bits wide");
    const double gm1 = gd.gamma - 1.0;
    unsigned parity = 0;
    for (int p0 = 0; p0 < item.z; p0 += GPB, gl += GPB, parity ^= 1u) {
        int c[DIM];
        unpack_coords<DIM>(grp.cpack, c);
        const int local = grp.cell & (TG::TC - 1);
        const int j0 = TG::node0_of(local, CM);
        const bool valid[2] = { 2 * l < grp.cnt, 2 * l + 1 < grp.cnt };
        double X[2][DIM];
        long long dst[2] = { -1, -1 };
        const int o = !BULK ? 2 * lane : valid[0] ? grp.first + 2 * l - w0 : 0;      // the lane's two particles inside the warp's window
        MPM_CHECK(o >= 0 && o + 2 <= kWin && (o & 1) == 0 && j0 >= 0 && j0 + corner_off<DIM>(NB - 1) < TG::NN);
        MPM_CHECK(!valid[0] || (grp.first >= 0 && (long long)grp.first + 2 * l + 1 < gd.slots && (grp.cell >> TG::LTC) == item.x));
        if (BULK) mbar_wait(&s_bar[warp][0], parity); // this pass's X and destination records have landed
        else cp_async_wait_but_one();
        // l.12: slot of a particle in the other buffer = first slot of its new cell + its rank there (the destination record
        // the gather kernel left).  The particles that stay in the group's cell share ONE offset, loaded here so that it
        // overlaps the gather; the others bin X' again after the move
        const uint2 trank = *reinterpret_cast<const uint2 *>(&s_dest[warp][o]);
        const int off_cell = __ldg(off_new + grp.cell);
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const double2 tx = *reinterpret_cast<const double2 *>(&s_pf[warp][a][o]);
            X[0][a] = valid[0] ? tx.x : 0.0; X[1][a] = valid[1] ? tx.y : 0.0;
        }
        if (BULK) __syncwarp();
        issue_x(nxt, w0n, wnn);                       // the window has been read: refill it for the next pass
        double W[2][DIM][2], xi[2][DIM], out[2][2 * DIM], Dh[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            weights_1d<DIM>(gd, X[i], c, xi[i], W[i]);
            events += (unsigned)(valid[i] && !in_unit_cell<DIM>(xi[i])) << 25;      // the exact-sort invariant (must never count)
        }
        gather_tile<DIM, CH, true>(s_tile + j0 * CH, W, out, Dh);
        // the fields that are only needed from here on stay in shared memory during the gather (register budget)
        if (BULK) mbar_wait(&s_bar[warp][1], parity); // ... they have landed (the next X may still be in flight)
        else cp_async_wait_but_one();
        double V[2][DIM], M[2], rho[2], E[2];
        int id[2];
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            const double2 tv = *reinterpret_cast<const double2 *>(&s_pf[warp][DIM + a][o]);
            V[0][a] = tv.x; V[1][a] = tv.y;      // an unused slot computes on whatever it holds: masked where it could be seen
        }
        {
            const double2 tm = gd.uniform_mass ? make_double2(gd.um, gd.um) : *reinterpret_cast<const double2 *>(&s_pf[warp][2 * DIM][o]);
            const double2 tr = *reinterpret_cast<const double2 *>(&s_pf[warp][2 * DIM + 1][o]),
                          te = *reinterpret_cast<const double2 *>(&s_pf[warp][2 * DIM + 2][o]);
            M[0] = valid[0] ? tm.x : 0.0; M[1] = valid[1] ? tm.y : 0.0;
            rho[0] = tr.x; rho[1] = tr.y;
            E[0] = te.x; E[1] = te.y;
            const int2 ti = ids ? *reinterpret_cast<const int2 *>(&s_id[warp][o]) : make_int2(0, 0);
            id[0] = ti.x; id[1] = ti.y;
        }
        if (BULK) __syncwarp();
        issue_rest(nxt, w0n, wnn);
        // the group record of the pass after the next: loaded here, unpacked at the end of this pass (staging the records in
        // shared memory as the gather kernel does was measured slower here: 4 x 8 KB less L1 per SM)
        const int4 nn_raw = raw_group(map.groups, (long long)item.y + gl + 2 * GPB, g_end);
        // per particle: the new state (what goes to memory), S' for the next step's force, and whether it stays in the
        // group's cell.  Straight-line code for both particles of the lane (an unused slot computes on M = 0, X = 0 and
        // whatever V, rho, E its slot holds -- possibly NaN -- and is masked by SELECTS, never by a multiplication with 0,
        // wherever it could be seen: counters, maxima, stores, scatter payloads).
        double Xo[2][DIM], Vo[2][DIM], Mo[2], Ro[2], Eo[2], Qo[2], Sn[2], xin[2][DIM];
        bool stay[2];
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const double D = Dh[i] * gd.inv_h;
#pragma unroll
            for (int a = 0; a < DIM; ++a) Vo[i][a] = V[i][a];      // V' = V + dt A, stored by the gather kernel
            // particle thermodynamics (eq. 4 with this step's D: reading A2).  P/rho = (gamma-1) E
            // and gamma P/rho = gamma (gamma-1) E are used in place of the quotients (one rounding apart).
            const double r = rho[i], e0 = E[i];
            const double cs0 = sqrt(gd.gamma * gm1 * e0);
            double Q, Q_over_rho;
            if (gd.visc_form == MPM_VISC_STANDARD) {
                Q_over_rho = gd.c0 * gd.h * gd.h * D * D - gd.c1 * gd.h * cs0 * D;
                Q = r * Q_over_rho;
            } else {
                Q = gd.c0 * (r * gd.h * D) * (r * gd.h * D) - gd.c1 * gd.h * cs0 * D;
                Q_over_rho = Q / r;
            }
            if (!(D < 0.0)) { Q = 0.0; Q_over_rho = 0.0; }      // eq. (4): only in compression
            double En = e0 - dt * (gm1 * e0 + Q_over_rho) * D;
            const double jac = fma(dt, D, 1.0);
            double rhon = r * rcp_newton(jac);      // rho' = rho / (1 + dt D); jac <= 0 is counted below
            if (valid[i]) {
                events += (unsigned)(jac <= 0.0) << 13;
                double vv = 0.0, vb2 = 0.0;
#pragma unroll
                for (int a = 0; a < DIM; ++a) { vv = fma(Vo[i][a], Vo[i][a], vv); vb2 = fma(out[i][a], out[i][a], vb2); }
                // E', rho', V' and Vbar (hence X' = X + dt Vbar) all finite?
                events += (unsigned)(!isfinite(En) || !isfinite(rhon) || !isfinite(vv + vb2)) << 19;
                vloc = fmax(vloc, fmax(vv, vb2));                // squared; the root is taken once at the end
                cloc = fmax(cloc, gd.gamma * gm1 * En);          // c_s^2 = gamma P'/rho' (the root is monotone: taken at the end)
            }
            double Mn = M[i];
            if (!move_inside<DIM>(gd, X[i], out[i], dt, Xo[i]) && valid[i]) {      // next to a domain face (rare)
                bool recycled;
                int nclamp;
                bool left = false;
                move_particle<DIM>(gd, X[i], out[i], dt, (long long)id[i], step, Xo[i], recycled, nclamp, &left);
                events += (unsigned)nclamp << 6;
                n_left += (int)left;
                if (recycled) {
#pragma unroll
                    for (int a = 0; a < DIM; ++a) Vo[i][a] = gd.inflow_v[a];
                    rhon = gd.inflow_rho; En = gd.inflow_e; Q = 0.0; Q_over_rho = 0.0; Mn = gd.inflow_mass;
                    events += 1u;
                }
            }
            Mo[i] = Mn; Ro[i] = rhon; Eo[i] = En; Qo[i] = Q;
            // S' = (P' + Q') M / rho' with P' = (gamma-1) rho' E' (eq. 3) and Q'/rho' = (Q'/rho) (1 + dt D)  (rho' = rho / (1 + dt D))
            Sn[i] = (gm1 * En + Q_over_rho * jac) * Mn;
            // l.12: still in the group's cell?  Then its slot follows from the cell's offset, else X' is binned again.  The
            // gather kernel took the same decision from the same X' (bit 31 of the record); a disagreement would corrupt the
            // re-ordering, so it is counted with the exact-sort invariant (n_out_of_cell: must never count)
            const unsigned rec = i ? trank.y : trank.x;
            stay[i] = stays_in_cell<DIM>(gd, Xo[i], c, xin[i]) && valid[i];
            events += (unsigned)(valid[i] && stay[i] != (bool)(rec >> 31)) << 25;
            if (valid[i]) {
                int key = grp.cell, first = off_cell;
                if (!stay[i]) { key = tiled_key_of_position<DIM, CM>(gd, Xo[i]); first = __ldg(off_new + key); }
                dst[i] = (long long)first + (long long)(rec & 0x7fffffffu);
                MPM_CHECK(key >= 0 && key < gd.Nkeys && dst[i] >= 0 && dst[i] < __ldg(off_new + key + 1) && dst[i] < gd.slots);
            }
        }
        // l.12: the particle goes to its cell-sorted slot of the other buffer; the two particles of a lane usually
        // keep adjacent slots (ranks of the stayers are consecutive), then each field is ONE 16-byte store
        if (valid[1] && dst[1] == dst[0] + 1 && (dst[0] & 1) == 0) {
            const long long d0 = dst[0];
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                st2(q.x[a], d0, Xo[0][a], Xo[1][a]);
                st2(q.v[a], d0, Vo[0][a], Vo[1][a]);
            }
            if (!gd.uniform_mass) st2(q.m, d0, Mo[0], Mo[1]);
            st2(q.rho, d0, Ro[0], Ro[1]);
            st2(q.e, d0, Eo[0], Eo[1]);
            if (store_q) st2(q.q, d0, Qo[0], Qo[1]);
            if (ids) *reinterpret_cast<int2 *>(q.id + d0) = make_int2(id[0], id[1]);
        } else {
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                if (!valid[i]) continue;
                const long long d = dst[i];
#pragma unroll
                for (int a = 0; a < DIM; ++a) { q.x[a][d] = Xo[i][a]; q.v[a][d] = Vo[i][a]; }
                if (!gd.uniform_mass) q.m[d] = Mo[i];
                q.rho[d] = Ro[i];
                q.e[d] = Eo[i];
                if (store_q) q.q[d] = Qo[i];
                if (ids) q.id[d] = id[i];
            }
        }
        // P2G#1 of the next step (eqs. 13, 14, 16, 18 at X')
#pragma unroll
        for (int i = 0; i < 2; ++i) {      // particles that leave the group's cell: scattered by the whole warp
            const unsigned mm = __ballot_sync(kFull, valid[i] && !stay[i]);
            if (mm) coop_p2g1<DIM, ACC32>(gd, gn, mm, Xo[i], Vo[i], Mo[i], Sn[i], lane);
        }
        double pay[2][DIM + 2], wnew[2][NB];      // the others join the group's butterfly: payload M, M V', S', weights at X'
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            swizzled_weights<DIM>(xin[i], l, wnew[i]);
            pay[i][0] = stay[i] ? Mo[i] : 0.0;
            pay[i][DIM + 1] = stay[i] ? Sn[i] : 0.0;
#pragma unroll
            for (int a = 0; a < DIM; ++a) pay[i][1 + a] = stay[i] ? Mo[i] * Vo[i][a] : 0.0;
        }
        {
            double tot[SM::NACC][2];
            const bool issue = p2g1_group_totals<DIM>(gd, l, grp.cnt > 0, pay, wnew, warp_one_cell(grp.cell, grp.cnt), tot);
            int phase = -1;
            if (COLOUR) {      // eligible groups add into the shared accumulator tile, one colour at a time
                phase = colour_phase<DIM>(pc, grp);
                __syncthreads();                                   // the previous pass's additions are complete
                if (phase == 0 && issue) tile_accumulate<DIM, SM::NACC>(s_acc, j0, l, tot);
                if (pc.hi != pc.lo) {
                    __syncthreads();
                    if (phase == 1 && issue) tile_accumulate<DIM, SM::NACC>(s_acc, j0, l, tot);
                }
            }
            if (phase < 0 && issue) p2g1_commit_global<DIM, ACC32>(gd, gn, c, l, tot);
        }
        grp = nxt;
        nxt = unpack_group(nn_raw);
        w0 = w0n;
        wn = wnn;
        warp_window<BULK>(nxt.first, nxt.cnt, w0n, wnn);
        if (COLOUR) { pc = pcn; pcn = pass_colours<DIM>(map.groups, item.y + p0 + 2 * GPB, g_end, GPB); }
    }
    if (COLOUR) {      // flush the accumulator tile: one global reduction per non-zero node value
        __syncthreads();
        for (int j = threadIdx.x; j < TG::NN; j += kTB) {
            int idx[DIM];
            const int node = tile_node_global<DIM>(gd, org, j, idx);
            if (node < 0) continue;
            const double *src = s_acc + j * SM::NACC;
            if (src[0] != 0.0) acc_add<false>(gn.m, node, src[0]);      // COLOUR: fp64 accumulation only
#pragma unroll
            for (int a = 0; a < DIM; ++a) {
                if (src[1 + a] != 0.0) acc_add<false>(gn.mv[a], node, src[1 + a]);
                if (src[1 + DIM + a] != 0.0) acc_add<false>(gn.f[a], node, src[1 + DIM + a]);
            }
        }
    }
    // block maxima -> at most one atomicMax per block (max is order-free, so this is exact)
    vloc = warp_max_nonneg(sqrt(vloc));
    cloc = warp_max_nonneg(cloc > 0.0 ? sqrt(cloc) : 0.0);
    if (lane == 0) { s_v[warp] = vloc; s_c[warp] = cloc; }
    int rec_sum = 0, neg_sum = 0, nf_sum = 0, clamp_sum = 0, ooc_sum = 0;
    if (__any_sync(kFull, events != 0u)) {      // rare
        rec_sum = __reduce_add_sync(kFull, (int)(events & 63u));
        clamp_sum = __reduce_add_sync(kFull, (int)((events >> 6) & 127u));
        neg_sum = __reduce_add_sync(kFull, (int)((events >> 13) & 63u));
        nf_sum = __reduce_add_sync(kFull, (int)((events >> 19) & 63u));
        ooc_sum = __reduce_add_sync(kFull, (int)((events >> 25) & 63u));
    }
    if (lane == 0) {
        if (rec_sum) atomicAdd(&sc->n_recycled, (unsigned long long)rec_sum);
        if (neg_sum) atomicAdd(&sc->n_negjac, (unsigned long long)neg_sum);
        if (nf_sum) atomicAdd(&sc->n_nonfinite, (unsigned long long)nf_sum);
        if (clamp_sum) atomicAdd(&sc->n_clamped, (unsigned long long)clamp_sum);
        if (ooc_sum) atomicAdd(&sc->n_out_of_cell, (unsigned long long)ooc_sum);
    }
    if (gd.has_open) {
        const int left_sum = __reduce_add_sync(kFull, n_left);
        if (lane == 0 && left_sum) atomicAdd(&sc->n_left_slab, (unsigned long long)left_sum);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = s_v[0], cc = s_c[0];
#pragma unroll
        for (int w = 1; w < kTB / 32; ++w) { v = fmax(v, s_v[w]); cc = fmax(cc, s_c[w]); }
        // a plain read filters out the blocks that cannot raise the maximum (it only ever grows during the kernel)
        const unsigned long long vb = (unsigned long long)__double_as_longlong(v), cb = (unsigned long long)__double_as_longlong(cc);
        if (vb > *(volatile unsigned long long *)&sc->vmax_bits) atomic_max_nonneg(&sc->vmax_bits, v);
        if (cb > *(volatile unsigned long long *)&sc->cmax_bits) atomic_max_nonneg(&sc->cmax_bits, cc);
    }
}

// ------------------------------------------------------------------------------------------------ cell map (Alg. 1 l.12)
// ONE kernel turns the per-key particle counts of the re-ordering into everything the next sweeps need (the grid-to-
// particle connectivity of PAPER.md:745-748: "count ... cumulative sum"):
//   off[key]    first slot of the key's particles: exclusive scan of the counts rounded up to even (even-aligned slots);
//   groups[]    one record {first slot, count, key, packed cell coordinates} per <= 2^d particles of a cell, key order;
//   items[]     work items of the tile kernels {tile, first group, groups, -}: item t < ntiles is the first
//               Chunk::GROUPS groups of tile t (possibly none), the further chunks of dense tiles are appended behind.
// Single pass: a block takes kMapKeys keys (whole tiles, kMapKeysPerThread per thread) in ticket order, scans (slots, groups) packed in one
// 64-bit word and gets its exclusive prefix by decoupled look-back over the published block states
// (flag << 62 | slots << 31 | groups; flag 1 = block aggregate, 2 = inclusive prefix).  `state` must be zero at launch.
struct CellMapState {
    unsigned long long ticket_done;      // low 32 bits: next block ticket; the kernel's last block resets nothing (memset per launch)
    int extra;                           // chunks appended behind the per-tile items
    int done;                            // blocks finished
    unsigned long long block[1];         // [n_blocks]
};
#ifndef MPM_MAP_KPT
#define MPM_MAP_KPT 16
#endif
constexpr int kMapBlock = 256, kMapKeysPerThread = MPM_MAP_KPT, kMapKeys = kMapBlock * kMapKeysPerThread;

template <int DIM>
__global__ void __launch_bounds__(kMapBlock) k_cell_map_tiled(GridDesc gd, const int *__restrict__ count, int *__restrict__ off,
                                                              int4 *__restrict__ groups, int *__restrict__ n_groups,
                                                              int4 *__restrict__ items, int *__restrict__ n_items,
                                                              CellMapState *state, int nkeys, int ntiles, int n_blocks, int per_item)
{
    constexpr int CAP = 1 << DIM, TPT = TileGeo<DIM>::TC / kMapKeysPerThread;      // threads per tile (64)
    constexpr unsigned long long FIELD = (1ull << 31) - 1ull;
    __shared__ unsigned long long s_warp[kMapBlock / 32], s_excl[kMapBlock + 1], s_prefix;
    __shared__ int s_bid;
    if (threadIdx.x == 0) s_bid = (int)atomicAdd(&state->ticket_done, 1ull);
    __syncthreads();
    const int bid = s_bid;
    const int key0 = bid * kMapKeys + (int)threadIdx.x * kMapKeysPerThread;
    int c[kMapKeysPerThread];
#pragma unroll
    for (int j = 0; j < kMapKeysPerThread; ++j) c[j] = 0;
    if (key0 < nkeys) {      // nkeys is a multiple of the tile size, hence of the keys per thread
#pragma unroll
        for (int j = 0; j < kMapKeysPerThread; j += 4) {
            const int4 t = __ldg(reinterpret_cast<const int4 *>(count + key0 + j));
            c[j] = t.x; c[j + 1] = t.y; c[j + 2] = t.z; c[j + 3] = t.w;
        }
    }
    unsigned long long mine = 0ull;
#pragma unroll
    for (int j = 0; j < kMapKeysPerThread; ++j)
        mine += ((unsigned long long)((c[j] + 1) & ~1) << 31) | (unsigned long long)((c[j] + CAP - 1) / CAP);
    // block-wide exclusive scan of `mine`
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned long long wbase = 0ull, total = 0ull;
#pragma unroll
    for (int w = 0; w < kMapBlock / 32; ++w) {
        if (w < warp) wbase += s_warp[w];
        total += s_warp[w];
    }
    const unsigned long long excl_local = wbase + incl - mine;
    s_excl[threadIdx.x] = excl_local;
    if (warp == 0) {      // decoupled look-back, 32 predecessors at a time
        volatile unsigned long long *st = state->block;
        constexpr unsigned long long VAL = (1ull << 62) - 1ull;
        unsigned long long prefix = 0ull;
        if (bid > 0 && lane == 0) st[bid] = (1ull << 62) | total;
        for (int j = bid - 1; j >= 0; j -= 32) {
            const int idx = j - lane;
            unsigned long long v;
            do { v = (idx >= 0) ? st[idx] : (2ull << 62); } while (__any_sync(0xffffffffu, (v >> 62) == 0ull));
            const unsigned full = __ballot_sync(0xffffffffu, (v >> 62) == 2ull);      // lanes that hold an inclusive prefix
            const int stop = full ? __ffs(full) - 1 : 32;                             // the nearest one ends the walk
            unsigned long long val = (lane <= stop) ? (v & VAL) : 0ull;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
            prefix += val;
            if (full) break;
        }
        if (lane == 0) {
            __threadfence();
            st[bid] = (2ull << 62) | (prefix + total);
            s_prefix = prefix;
            s_excl[kMapBlock] = total;
        }
    }
    __syncthreads();
    const unsigned long long base = s_prefix + excl_local;
    int slot = (int)(base >> 31), g = (int)(base & FIELD);
    if (key0 < nkeys) {
        int o4[kMapKeysPerThread];
#pragma unroll
        for (int j = 0; j < kMapKeysPerThread; ++j) {
            o4[j] = slot;
            const int key = key0 + j;
            if (c[j] > 0) {
                int cc[DIM];
                tiled_cell_of_key<DIM>(gd, key, cc);
                const int cpack = (DIM == 3) ? (cc[0] | (cc[1] << 10) | (cc[DIM - 1] << 20)) : (cc[0] | (cc[1] << 16));
                for (int first = 0; first < c[j]; first += CAP, ++g) {
                    MPM_CHECK(g >= 0 && g < gd.max_groups && (long long)slot + c[j] <= gd.slots);
                    groups[g] = make_int4(slot + first, min(CAP, c[j] - first) | (c[j] > CAP ? 0x100 : 0), key, cpack);
                }
            }
            slot += (c[j] + 1) & ~1;
        }
#pragma unroll
        for (int j = 0; j < kMapKeysPerThread; j += 4) *reinterpret_cast<int4 *>(off + key0 + j) = make_int4(o4[j], o4[j + 1], o4[j + 2], o4[j + 3]);
        // work items of the tile this thread starts
        if ((threadIdx.x % TPT) == 0) {
            const int tile = key0 >> TileGeo<DIM>::LTC;
            const int gfirst = (int)((s_prefix + excl_local) & FIELD);
            const int ng = (int)((s_excl[threadIdx.x + TPT] - excl_local) & FIELD);
            items[tile] = make_int4(tile, gfirst, min(ng, per_item), 0);
            if (ng > per_item) {
                const int more = (ng - 1) / per_item;
                int at = ntiles + atomicAdd(&state->extra, more);
                for (int done = per_item; done < ng; done += per_item) {
                    MPM_CHECK(at >= 0 && at < gd.max_items);
                    items[at++] = make_int4(tile, gfirst + done, min(per_item, ng - done), 0);
                }
            }
        }
    }
    if (bid == n_blocks - 1 && threadIdx.x == 0) {
        const unsigned long long all = s_prefix + s_excl[kMapBlock];
        off[nkeys] = (int)(all >> 31);
        *n_groups = (int)(all & FIELD);
    }
    // the last block to finish publishes the item count
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&state->done, 1) == n_blocks - 1) *n_items = ntiles + atomicAdd(&state->extra, 0);
    }
}

// dst[id] = src[slot] for every occupied slot (one thread per group); coff != NULL: dst[compact storage index] instead
__global__ void __launch_bounds__(kBlock) k_gather_by_id_groups(const double *src, const int *id, double *dst, SortedMap map,
                                                                const int *coff, const int *off)
{
    const int n_groups = *map.n_groups;
    for (long long gq = (long long)blockIdx.x * kBlock + threadIdx.x; gq < n_groups; gq += (long long)gridDim.x * kBlock) {
        const int4 r = map.groups[gq];
        for (int j = 0; j < (r.y & 0xff); ++j) {
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
        for (int j = 0; j < (r.y & 0xff); ++j) {
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


__global__ void __launch_bounds__(kBlock) k_mass_differs(const double *__restrict__ m, long long n, int *flag)
{
    const long long first = __double_as_longlong(m[0]);
    bool differs = false;
    for (long long k = (long long)blockIdx.x * kBlock + threadIdx.x; k < n; k += (long long)gridDim.x * kBlock)
        differs = differs || __double_as_longlong(m[k]) != first;
    if (__any_sync(0xffffffffu, differs) && (threadIdx.x & 31) == 0) atomicOr(flag, 1);
}

__global__ void __launch_bounds__(kBlock) k_fill(double *m, long long n, double value)
{
    for (long long k = (long long)blockIdx.x * kBlock + threadIdx.x; k < n; k += (long long)gridDim.x * kBlock) m[k] = value;
}

// persistent launch: as many blocks as are resident at once (occupancy query), never more than there are chunks
template <typename Kernel>
inline unsigned persistent_blocks(long long max_groups, int groups_per_block, Kernel kernel)
{
    int dev = 0, sms = 148, per_sm = 1;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kBlock, 0) != cudaSuccess || per_sm < 1) per_sm = 1;
    const long long want = (long long)sms * per_sm;
    const long long need = (max_groups + groups_per_block - 1) / groups_per_block;
    return (unsigned)(need < want ? (need > 0 ? need : 1) : want);
}

}  // namespace

// checked build: publish the array bounds the raw access helpers test against
static void set_checked_bounds(const GridDesc &gd, cudaStream_t s)
{
#if defined(MPM_CHECKED) && MPM_CHECKED
    cudaMemcpyToSymbolAsync(g_checked_nodes, &gd.Nn, sizeof(long long), 0, cudaMemcpyHostToDevice, s);
    cudaMemcpyToSymbolAsync(g_checked_slots, &gd.slots, sizeof(long long), 0, cudaMemcpyHostToDevice, s);
#else
    (void)gd; (void)s;
#endif
}

size_t cell_map_state_bytes(const GridDesc &gd)
{
    const long long n_blocks = (gd.Nkeys + kMapKeys - 1) / kMapKeys;
    return sizeof(CellMapState) + sizeof(unsigned long long) * (size_t)n_blocks;
}

void launch_cell_map_tiled(const GridDesc &gd, const int *count, int *off, int4 *groups, int *n_groups, int4 *items, int *n_items,
                           void *state, cudaStream_t s)
{
    long long ntiles = 1;
    for (int a = 0; a < gd.dim; ++a) ntiles *= gd.ntile[a];
    const int nkeys = (int)gd.Nkeys, n_blocks = (nkeys + kMapKeys - 1) / kMapKeys;
    cudaMemsetAsync(state, 0, cell_map_state_bytes(gd), s);
    CellMapState *st = reinterpret_cast<CellMapState *>(state);
    if (gd.dim == 2)
        k_cell_map_tiled<2><<<n_blocks, kMapBlock, 0, s>>>(gd, count, off, groups, n_groups, items, n_items, st, nkeys, (int)ntiles, n_blocks, Chunk<2>::GROUPS);
    else
        k_cell_map_tiled<3><<<n_blocks, kMapBlock, 0, s>>>(gd, count, off, groups, n_groups, items, n_items, st, nkeys, (int)ntiles, n_blocks, Chunk<3>::GROUPS);
}

void launch_p2g1_tiled(const GridDesc &gd, const PArr &p, const GArr &g, const SortedMap &map, long long max_groups, cudaStream_t s)
{
    if (max_groups <= 0) return;
    set_checked_bounds(gd, s);
#define MPM_LAUNCH_P2G1(D, A) \
    k_p2g1_tiled<D, A><<<persistent_blocks(max_groups, Geo<D>::GPB, k_p2g1_tiled<D, A>), kBlock, 0, s>>>(gd, p, g, map)
    if (gd.dim == 2) { if (gd.acc32) MPM_LAUNCH_P2G1(2, true); else MPM_LAUNCH_P2G1(2, false); }
    else { if (gd.acc32) MPM_LAUNCH_P2G1(3, true); else MPM_LAUNCH_P2G1(3, false); }
#undef MPM_LAUNCH_P2G1
}

void launch_mass_differs(const double *m, long long n, int *flag, cudaStream_t s)
{
    if (n > 0) k_mass_differs<<<148 * 8, kBlock, 0, s>>>(m, n, flag);
}

void launch_fill(double *m, long long n, double value, cudaStream_t s)
{
    if (n > 0) k_fill<<<148 * 8, kBlock, 0, s>>>(m, n, value);
}

long long max_items_tiled(const GridDesc &gd, long long max_groups)
{
    long long ntiles = 1;
    for (int a = 0; a < gd.dim; ++a) ntiles *= gd.ntile[a];
    const int per = gd.dim == 2 ? Chunk<2>::GROUPS : Chunk<3>::GROUPS;
    return ntiles + max_groups / per + 1;      // one item per tile + the further chunks of dense tiles
}

void launch_g2p_p2g2_tiled(const GridDesc &gd, const PArr &p, const GArr &g, const DevScalars *sc,
                           const SortedMap &map, const int4 *items, const int *n_items, long long max_items, int *count,
                           unsigned *dest, cudaStream_t s)
{
    if (max_items <= 0) return;
    set_checked_bounds(gd, s);
#define MPM_LAUNCH_G2P(D, A, B, C, CM) \
    k_g2p_p2g2_tiled<D, A, B, C, CM><<<(unsigned)max_items, kTB, 0, s>>>(gd, p, g, sc, map, items, n_items, count, dest, \
                                                                         const_cast<unsigned long long *>(&sc->n_cell_changes))
#define MPM_LAUNCH_G2P_A(D, A) do { if (gd.bulk_stream) MPM_LAUNCH_G2P(D, A, true, false, false); else MPM_LAUNCH_G2P(D, A, false, false, false); } while (0)
    if (gd.p2g_mode & MPM_P2G_COLOUR_G2P) {      // fp64 accumulation and the cp.async stream only (mpm_create checks)
        if (gd.dim == 2) MPM_LAUNCH_G2P(2, false, false, true, true); else MPM_LAUNCH_G2P(3, false, false, true, true);
    } else if (gd.colour_major) {                // the update kernel accumulates by colour: same cell numbering here
        if (gd.dim == 2) MPM_LAUNCH_G2P(2, false, false, false, true); else MPM_LAUNCH_G2P(3, false, false, false, true);
    } else if (gd.dim == 2) { if (gd.acc32) MPM_LAUNCH_G2P_A(2, true); else MPM_LAUNCH_G2P_A(2, false); }
    else { if (gd.acc32) MPM_LAUNCH_G2P_A(3, true); else MPM_LAUNCH_G2P_A(3, false); }
#undef MPM_LAUNCH_G2P_A
#undef MPM_LAUNCH_G2P
}

void launch_update_tiled(const GridDesc &gd, const PArr &p, const PArr &q, const GArr &g, DevScalars *sc,
                         const SortedMap &map, const int4 *items, const int *n_items, long long max_items, const int *off_new,
                         const unsigned *dest, const GArr &g_next, bool store_q, cudaStream_t s)
{
    if (max_items <= 0) return;
    set_checked_bounds(gd, s);
    const int sq = store_q ? 1 : 0;
    static_assert(UpdSmem<2>::BYTES % 16 == 0 && UpdSmem<3>::BYTES % 16 == 0, "the accumulator tile starts 16-byte aligned");
    // more than 48 KB of dynamic shared memory needs the opt-in; the attribute is per device, so it is set at every launch (a
    // host-side call without a synchronisation)
#define MPM_LAUNCH_UPD(D, A, B, C, CM, BYTES) do { \
    if ((BYTES) > 48 * 1024) cudaFuncSetAttribute(k_update_tiled<D, A, B, C, CM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(BYTES)); \
    k_update_tiled<D, A, B, C, CM><<<(unsigned)max_items, kTB, BYTES, s>>>(gd, p, q, g, sc, map, items, n_items, off_new, dest, g_next, sq); } while (0)
#define MPM_LAUNCH_UPD_A(D, A) do { if (gd.bulk_stream) MPM_LAUNCH_UPD(D, A, true, false, false, UpdSmem<D>::BYTES); else MPM_LAUNCH_UPD(D, A, false, false, false, UpdSmem<D>::BYTES); } while (0)
    if (gd.p2g_mode & MPM_P2G_COLOUR_UPDATE) {   // fp64 accumulation and the cp.async stream only (mpm_create checks)
        if (gd.dim == 2) MPM_LAUNCH_UPD(2, false, false, true, true, UpdSmem<2>::BYTES + UpdSmem<2>::ACC);
        else MPM_LAUNCH_UPD(3, false, false, true, true, UpdSmem<3>::BYTES + UpdSmem<3>::ACC);
    } else if (gd.colour_major) {                // the gather kernel accumulates by colour: same cell numbering here
        if (gd.dim == 2) MPM_LAUNCH_UPD(2, false, false, false, true, UpdSmem<2>::BYTES); else MPM_LAUNCH_UPD(3, false, false, false, true, UpdSmem<3>::BYTES);
    } else if (gd.dim == 2) { if (gd.acc32) MPM_LAUNCH_UPD_A(2, true); else MPM_LAUNCH_UPD_A(2, false); }
    else { if (gd.acc32) MPM_LAUNCH_UPD_A(3, true); else MPM_LAUNCH_UPD_A(3, false); }
#undef MPM_LAUNCH_UPD_A
#undef MPM_LAUNCH_UPD
}

// fp32 accumulators (node-major nm[N_n][8], v2[N_n][4]) brought to component-major fp64 arrays for mpm_read_grid
__global__ void __launch_bounds__(256) k_widen(const float4 *__restrict__ nm, const float4 *__restrict__ v2, GArr dst, int dim, long long n)
{
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
        const float4 a = nm[2 * i], b = nm[2 * i + 1], c = v2[i];
        dst.m[i] = a.x;
        dst.mv[0][i] = a.y; dst.mv[1][i] = a.z;
        dst.f[0][i] = b.x; dst.f[1][i] = b.y;
        dst.mv2[0][i] = c.x; dst.mv2[1][i] = c.y;
        if (dim == 3) { dst.mv[2][i] = a.w; dst.f[2][i] = b.z; dst.mv2[2][i] = c.z; }
    }
}
__global__ void __launch_bounds__(256) k_add_into(double *__restrict__ dst, const double *__restrict__ src, long long n)
{
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) dst[i] += src[i];
}
void launch_add_into(double *dst, const double *src, long long n, cudaStream_t s)
{
    if (n > 0) k_add_into<<<(unsigned)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8), 256, 0, s>>>(dst, src, n);
}
void launch_widen(const GridDesc &gd, const GArr &src32, const GArr &dst64, cudaStream_t s)
{
    if (gd.Nn > 0)
        k_widen<<<148 * 8, 256, 0, s>>>(reinterpret_cast<const float4 *>(src32.m), reinterpret_cast<const float4 *>(src32.mv2[0]), dst64, gd.dim, gd.Nn);
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
