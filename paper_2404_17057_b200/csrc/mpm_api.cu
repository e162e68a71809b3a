// mpm_api.cu -- the C ABI of include/mpm.h: handle, device memory, step sequencing.  Host code only enqueues;
// dt, t, the CFL maxima and all counters live in device memory (control stays on the device).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "mpm_internal.cuh"

using namespace mpm;

struct mpm_handle {
    mpm_config cfg;
    GridDesc gd;
    int variant;
    cudaStream_t stream;
    PArr pbuf[2];
    int cur;
    long long n, cap;
    GArr g;
    unsigned char *d_flag;
    double *d_normal[3];
    std::vector<unsigned char> h_flag;
    std::vector<double> h_normal;   // [dim][Nn]
    int *key, *rank, *count, *scan_aux;
    // TILED family: even-aligned slot offsets of the cell keys, group map, destination records
    int *off[1];
    int *coff;            // TILED: compact storage offsets, allocated on the first storage-order read
    // TILED: the node accumulators m, mv, f are double-buffered: the update kernel of step n already scatters P2G#1 of
    // step n+1 into the other set.  acc[acur] = the set the current / next mpm_step starts from (raw P2G#1).
    double *acc_m[2], *acc_mv[2][3], *acc_f[2][3], *acc_mv2[2][3];
    // TILED with fp32 accumulation: the sums are node-major instead, nm[N_n][8] = { m, mv[3], f[3], - } and v2[N_n][4] = { mv2[3], - }
    // (vector reductions, mpm_kernels_tiled.cu); the kernels find them behind g.m and g.mv2[0]
    float *acc32_nm[2], *acc32_v2[2];
    // TILED: the next step's accumulator set is cleared on a second stream while the gather kernel runs
    cudaStream_t side;
    cudaEvent_t ev_fork, ev_join;
    int acur;
    bool grid_final;      // TILED: the last step's m, mv, f, mv2 have been brought to their post-BC form for mpm_read_grid
    long long slots;      // TILED: allocated slots per particle array (particles + one spare slot per odd cell)
    int *n_groups;
    int4 *groups;
    int4 *items;          // TILED: work items of the tile kernels (one block each), rebuilt with the groups
    int *n_items;
    // TILED: the cell map (groups, items) of the NEXT step is built between the two sweeps of a step, while the update
    // kernel still walks the current one: second set, swapped at the end of the step
    int4 *groups_alt, *items_alt;
    int *n_groups_alt, *n_items_alt;
    void *map_state;      // scratch of launch_cell_map_tiled
    // TILED with fp32 accumulators: fp64 copies of the last step's m, mv, f, mv2 for mpm_read_grid (allocated on first use)
    double *rg_m, *rg_mv[3], *rg_f[3], *rg_mv2[3];
    long long max_items;
    unsigned long long *dest;   // TILED: destination records of l.12, one 32-bit rank per slot (8 bytes per slot are allocated:
                                // mpm_load_particles_ex stages the caller's 64-bit ids here)
    long long max_groups;
    DevScalars *sc;
    long long launches;
    long long steps_done;
    double *id_wide;      // scratch of mpm_read_particles(MPM_P_ID): ids as doubles, 2 x id_wide_slots
    long long id_wide_slots;
    bool external_ids;    // the caller chose the persistent ids (mpm_load_particles_ex): no read-back in id order
    std::vector<void *> allocations;
    std::string err;
    // optional per-kernel-class timers (CUDA events on the launching stream)
    bool profiling;
    struct Span { int cls; cudaEvent_t a, b; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> event_pool;
    double kernel_ms[MPM_K_COUNT];
    long long kernel_calls[MPM_K_COUNT];
};

static std::string g_create_error = "";

namespace {

// Every entry point runs on the handle's device whatever the caller's current device is, and restores the caller's
// device on return (one process may drive handles on several GPUs).
struct DeviceGuard {
    int prev;
    bool switched;
    explicit DeviceGuard(int device) : prev(-1), switched(false)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard &) = delete;
    DeviceGuard &operator=(const DeviceGuard &) = delete;
};

int fail(mpm_handle *h, int code, const std::string &msg)
{
    if (h) h->err = msg; else g_create_error = msg;
    return code;
}

#define MPM_CUDA(h, expr)                                                                        \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess)                                                                  \
            return fail(h, e__ == cudaErrorMemoryAllocation ? MPM_E_OOM : MPM_E_CUDA,            \
                        std::string(#expr) + ": " + cudaGetErrorString(e__));                    \
    } while (0)

void *dev_alloc(mpm_handle *h, size_t bytes)
{
    if (bytes == 0) bytes = 8;
    void *p = nullptr;
    if (h->cfg.alloc) p = h->cfg.alloc(bytes, (void *)h->stream, h->cfg.alloc_user);
    else if (cudaMalloc(&p, bytes) != cudaSuccess) p = nullptr;
    if (p) h->allocations.push_back(p);
    return p;
}

void dev_free(mpm_handle *h, void *p)
{
    if (!p) return;
    for (size_t i = 0; i < h->allocations.size(); ++i)
        if (h->allocations[i] == p) { h->allocations.erase(h->allocations.begin() + i); break; }
    if (h->cfg.free) h->cfg.free(p, h->cfg.alloc_user); else cudaFree(p);
}

template <typename T>
bool dev_alloc_t(mpm_handle *h, T **out, size_t count)
{
    *out = (T *)dev_alloc(h, sizeof(T) * count);
    return *out != nullptr;
}

// ---- obstacle setup on the host (setup only; normals are computed once) ------------------------

struct MaskView {
    const unsigned char *mask;
    const GridDesc *gd;
    // returns 1 masked, 0 free, -1 outside the domain
    int at(int cx, int cy, int cz) const
    {
        int c[3] = { cx, cy, cz };
        for (int a = 0; a < gd->dim; ++a) {
            if (gd->per[a]) c[a] = ((c[a] % gd->nc[a]) + gd->nc[a]) % gd->nc[a];
            else if (c[a] < 0 || c[a] >= gd->nc[a]) return -1;
        }
        return mask[(size_t)c[0] + (size_t)gd->nc[0] * ((size_t)c[1] + (size_t)gd->nc[1] * (size_t)c[2])] ? 1 : 0;
    }
};

// windowed signed distance of reading A7: nearest masked-cell centre minus nearest free-cell centre, +-4 cells
double signed_distance(const MaskView &mv, const int node[3])
{
    const int W = 4;
    const GridDesc &gd = *mv.gd;
    double d_solid = (W + 1) * gd.h, d_free = (W + 1) * gd.h;
    int lo[3] = { 0, 0, 0 }, hi[3] = { 0, 0, 0 };
    for (int a = 0; a < gd.dim; ++a) { lo[a] = node[a] - W; hi[a] = node[a] + W - 1; }
    for (int cz = lo[2]; cz <= hi[2]; ++cz)
        for (int cy = lo[1]; cy <= hi[1]; ++cy)
            for (int cx = lo[0]; cx <= hi[0]; ++cx) {
                const int kind = mv.at(cx, cy, cz);
                if (kind < 0) continue;
                const int c[3] = { cx, cy, cz };
                double r2 = 0.0;
                for (int a = 0; a < gd.dim; ++a) {
                    const double d = ((double)c[a] + 0.5 - (double)node[a]) * gd.h;
                    r2 += d * d;
                }
                const double r = std::sqrt(r2);
                if (kind == 1) d_solid = std::min(d_solid, r); else d_free = std::min(d_free, r);
            }
    return d_solid - d_free;
}

void build_obstacle(mpm_handle *h, const unsigned char *mask, const double *normals)
{
    const GridDesc &gd = h->gd;
    h->h_flag.assign((size_t)gd.Nn, 0);
    h->h_normal.assign((size_t)gd.Nn * gd.dim, 0.0);
    MaskView mv{ mask, &gd };
    for (int iz = 0; iz < gd.nn[2]; ++iz)
        for (int iy = 0; iy < gd.nn[1]; ++iy)
            for (int ix = 0; ix < gd.nn[0]; ++ix) {
                bool flagged = false;   // node touches a solid cell
                for (int ib = 0; ib < (1 << gd.dim) && !flagged; ++ib) {
                    const int cz = gd.dim == 3 ? iz - ((ib >> 2) & 1) : 0;
                    flagged = mv.at(ix - (ib & 1), iy - ((ib >> 1) & 1), cz) == 1;
                }
                h->h_flag[(size_t)ix + (size_t)gd.nn[0] * ((size_t)iy + (size_t)gd.nn[1] * iz)] = flagged;
            }
    if (normals) {
        std::memcpy(h->h_normal.data(), normals, sizeof(double) * (size_t)gd.Nn * gd.dim);
        return;
    }
    for (int iz = 0; iz < gd.nn[2]; ++iz)
        for (int iy = 0; iy < gd.nn[1]; ++iy)
            for (int ix = 0; ix < gd.nn[0]; ++ix) {
                const size_t I = (size_t)ix + (size_t)gd.nn[0] * ((size_t)iy + (size_t)gd.nn[1] * iz);
                if (!h->h_flag[I]) continue;
                double grad[3] = { 0, 0, 0 }, nrm2 = 0.0;
                for (int a = 0; a < gd.dim; ++a) {
                    int up[3] = { ix, iy, iz }, dn[3] = { ix, iy, iz };
                    up[a] += 1; dn[a] -= 1;
                    grad[a] = (signed_distance(mv, up) - signed_distance(mv, dn)) / (2.0 * gd.h);   // eq. (24)
                    nrm2 += grad[a] * grad[a];
                }
                const double nrm = std::sqrt(nrm2);
                for (int a = 0; a < gd.dim; ++a) h->h_normal[(size_t)a * gd.Nn + I] = nrm > 0.0 ? grad[a] / nrm : 0.0;
            }
}

cudaEvent_t take_event(mpm_handle *h)
{
    if (!h->event_pool.empty()) { cudaEvent_t e = h->event_pool.back(); h->event_pool.pop_back(); return e; }
    cudaEvent_t e;
    cudaEventCreate(&e);
    return e;
}

// fold finished spans into kernel_ms (synchronises the stream)
void drain_spans(mpm_handle *h)
{
    if (h->spans.empty()) return;
    cudaStreamSynchronize(h->stream);
    for (auto &sp : h->spans) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, sp.a, sp.b) == cudaSuccess) { h->kernel_ms[sp.cls] += ms; h->kernel_calls[sp.cls] += 1; }
        h->event_pool.push_back(sp.a);
        h->event_pool.push_back(sp.b);
    }
    h->spans.clear();
}

struct Timed {   // RAII bracket of one kernel class
    mpm_handle *h; int cls; cudaEvent_t a;
    Timed(mpm_handle *h_, int cls_) : h(h_), cls(cls_), a(nullptr)
    {
        if (h->profiling) { a = take_event(h); cudaEventRecord(a, h->stream); }
    }
    ~Timed()
    {
        if (!a) return;
        cudaEvent_t b = take_event(h);
        cudaEventRecord(b, h->stream);
        h->spans.push_back({ cls, a, b });
        if (h->spans.size() >= 4096) drain_spans(h);
    }
};

void free_particles(mpm_handle *h)
{
    for (int b = 0; b < 2; ++b) {
        PArr &p = h->pbuf[b];
        for (int a = 0; a < 3; ++a) { dev_free(h, p.x[a]); dev_free(h, p.v[a]); p.x[a] = p.v[a] = nullptr; }
        dev_free(h, p.m); dev_free(h, p.rho); dev_free(h, p.e); dev_free(h, p.q); dev_free(h, p.id);
        p.m = p.rho = p.e = p.q = nullptr; p.id = nullptr;
    }
    dev_free(h, h->key); dev_free(h, h->rank);
    h->key = h->rank = nullptr;
    dev_free(h, h->dest); dev_free(h, h->groups);
    h->dest = nullptr; h->groups = nullptr;
    dev_free(h, h->items); dev_free(h, h->items_alt); dev_free(h, h->groups_alt);
    h->items = h->items_alt = nullptr; h->groups_alt = nullptr; h->max_items = 0;
    h->n = h->cap = 0;
}

int alloc_particles(mpm_handle *h, long long n)
{
    free_particles(h);
    // TILED: every cell's slot range starts at an even slot -> at most one unused slot per occupied cell
    const bool tiled = h->variant == MPM_VARIANT_TILED;
    h->slots = tiled ? n + (n < h->gd.Nc ? n : h->gd.Nc) + 8 : n;
    // slot indices, slot offsets and the look-back state of the cell map are 32-bit / 31-bit quantities
    if (h->slots >= (1ll << 31) - 1) return fail(h, MPM_E_ARG, "mpm_load_particles: too many particles for 32-bit slot indices");
    const size_t N = (size_t)(h->slots > 0 ? h->slots : 1);
    bool ok = true;
    for (int b = 0; b < 2 && ok; ++b) {
        PArr &p = h->pbuf[b];
        for (int a = 0; a < h->gd.dim && ok; ++a) ok = dev_alloc_t(h, &p.x[a], N) && dev_alloc_t(h, &p.v[a], N);
        ok = ok && dev_alloc_t(h, &p.m, N) && dev_alloc_t(h, &p.rho, N) && dev_alloc_t(h, &p.e, N) &&
             dev_alloc_t(h, &p.q, N) && dev_alloc_t(h, &p.id, N);
    }
    ok = ok && dev_alloc_t(h, &h->key, N) && dev_alloc_t(h, &h->rank, N);
    if (ok && tiled) {
        const long long gs = 1ll << h->gd.dim;
        h->max_groups = n / gs + (n < h->gd.Nc ? n : h->gd.Nc) + 1;
        ok = dev_alloc_t(h, &h->dest, N) && dev_alloc_t(h, &h->groups, (size_t)h->max_groups);
        if (ok) {
            h->max_items = max_items_tiled(h->gd, h->max_groups);
            ok = dev_alloc_t(h, &h->items, (size_t)h->max_items) && dev_alloc_t(h, &h->items_alt, (size_t)h->max_items) &&
                 dev_alloc_t(h, &h->groups_alt, (size_t)h->max_groups);
        }
    }
    if (!ok) { free_particles(h); return fail(h, MPM_E_OOM, "out of device memory for particle arrays"); }
    if (tiled) {   // unused slots are read (and masked) by the 128-bit loads: keep them finite
        for (int b = 0; b < 2; ++b) {
            PArr &p = h->pbuf[b];
            for (int a = 0; a < h->gd.dim; ++a) { cudaMemsetAsync(p.x[a], 0, 8 * N, h->stream); cudaMemsetAsync(p.v[a], 0, 8 * N, h->stream); }
            cudaMemsetAsync(p.m, 0, 8 * N, h->stream); cudaMemsetAsync(p.rho, 0, 8 * N, h->stream);
            cudaMemsetAsync(p.e, 0, 8 * N, h->stream); cudaMemsetAsync(p.q, 0, 8 * N, h->stream);
            cudaMemsetAsync(p.id, 0, 4 * N, h->stream);
        }
        cudaMemsetAsync(h->dest, 0, 8 * N, h->stream);
    }
    h->n = n; h->cap = n; h->cur = 0;
    h->gd.slots = h->slots; h->gd.max_groups = h->max_groups; h->gd.max_items = h->max_items;
    return MPM_OK;
}

// TILED: view of the grid arrays with (m, mv, f) = accumulator set `which`
GArr tiled_acc(const mpm_handle *h, int which)
{
    GArr g = h->g;
    g.m = h->acc_m[which];
    for (int a = 0; a < 3; ++a) { g.mv[a] = h->acc_mv[which][a]; g.f[a] = h->acc_f[which][a]; g.mv2[a] = h->acc_mv2[which][a]; }
    if (h->gd.acc32) {
        g.m = reinterpret_cast<double *>(h->acc32_nm[which]);
        g.mv2[0] = reinterpret_cast<double *>(h->acc32_v2[which]);
    }
    return g;
}

// Alg. 1 l.2 for an accumulator set of the TILED family: m, mv, f (the targets of P2G#1) / mv2 (of P2G#2)
void clear_p2g1(const mpm_handle *h, const GArr &g, cudaStream_t s)
{
    if (h->gd.acc32) cudaMemsetAsync(g.m, 0, sizeof(float) * 8 * (size_t)h->gd.Nn, s);
    else launch_grid_clear(h->gd, g, s);
}
void clear_p2g2(const mpm_handle *h, const GArr &g, cudaStream_t s)
{
    if (h->gd.acc32) { cudaMemsetAsync(g.mv2[0], 0, sizeof(float) * 4 * (size_t)h->gd.Nn, s); return; }
    for (int a = 0; a < h->gd.dim; ++a) cudaMemsetAsync(g.mv2[a], 0, sizeof(double) * (size_t)h->gd.Nn, s);
}

// cell-key counting sort of all particle arrays into the other buffer (Alg. 1 l.12).  TILED family: only after a
// load (every later step re-orders inside its own sweeps); it also builds the cell map and does the first P2G#1.
void reorder(mpm_handle *h)
{
    Timed timer(h, MPM_K_SORT);
    const PArr &src = h->pbuf[h->cur];
    const PArr &dst = h->pbuf[h->cur ^ 1];
    if (h->variant == MPM_VARIANT_TILED) {
        // counts per tile-major key -> even-rounded slot offsets -> permutation; then groups and the force payload
        launch_key_rank(h->gd, src, h->key, h->rank, h->count, h->n, h->stream);
        launch_cell_map_tiled(h->gd, h->count, h->off[0], h->groups, h->n_groups, h->items, h->n_items, h->map_state, h->stream);
        launch_permute(h->gd, src, dst, h->key, h->rank, h->off[0], h->n, h->stream);
        h->cur ^= 1;
        // P2G#1 of the first step (Alg. 1 l.3); every later one comes out of the update kernel of the step before
        h->acur = 0;
        h->grid_final = false;
        GArr g0 = tiled_acc(h, 0);
        clear_p2g1(h, g0, h->stream);
        clear_p2g2(h, g0, h->stream);
        launch_p2g1_tiled(h->gd, dst, g0, SortedMap{ h->groups, h->n_groups }, h->max_groups, h->stream);
        h->launches += 6;
        return;
    }
    launch_key_rank(h->gd, src, h->key, h->rank, h->count, h->n, h->stream);
    launch_exclusive_scan(h->count, h->gd.Nc + 1, h->scan_aux, h->stream);
    launch_permute(h->gd, src, dst, h->key, h->rank, h->count, h->n, h->stream);
    h->cur ^= 1;
    h->launches += 6;
}

// one step of Algorithm 1 with the TILED kernel family (see mpm_kernels_tiled.cu): l.3 of this step was done by the
// previous step's update kernel (or by the load), l.3 of the next step is done by this step's update kernel
// first half: dt, reset of the next accumulators, l.4-8 (gather kernel)
void step_tiled_gather(mpm_handle *h)
{
    const GridDesc &gd = h->gd;
    cudaStream_t s = h->stream;
    const PArr &p = h->pbuf[h->cur];
    const SortedMap map{ h->groups, h->n_groups };
    const GArr gc = tiled_acc(h, h->acur), gnx = tiled_acc(h, h->acur ^ 1);
    {
        Timed t(h, MPM_K_MISC);
        launch_begin_step(h->sc, gd.h, true, s);                                          // dt (eq. 25/29)
        // l.2 for the next step: its accumulator set (m, mv, f for l.3, mv2 for l.8; last read by the previous step's
        // update kernel) is cleared on the second stream while this step's gather kernel runs
        cudaEventRecord(h->ev_fork, s);
        cudaStreamWaitEvent(h->side, h->ev_fork, 0);
        clear_p2g1(h, gnx, h->side);
        clear_p2g2(h, gnx, h->side);
        cudaEventRecord(h->ev_join, h->side);
        cudaMemsetAsync(h->count, 0, sizeof(int) * (size_t)(gd.Nkeys + 1), s);            // per-cell counters of l.12
    }
    // l.4-5 and l.9 (BC, obstacle, mv' = mv + dt f, the quotients by m) have no kernel of their own: the two particle
    // kernels evaluate them per tile node while staging the tile (stage_tile)
    { Timed t(h, MPM_K_G2P_P2G2);
      launch_g2p_p2g2_tiled(gd, p, gc, h->sc, map, h->items, h->n_items, h->max_items, h->count, reinterpret_cast<unsigned *>(h->dest), s); }          // l.4-8
    h->launches += 2;      // kernels only (begin_step, gather); the memsets are not counted
}

// second half: cell map, l.9-13 and l.3 of the next step (update kernel), time advance
void step_tiled_update(mpm_handle *h, bool last_of_call)
{
    const GridDesc &gd = h->gd;
    cudaStream_t s = h->stream;
    const PArr &p = h->pbuf[h->cur];
    const PArr &q = h->pbuf[h->cur ^ 1];
    const SortedMap map{ h->groups, h->n_groups };
    const GArr gc = tiled_acc(h, h->acur), gnx = tiled_acc(h, h->acur ^ 1);
    { Timed t(h, MPM_K_SORT);                                                         // l.12: offsets, next step's groups and work items
      launch_cell_map_tiled(gd, h->count, h->off[0], h->groups_alt, h->n_groups_alt, h->items_alt, h->n_items_alt, h->map_state, s); }
    cudaStreamWaitEvent(s, h->ev_join, 0);
    { Timed t(h, MPM_K_UPDATE);
      launch_update_tiled(gd, p, q, gc, h->sc, map, h->items, h->n_items, h->max_items, h->off[0], reinterpret_cast<const unsigned *>(h->dest), gnx, last_of_call, s); }   // l.9-12, next l.3
    { Timed t(h, MPM_K_MISC); launch_end_step(h->sc, gd.h, s); }                                                   // l.13-14
    { int4 *t4 = h->groups; h->groups = h->groups_alt; h->groups_alt = t4; t4 = h->items; h->items = h->items_alt; h->items_alt = t4;
      int *t1 = h->n_groups; h->n_groups = h->n_groups_alt; h->n_groups_alt = t1; t1 = h->n_items; h->n_items = h->n_items_alt; h->n_items_alt = t1; }
    h->cur ^= 1;
    h->acur ^= 1;
    h->grid_final = false;
    h->launches += 3;      // kernels only (cell map, update, end_step)
}

void step_tiled(mpm_handle *h, bool last_of_call)
{
    step_tiled_gather(h);
    step_tiled_update(h, last_of_call);
}

int copy_in(mpm_handle *h, double *dst, const double *src, long long n, int loc)
{
    MPM_CUDA(h, cudaMemcpyAsync(dst, src, sizeof(double) * (size_t)n,
                                loc == MPM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
    return MPM_OK;
}

int copy_out(mpm_handle *h, double *dst, const double *src, long long n, int loc)
{
    MPM_CUDA(h, cudaMemcpyAsync(dst, src, sizeof(double) * (size_t)n,
                                loc == MPM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    return MPM_OK;
}

}  // namespace

extern "C" {

int mpm_abi_version(void) { return MPM_ABI_VERSION; }

const char *mpm_last_error(const mpm_handle *h) { return h ? h->err.c_str() : g_create_error.c_str(); }

namespace {
// a handle that never became visible to the caller: release what mpm_create has made so far
void discard(mpm_handle *h)
{
    if (h->side) cudaStreamDestroy(h->side);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    std::vector<void *> all = h->allocations;
    for (void *p : all) dev_free(h, p);
    delete h;
}
}  // namespace

int mpm_create(const mpm_config *cfg, mpm_handle **out)
{
    if (!cfg || !out) return fail(nullptr, MPM_E_ARG, "mpm_create: null argument");
    *out = nullptr;
    if (cfg->dim != 2 && cfg->dim != 3) return fail(nullptr, MPM_E_ARG, "mpm_create: dim must be 2 or 3");
    if (!(cfg->dx > 0.0) || !(cfg->gamma > 1.0)) return fail(nullptr, MPM_E_ARG, "mpm_create: need dx > 0 and gamma > 1");
    if (cfg->sort_every < 0) return fail(nullptr, MPM_E_ARG, "mpm_create: sort_every must be >= 0");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0)
        return fail(nullptr, MPM_E_CUDA, "mpm_create: no CUDA device (this library has no CPU fallback)");
    if (cfg->device < 0 || cfg->device >= ndev) return fail(nullptr, MPM_E_ARG, "mpm_create: bad device ordinal");
    DeviceGuard guard(cfg->device);
    {
        int now = -1;
        if (cudaGetDevice(&now) != cudaSuccess || now != cfg->device) return fail(nullptr, MPM_E_CUDA, "mpm_create: cudaSetDevice failed");
    }

    mpm_handle *h = new (std::nothrow) mpm_handle();
    if (!h) return fail(nullptr, MPM_E_OOM, "mpm_create: host allocation failed");
    h->cfg = *cfg;
    h->stream = (cudaStream_t)cfg->stream;
    h->side = nullptr; h->ev_fork = h->ev_join = nullptr;
    if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess) {
        discard(h);
        return fail(nullptr, MPM_E_CUDA, "mpm_create: cannot create the second stream");
    }
    h->cur = 0; h->n = h->cap = 0; h->launches = 0; h->steps_done = 0; h->external_ids = false; h->id_wide = nullptr; h->id_wide_slots = 0;
    h->profiling = false;
    for (int k = 0; k < MPM_K_COUNT; ++k) { h->kernel_ms[k] = 0.0; h->kernel_calls[k] = 0; }
    h->d_flag = nullptr; h->key = h->rank = h->count = h->scan_aux = nullptr; h->sc = nullptr;
    h->off[0] = nullptr; h->n_groups = nullptr; h->groups = nullptr;
    h->items = nullptr; h->n_items = nullptr; h->max_items = 0;
    h->rg_m = nullptr; for (int a = 0; a < 3; ++a) h->rg_mv[a] = h->rg_f[a] = h->rg_mv2[a] = nullptr;
    h->acc32_nm[0] = h->acc32_nm[1] = h->acc32_v2[0] = h->acc32_v2[1] = nullptr;
    h->groups_alt = h->items_alt = nullptr; h->n_groups_alt = h->n_items_alt = nullptr; h->map_state = nullptr;
    h->dest = nullptr; h->max_groups = 0; h->coff = nullptr; h->slots = 0;
    std::memset(h->pbuf, 0, sizeof(h->pbuf));
    std::memset(&h->g, 0, sizeof(h->g));
    for (int a = 0; a < 3; ++a) h->d_normal[a] = nullptr;

    GridDesc &gd = h->gd;
    std::memset(&gd, 0, sizeof(gd));
    gd.dim = cfg->dim; gd.h = cfg->dx; gd.inv_h = 1.0 / cfg->dx;
    gd.gamma = cfg->gamma; gd.c0 = cfg->c0; gd.c1 = cfg->c1; gd.visc_form = cfg->visc_form;
    gd.Nn = 1; gd.Nc = 1;
    for (int a = 0; a < 3; ++a) {
        if (a < gd.dim) {
            const bool p0 = cfg->bc[a][0] == MPM_BC_PERIODIC, p1 = cfg->bc[a][1] == MPM_BC_PERIODIC;
            if (cfg->n[a] < 1 || p0 != p1) {
                discard(h);
                return fail(nullptr, MPM_E_ARG, "mpm_create: n[a] >= 1 and PERIODIC on both sides of an axis required");
            }
            gd.nc[a] = cfg->n[a]; gd.per[a] = p0; gd.nn[a] = p0 ? cfg->n[a] : cfg->n[a] + 1;
            gd.L[a] = (double)cfg->n[a] * cfg->dx;
            gd.bc[a][0] = cfg->bc[a][0]; gd.bc[a][1] = cfg->bc[a][1];
        } else {
            gd.nc[a] = 1; gd.nn[a] = 1; gd.per[a] = 0; gd.L[a] = 0.0;
        }
        gd.Nn *= gd.nn[a]; gd.Nc *= gd.nc[a];
    }
    if (gd.Nc >= (1ll << 31) - 2 || gd.Nn >= (1ll << 31) - 2) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: grid too large for 32-bit cell keys");
    }
    gd.in_axis = -1; gd.in_side = 0;
    for (int a = 0; a < gd.dim && gd.in_axis < 0; ++a)
        for (int s = 0; s < 2; ++s)
            if (cfg->bc[a][s] == MPM_BC_INFLOW) { gd.in_axis = a; gd.in_side = s; break; }
    for (int a = 0; a < 3; ++a) gd.inflow_v[a] = cfg->inflow_v[a];
    gd.inflow_rho = cfg->inflow_rho;
    gd.inflow_e = cfg->inflow_p / ((cfg->gamma - 1.0) * cfg->inflow_rho);
    double vol = 1.0;
    for (int a = 0; a < gd.dim; ++a) vol *= gd.h;
    gd.inflow_mass = cfg->inflow_rho * vol / (cfg->ppc_inflow > 0.0 ? cfg->ppc_inflow : 1.0);
    gd.recycle_seed = cfg->recycle_seed;
    gd.has_obstacle = cfg->obstacle_mask != nullptr;

    h->variant = cfg->variant == MPM_VARIANT_AUTO
                     ? (cfg->sort_every == 1 && cfg->basis == MPM_BASIS_Q1 ? MPM_VARIANT_TILED : MPM_VARIANT_ATOMIC)
                     : cfg->variant;
    if (h->variant != MPM_VARIANT_ATOMIC && h->variant != MPM_VARIANT_TILED) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, cfg->variant == MPM_VARIANT_SORTED_RETIRED
                                            ? "mpm_create: the SORTED kernel family was retired (superseded by TILED)"
                                            : "mpm_create: unknown kernel variant");
    }
    const bool tiled = h->variant == MPM_VARIANT_TILED;
    const bool sorted = tiled;
    if (cfg->grid_accum != MPM_ACCUM_FP64 && !(cfg->grid_accum == MPM_ACCUM_FP32 && tiled)) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: grid_accum must be MPM_ACCUM_FP64, or MPM_ACCUM_FP32 with the TILED family");
    }
    if (cfg->particle_stream != MPM_STREAM_CP_ASYNC && !(cfg->particle_stream == MPM_STREAM_BULK && tiled)) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: particle_stream must be MPM_STREAM_CP_ASYNC, or MPM_STREAM_BULK with the TILED family");
    }
    if (cfg->p2g_mode != MPM_P2G_RED &&
        !(cfg->p2g_mode > 0 && cfg->p2g_mode <= MPM_P2G_COLOUR_BOTH && tiled && cfg->grid_accum == MPM_ACCUM_FP64 &&
          cfg->particle_stream == MPM_STREAM_CP_ASYNC)) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: p2g_mode MPM_P2G_COLOUR_* needs the TILED family, fp64 accumulation and the cp.async stream");
    }
    if (cfg->particle_ids != MPM_IDS_TRACK && cfg->particle_ids != MPM_IDS_NONE) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: particle_ids must be MPM_IDS_TRACK or MPM_IDS_NONE");
    }
    if (cfg->basis != MPM_BASIS_Q1) {
        bool ok = cfg->basis == MPM_BASIS_QUADRATIC && !tiled && !cfg->obstacle_mask;
        for (int a = 0; a < gd.dim; ++a) ok = ok && gd.per[a] && gd.nc[a] >= 3;
        if (!ok) {
            discard(h);
            return fail(nullptr, MPM_E_ARG, "mpm_create: MPM_BASIS_QUADRATIC needs the ATOMIC family and a fully periodic grid of >= 3 cells per axis without obstacle");
        }
    }
    gd.quadratic = cfg->basis == MPM_BASIS_QUADRATIC ? 1 : 0;
    // persistent ids: dropped on request by the TILED family when nothing on the device needs them (the recycling generator of
    // an INFLOW face is keyed on them, reading A8)
    gd.track_ids = (cfg->particle_ids == MPM_IDS_NONE && tiled && gd.in_axis < 0) ? 0 : 1;
    if (cfg->slab_global_n < 0 || cfg->slab_offset < 0 ||
        (cfg->slab_global_n > 0 && cfg->slab_offset + gd.nc[gd.dim - 1] > cfg->slab_global_n)) {
        discard(h);
        return fail(nullptr, MPM_E_ARG, "mpm_create: slab_offset + n[last] must not exceed slab_global_n");
    }
    gd.slab_global_n = cfg->slab_global_n; gd.slab_offset = cfg->slab_offset;
    gd.has_open = 0;
    for (int a = 0; a < gd.dim; ++a)
        for (int sd = 0; sd < 2; ++sd)
            if (cfg->bc[a][sd] == MPM_BC_OPEN) gd.has_open = 1;
    gd.tiled = tiled ? 1 : 0;
    gd.acc32 = cfg->grid_accum == MPM_ACCUM_FP32 ? 1 : 0;
    gd.bulk_stream = cfg->particle_stream == MPM_STREAM_BULK ? 1 : 0;
    gd.p2g_mode = cfg->p2g_mode;
    gd.colour_major = cfg->p2g_mode != MPM_P2G_RED ? 1 : 0;
    gd.Nkeys = gd.Nc;
    if (tiled) {    // tile-major key space (TileGeo): whole tiles, so it can be larger than the number of cells
        long long nt = 1;
        for (int a = 0; a < 3; ++a) {
            const int lt = gd.dim == 3 ? (a == 0 ? TileGeo<3>::LT0 : a == 1 ? TileGeo<3>::LT1 : TileGeo<3>::LT2)
                                       : (a == 0 ? TileGeo<2>::LT0 : a == 1 ? TileGeo<2>::LT1 : 0);
            gd.ntile[a] = a < gd.dim ? (gd.nc[a] + (1 << lt) - 1) >> lt : 1;
            nt *= gd.ntile[a];
        }
        gd.Nkeys = nt * (gd.dim == 3 ? TileGeo<3>::TC : TileGeo<2>::TC);
        if (gd.Nkeys >= (1ll << 31) - 2) { discard(h); return fail(nullptr, MPM_E_ARG, "mpm_create: grid too large for 32-bit tile keys"); }
    }
    if (sorted) {   // the group records pack the cell coordinates into one int
        const int lim = gd.dim == 3 ? 1024 : 65535;
        for (int a = 0; a < gd.dim; ++a)
            if (gd.nc[a] > lim) { discard(h); return fail(nullptr, MPM_E_ARG, "mpm_create: TILED family needs n[a] <= 1024 (3D) / 65535 (2D)"); }
    }

    // grid arrays
    bool ok = dev_alloc_t(h, &h->g.m, (size_t)gd.Nn);
    for (int a = 0; a < gd.dim && ok; ++a) {
        ok = dev_alloc_t(h, &h->g.mv[a], (size_t)gd.Nn) && dev_alloc_t(h, &h->g.f[a], (size_t)gd.Nn) &&
             dev_alloc_t(h, &h->g.mv2[a], (size_t)gd.Nn);
        if (ok && !sorted)
            ok = dev_alloc_t(h, &h->g.vbar[a], (size_t)gd.Nn) && dev_alloc_t(h, &h->g.acc[a], (size_t)gd.Nn) &&
                 dev_alloc_t(h, &h->g.v2[a], (size_t)gd.Nn);
    }
    h->acur = 0; h->grid_final = true;
    h->acc_m[0] = h->g.m; h->acc_m[1] = nullptr;
    for (int a = 0; a < 3; ++a) { h->acc_mv2[0][a] = h->g.mv2[a]; h->acc_mv2[1][a] = nullptr; }
    for (int a = 0; a < 3; ++a) { h->acc_mv[0][a] = h->g.mv[a]; h->acc_f[0][a] = h->g.f[a]; h->acc_mv[1][a] = h->acc_f[1][a] = nullptr; }
    if (ok && tiled) {
        ok = dev_alloc_t(h, &h->acc_m[1], (size_t)gd.Nn);
        for (int a = 0; a < gd.dim && ok; ++a)
            ok = dev_alloc_t(h, &h->acc_mv[1][a], (size_t)gd.Nn) && dev_alloc_t(h, &h->acc_f[1][a], (size_t)gd.Nn) &&
                 dev_alloc_t(h, &h->acc_mv2[1][a], (size_t)gd.Nn);
    }
    if (ok && tiled && gd.acc32)
        for (int b = 0; b < 2 && ok; ++b)
            ok = dev_alloc_t(h, &h->acc32_nm[b], 8 * (size_t)gd.Nn) && dev_alloc_t(h, &h->acc32_v2[b], 4 * (size_t)gd.Nn);
    if (ok && sorted)
        ok = dev_alloc_t(h, &h->off[0], (size_t)gd.Nkeys + 1) && dev_alloc_t(h, &h->n_groups, 1) && dev_alloc_t(h, &h->n_items, 1);
    if (ok && tiled) {
        unsigned char *st = nullptr;
        ok = dev_alloc_t(h, &h->n_groups_alt, 1) && dev_alloc_t(h, &h->n_items_alt, 1) && dev_alloc_t(h, &st, cell_map_state_bytes(gd));
        h->map_state = st;
    }
    // the scan's block sums: one int per 4096 scanned elements
    ok = ok && dev_alloc_t(h, &h->count, (size_t)gd.Nkeys + 1) && dev_alloc_t(h, &h->scan_aux, (size_t)gd.Nkeys / 4096 + 8) &&
         dev_alloc_t(h, &h->sc, 1);
    if (gd.has_obstacle && ok) {
        build_obstacle(h, cfg->obstacle_mask, cfg->node_normals);
        ok = dev_alloc_t(h, &h->d_flag, (size_t)gd.Nn);
        for (int a = 0; a < gd.dim && ok; ++a) ok = dev_alloc_t(h, &h->d_normal[a], (size_t)gd.Nn);
    }
    if (!ok) { mpm_destroy(h); return fail(nullptr, MPM_E_OOM, "mpm_create: out of device memory for the grid"); }
    h->cfg.obstacle_mask = nullptr; h->cfg.node_normals = nullptr;

    cudaError_t e = cudaSuccess;
    if (gd.has_obstacle) {
        e = cudaMemcpyAsync(h->d_flag, h->h_flag.data(), (size_t)gd.Nn, cudaMemcpyHostToDevice, h->stream);
        for (int a = 0; a < gd.dim && e == cudaSuccess; ++a)
            e = cudaMemcpyAsync(h->d_normal[a], h->h_normal.data() + (size_t)a * gd.Nn, sizeof(double) * (size_t)gd.Nn,
                                cudaMemcpyHostToDevice, h->stream);
        h->g.flag = h->d_flag;
        for (int a = 0; a < gd.dim; ++a) h->g.normal[a] = h->d_normal[a];
    }
    if (e == cudaSuccess) e = cudaMemsetAsync(h->sc, 0, sizeof(DevScalars), h->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->g.m, 0, sizeof(double) * (size_t)gd.Nn, h->stream);
    for (int a = 0; a < gd.dim && e == cudaSuccess; ++a) {
        double *arrs[6] = { h->g.mv[a], h->g.f[a], h->g.mv2[a], h->g.vbar[a], h->g.acc[a], h->g.v2[a] };
        for (int j = 0; j < 6 && e == cudaSuccess; ++j)
            if (arrs[j]) e = cudaMemsetAsync(arrs[j], 0, sizeof(double) * (size_t)gd.Nn, h->stream);
    }
    if (sorted && e == cudaSuccess) e = cudaMemsetAsync(h->n_groups, 0, sizeof(int), h->stream);
    if (sorted && e == cudaSuccess) e = cudaMemsetAsync(h->n_items, 0, sizeof(int), h->stream);
    for (int b = 0; b < 2 && tiled && gd.acc32 && e == cudaSuccess; ++b) {
        e = cudaMemsetAsync(h->acc32_nm[b], 0, sizeof(float) * 8 * (size_t)gd.Nn, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->acc32_v2[b], 0, sizeof(float) * 4 * (size_t)gd.Nn, h->stream);
    }
    if (tiled && e == cudaSuccess) e = cudaMemsetAsync(h->acc_m[1], 0, sizeof(double) * (size_t)gd.Nn, h->stream);
    for (int a = 0; a < gd.dim && tiled && e == cudaSuccess; ++a) {
        e = cudaMemsetAsync(h->acc_mv[1][a], 0, sizeof(double) * (size_t)gd.Nn, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->acc_f[1][a], 0, sizeof(double) * (size_t)gd.Nn, h->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(h->acc_mv2[1][a], 0, sizeof(double) * (size_t)gd.Nn, h->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess) {
        std::string msg = std::string("mpm_create: ") + cudaGetErrorString(e);
        mpm_destroy(h);
        return fail(nullptr, MPM_E_CUDA, msg);
    }
    *out = h;
    return MPM_OK;
}

void mpm_destroy(mpm_handle *h)
{
    if (!h) return;
    DeviceGuard guard(h->cfg.device);
    drain_spans(h);
    cudaStreamSynchronize(h->stream);
    for (cudaEvent_t e : h->event_pool) cudaEventDestroy(e);
    if (h->side) { cudaStreamSynchronize(h->side); cudaStreamDestroy(h->side); }
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    std::vector<void *> all = h->allocations;
    for (void *p : all) dev_free(h, p);
    delete h;
}

namespace {
int load_impl(mpm_handle *h, int64_t n, const double *const *x, const double *const *v, const double *mass,
              const double *rho, const double *e, const double *q, const int64_t *ids, int ptr_location, bool keep_time);

// id[k] = (int)ids64[k]; out[k] = (double)id[k]
__global__ void k_ids_from_i64(int *__restrict__ id, const long long *__restrict__ ids64, long long n, int *bad)
{
    for (long long k = (long long)blockIdx.x * 256 + threadIdx.x; k < n; k += (long long)gridDim.x * 256) {
        const long long v = ids64[k];
        if (v < 0 || v >= (1ll << 31)) atomicOr(bad, 1);
        id[k] = (int)v;
    }
}
__global__ void k_ids_to_double(const int *__restrict__ id, double *__restrict__ out, long long n)
{
    for (long long k = (long long)blockIdx.x * 256 + threadIdx.x; k < n; k += (long long)gridDim.x * 256) out[k] = (double)id[k];
}
}

int mpm_load_particles(mpm_handle *h, int64_t n, const double *const *x, const double *const *v, const double *mass,
                       const double *rho, const double *e, const double *q, int ptr_location)
{
    if (!h) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    return load_impl(h, n, x, v, mass, rho, e, q, nullptr, ptr_location, false);
}

int mpm_load_particles_ex(mpm_handle *h, int64_t n, const double *const *x, const double *const *v, const double *mass,
                          const double *rho, const double *e, const double *q, const int64_t *ids, int ptr_location, int flags)
{
    if (!h) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (flags & ~MPM_LOAD_KEEP_TIME) return fail(h, MPM_E_ARG, "mpm_load_particles_ex: unknown flag");
    const bool keep = (flags & MPM_LOAD_KEEP_TIME) != 0;
    if (keep && !h->pbuf[0].m) return fail(h, MPM_E_STATE, "mpm_load_particles_ex: MPM_LOAD_KEEP_TIME needs a loaded particle set");
    return load_impl(h, n, x, v, mass, rho, e, q, ids, ptr_location, keep);
}

namespace {
int load_impl(mpm_handle *h, int64_t n, const double *const *x, const double *const *v, const double *mass,
              const double *rho, const double *e, const double *q, const int64_t *ids, int ptr_location, bool keep_time)
{
    if (n < 0 || n >= (1ll << 31) - 1 || !x || !v || !mass || !rho || !e)
        return fail(h, MPM_E_ARG, "mpm_load_particles: bad argument");
    if (ptr_location != MPM_HOST && ptr_location != MPM_DEVICE) return fail(h, MPM_E_ARG, "mpm_load_particles: bad ptr_location");
    for (int a = 0; a < h->gd.dim; ++a)
        if (!x[a] || !v[a]) return fail(h, MPM_E_ARG, "mpm_load_particles: null component pointer");
    if (n != h->cap || !h->pbuf[0].m) {
        int rc = alloc_particles(h, n);
        if (rc != MPM_OK) return rc;
    }
    h->n = n; h->cur = 0;
    PArr &p = h->pbuf[0];
    int rc = MPM_OK;
    for (int a = 0; a < h->gd.dim && rc == MPM_OK; ++a) {
        rc = copy_in(h, p.x[a], x[a], n, ptr_location);
        if (rc == MPM_OK) rc = copy_in(h, p.v[a], v[a], n, ptr_location);
    }
    if (rc == MPM_OK) rc = copy_in(h, p.m, mass, n, ptr_location);
    if (rc == MPM_OK) rc = copy_in(h, p.rho, rho, n, ptr_location);
    if (rc == MPM_OK) rc = copy_in(h, p.e, e, n, ptr_location);
    if (rc != MPM_OK) return rc;
    if (q) { rc = copy_in(h, p.q, q, n, ptr_location); if (rc != MPM_OK) return rc; }
    else MPM_CUDA(h, cudaMemsetAsync(p.q, 0, sizeof(double) * (size_t)(n > 0 ? n : 1), h->stream));
    h->gd.uniform_mass = 0;
    h->gd.um = 0.0;
    if (h->variant == MPM_VARIANT_TILED && n > 0) {
        // equal particle masses (configs 4 and 5; with an inflow face the recycled mass must be the same too): the sweeps
        // then neither read nor write the mass array -- 24 B per particle and step less
        struct { int differs; int pad; double first; } probe = { 0, 0, 0.0 };
        MPM_CUDA(h, cudaMemsetAsync(h->n_items_alt, 0, sizeof(int), h->stream));      // free until the first step
        launch_mass_differs(p.m, n, h->n_items_alt, h->stream);
        MPM_CUDA(h, cudaMemcpyAsync(&probe.differs, h->n_items_alt, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        MPM_CUDA(h, cudaMemcpyAsync(&probe.first, p.m, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
        MPM_CUDA(h, cudaStreamSynchronize(h->stream));
        const bool inflow_ok = h->gd.in_axis < 0 || h->gd.inflow_mass == probe.first;
        if (!probe.differs && inflow_ok) { h->gd.uniform_mass = 1; h->gd.um = probe.first; }
        h->launches += 1;
    }
    if (ids && !h->gd.track_ids) return fail(h, MPM_E_ARG, "mpm_load_particles_ex: created with MPM_IDS_NONE: no caller-chosen ids");
    h->external_ids = ids != nullptr;
    if (ids && n > 0) {      // caller-chosen persistent ids: staged in the (free) destination-record array, narrowed to 32 bits
        if (!h->dest) return fail(h, MPM_E_STATE, "mpm_load_particles_ex: caller-chosen ids are offered by the TILED family");
        long long *stage = reinterpret_cast<long long *>(h->dest);
        MPM_CUDA(h, cudaMemcpyAsync(stage, ids, sizeof(long long) * (size_t)n,
                                    ptr_location == MPM_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, h->stream));
        int bad = 0;
        MPM_CUDA(h, cudaMemsetAsync(h->n_items_alt, 0, sizeof(int), h->stream));
        k_ids_from_i64<<<148 * 4, 256, 0, h->stream>>>(p.id, stage, n, h->n_items_alt);
        MPM_CUDA(h, cudaMemcpyAsync(&bad, h->n_items_alt, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        MPM_CUDA(h, cudaStreamSynchronize(h->stream));
        if (bad) return fail(h, MPM_E_ARG, "mpm_load_particles_ex: ids must lie in [0, 2^31)");
    } else launch_iota(p.id, n, h->stream);
    if (h->variant == MPM_VARIANT_TILED && n == 0) {
        // an empty slab still takes part in the halo exchanges: its accumulators must read zero
        h->acur = 0;
        h->grid_final = false;
        const GArr g0 = tiled_acc(h, 0);
        clear_p2g1(h, g0, h->stream);
        clear_p2g2(h, g0, h->stream);
    }
    if (!keep_time) {
        MPM_CUDA(h, cudaMemsetAsync(h->sc, 0, sizeof(DevScalars), h->stream));
        launch_initial_cfl(h->gd, p, h->sc, n, h->stream);
        h->steps_done = 0;
    }
    h->launches += 3;
    if ((h->cfg.sort_every > 0 || h->variant != MPM_VARIANT_ATOMIC) && n > 0) reorder(h);
    if (h->gd.uniform_mass) {      // every slot of both buffers holds the mass: nothing moves it any more
        launch_fill(h->pbuf[0].m, h->slots, h->gd.um, h->stream);
        launch_fill(h->pbuf[1].m, h->slots, h->gd.um, h->stream);
        h->launches += 2;
    }
    MPM_CUDA(h, cudaGetLastError());
    if (ptr_location == MPM_HOST) MPM_CUDA(h, cudaStreamSynchronize(h->stream));   // caller may reuse its buffers
    return MPM_OK;
}
}  // namespace

namespace {
__global__ void k_set_mode(DevScalars *sc, double dt_fixed, double alpha)
{
    sc->dt_fixed = dt_fixed;
    sc->alpha = alpha;
}
}  // namespace

int mpm_step(mpm_handle *h, double dt, double cfl, int32_t nsteps, double *dt_last)
{
    if (!h) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (!h->pbuf[0].m) return fail(h, MPM_E_STATE, "mpm_step: no particles loaded");
    if (nsteps < 0 || (!(dt > 0.0) && !(cfl > 0.0))) return fail(h, MPM_E_ARG, "mpm_step: need nsteps >= 0 and dt > 0 or cfl > 0");
    const GridDesc &gd = h->gd;
    cudaStream_t s = h->stream;
    k_set_mode<<<1, 1, 0, s>>>(h->sc, dt > 0.0 ? dt : 0.0, cfl);
    h->launches += 1;
    for (int it = 0; it < nsteps; ++it) {
        if (h->variant != MPM_VARIANT_ATOMIC) {
            if (h->n > 0) step_tiled(h, it == nsteps - 1);
            else {
                launch_begin_step(h->sc, gd.h, false, s);
                launch_grid_clear(gd, h->g, s);
                if (gd.acc32) clear_p2g1(h, tiled_acc(h, 0), s);
                launch_end_step(h->sc, gd.h, s);
                h->launches += 2;
            }
            h->steps_done += 1;
            continue;
        }
        const PArr &p = h->pbuf[h->cur];
        { Timed t(h, MPM_K_MISC); launch_begin_step(h->sc, gd.h, h->n > 0, s); launch_grid_clear(gd, h->g, s); }   // dt (eq. 25/29); l.2
        { Timed t(h, MPM_K_P2G1); launch_p2g1_atomic(gd, p, h->g, h->n, s); }                  // l.3
        { Timed t(h, MPM_K_NODE1); launch_node1(gd, h->g, h->sc, s); }                         // l.4-5
        { Timed t(h, MPM_K_G2P_P2G2); launch_g2p_p2g2_atomic(gd, p, h->g, h->sc, h->n, s); }   // l.6-8
        { Timed t(h, MPM_K_NODE2); launch_node2(gd, h->g, s); }                                // l.9
        { Timed t(h, MPM_K_UPDATE); launch_update_atomic(gd, p, h->g, h->sc, h->n, s); }       // l.10-11, maxima of l.13
        { Timed t(h, MPM_K_MISC); launch_end_step(h->sc, gd.h, s); }                           // l.13-14
        h->launches += 7;
        h->steps_done += 1;
        if (h->cfg.sort_every > 0 && h->steps_done % h->cfg.sort_every == 0) reorder(h);   // l.12
    }
    MPM_CUDA(h, cudaGetLastError());
    if (dt_last) {
        DevScalars host;
        MPM_CUDA(h, cudaMemcpyAsync(&host, h->sc, sizeof(host), cudaMemcpyDeviceToHost, s));
        MPM_CUDA(h, cudaStreamSynchronize(s));
        *dt_last = host.dt;
        if (host.n_nonfinite) return fail(h, MPM_E_NONFINITE, "mpm_step: non-finite particle state encountered");
        if (host.n_bad_dt) return fail(h, MPM_E_NONFINITE, "mpm_step: no positive finite CFL time step (v_max + c_max is zero or not finite)");
    }
    return MPM_OK;
}

int mpm_step_phase(mpm_handle *h, int phase, double dt)
{
    if (!h) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (!h->pbuf[0].m) return fail(h, MPM_E_STATE, "mpm_step_phase: no particles loaded");
    if (h->variant != MPM_VARIANT_TILED) return fail(h, MPM_E_STATE, "mpm_step_phase: the phase interface is offered by the TILED family");
    if (phase == MPM_PHASE_GATHER) {
        if (!(dt > 0.0)) return fail(h, MPM_E_ARG, "mpm_step_phase(GATHER): dt must be > 0 (the caller forms the global CFL step)");
        k_set_mode<<<1, 1, 0, h->stream>>>(h->sc, dt, 0.0);
        h->launches += 1;
        if (h->n > 0) step_tiled_gather(h);
        else {      // an empty slab: nothing to gather, but its mv2 plane is exported next
            launch_begin_step(h->sc, h->gd.h, false, h->stream);
            const GArr gc = tiled_acc(h, h->acur);
            clear_p2g2(h, gc, h->stream);
            h->launches += 1;
        }
    } else if (phase == MPM_PHASE_UPDATE) {
        if (h->n > 0) step_tiled_update(h, true);
        else {
            clear_p2g1(h, tiled_acc(h, h->acur ^ 1), h->stream);
            h->acur ^= 1;
            launch_end_step(h->sc, h->gd.h, h->stream);
            h->launches += 1;
        }
        h->steps_done += 1;
    } else return fail(h, MPM_E_ARG, "mpm_step_phase: unknown phase");
    MPM_CUDA(h, cudaGetLastError());
    return MPM_OK;
}

int mpm_peek(mpm_handle *h, double out[4])
{
    if (!h || !out) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    DevScalars host;
    MPM_CUDA(h, cudaMemcpyAsync(&host, h->sc, sizeof(host), cudaMemcpyDeviceToHost, h->stream));
    MPM_CUDA(h, cudaStreamSynchronize(h->stream));
    out[0] = host.vmax; out[1] = host.cmax; out[2] = (double)host.n_left_slab; out[3] = host.t;
    return MPM_OK;
}

int mpm_halo(mpm_handle *h, int which, int side, int op, double *buf, int ptr_location)
{
    if (!h || !buf) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (h->variant != MPM_VARIANT_TILED || h->gd.acc32) return fail(h, MPM_E_STATE, "mpm_halo: TILED family with fp64 accumulation only");
    if ((which != MPM_HALO_P2G1 && which != MPM_HALO_P2G2) || (side != 0 && side != 1) || (op != MPM_HALO_EXPORT && op != MPM_HALO_ADD) ||
        (ptr_location != MPM_HOST && ptr_location != MPM_DEVICE))
        return fail(h, MPM_E_ARG, "mpm_halo: bad argument");
    const GridDesc &gd = h->gd;
    const int last = gd.dim - 1;
    const long long plane = gd.Nn / gd.nn[last];                              // the last axis is the slowest: a plane is contiguous
    const long long at = side ? (long long)(gd.nn[last] - 1) * plane : 0;
    const GArr g = tiled_acc(h, h->acur);                                       // the set the next GATHER phase reads / has written
    std::vector<double *> ch;
    if (which == MPM_HALO_P2G1) {
        ch.push_back(g.m);
        for (int a = 0; a < gd.dim; ++a) ch.push_back(g.mv[a]);
        for (int a = 0; a < gd.dim; ++a) ch.push_back(g.f[a]);
    } else for (int a = 0; a < gd.dim; ++a) ch.push_back(g.mv2[a]);
    double *stage = nullptr;
    if (op == MPM_HALO_ADD && ptr_location == MPM_HOST) {                       // host data are staged in the inactive particle buffer
        stage = h->pbuf[h->cur ^ 1].x[0];
        if ((long long)ch.size() * plane > h->slots) return fail(h, MPM_E_STATE, "mpm_halo: plane larger than the staging buffer");
        MPM_CUDA(h, cudaMemcpyAsync(stage, buf, sizeof(double) * ch.size() * (size_t)plane, cudaMemcpyHostToDevice, h->stream));
    }
    for (size_t c = 0; c < ch.size(); ++c) {
        double *node = ch[c] + at, *user = buf + c * plane;
        if (op == MPM_HALO_EXPORT) {
            int rc = copy_out(h, user, node, plane, ptr_location);
            if (rc != MPM_OK) return rc;
        } else launch_add_into(node, stage ? stage + c * plane : user, plane, h->stream);
    }
    h->launches += op == MPM_HALO_ADD ? (long long)ch.size() : 0;
    h->grid_final = false;
    MPM_CUDA(h, cudaGetLastError());
    if (ptr_location == MPM_HOST) MPM_CUDA(h, cudaStreamSynchronize(h->stream));
    return MPM_OK;
}

int mpm_read_particles(mpm_handle *h, uint32_t field_mask, double *const *out, int order, int ptr_location)
{
    if (!h || !out) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (!h->pbuf[0].m) return fail(h, MPM_E_STATE, "mpm_read_particles: no particles loaded");
    if (ptr_location != MPM_HOST && ptr_location != MPM_DEVICE) return fail(h, MPM_E_ARG, "mpm_read_particles: bad ptr_location");
    const PArr &p = h->pbuf[h->cur];
    const PArr &scratch = h->pbuf[h->cur ^ 1];   // the inactive buffer is free outside a re-ordering
    const int d = h->gd.dim;
    std::vector<const double *> src;
    std::vector<double *> tmp;
    if (field_mask & MPM_P_X) for (int a = 0; a < d; ++a) { src.push_back(p.x[a]); tmp.push_back(scratch.x[a]); }
    if (field_mask & MPM_P_V) for (int a = 0; a < d; ++a) { src.push_back(p.v[a]); tmp.push_back(scratch.v[a]); }
    if (field_mask & MPM_P_M) { src.push_back(p.m); tmp.push_back(scratch.m); }
    if (field_mask & MPM_P_RHO) { src.push_back(p.rho); tmp.push_back(scratch.rho); }
    if (field_mask & MPM_P_E) { src.push_back(p.e); tmp.push_back(scratch.e); }
    if (field_mask & MPM_P_Q) { src.push_back(p.q); tmp.push_back(scratch.q); }
    if (h->external_ids && order == 0)
        return fail(h, MPM_E_STATE, "mpm_read_particles: caller-chosen ids: read in storage order (order = 1) with MPM_P_ID");
    if (!h->gd.track_ids && (order == 0 || (field_mask & MPM_P_ID)))
        return fail(h, MPM_E_STATE, "mpm_read_particles: created with MPM_IDS_NONE: storage order (order = 1) only, no MPM_P_ID");
    if (field_mask & MPM_P_ID) {      // ids widened to fp64 in a scratch pair of their own (allocated on first use)
        const size_t N = (size_t)(h->slots > 0 ? h->slots : 1);
        if (h->id_wide_slots < (long long)N) {
            dev_free(h, h->id_wide);
            h->id_wide = nullptr;
            if (!dev_alloc_t(h, &h->id_wide, 2 * N)) return fail(h, MPM_E_OOM, "mpm_read_particles: out of device memory");
            h->id_wide_slots = (long long)N;
        }
        k_ids_to_double<<<148 * 4, 256, 0, h->stream>>>(p.id, h->id_wide, (long long)N);
        h->launches += 1;
        src.push_back(h->id_wide);
        tmp.push_back(h->id_wide + N);
    }
    const bool tiled = h->variant == MPM_VARIANT_TILED && h->n > 0;
    const SortedMap map{ h->groups, h->n_groups };
    if (tiled && order != 0) {   // storage order without the unused slots: compact offsets = scan of the per-key counts
        if (!h->coff && !dev_alloc_t(h, &h->coff, (size_t)h->gd.Nkeys + 1)) return fail(h, MPM_E_OOM, "mpm_read_particles: out of device memory");
        launch_exclusive_scan_from(h->count, h->coff, h->gd.Nkeys + 1, h->scan_aux, false, h->stream);
        h->launches += 3;
    }
    for (size_t j = 0; j < src.size(); ++j) {
        if (!out[j]) return fail(h, MPM_E_ARG, "mpm_read_particles: null output pointer");
        const double *from = src[j];
        if (tiled) {
            launch_gather_by_id_groups(src[j], p.id, tmp[j], map, h->max_groups, order == 0 ? nullptr : h->coff, h->off[0], h->stream);
            h->launches += 1;
            from = tmp[j];
        } else if (order == 0) {
            launch_gather_by_id(src[j], p.id, tmp[j], h->n, h->stream);
            h->launches += 1;
            from = tmp[j];
        }
        int rc = copy_out(h, out[j], from, h->n, ptr_location);
        if (rc != MPM_OK) return rc;
    }
    MPM_CUDA(h, cudaStreamSynchronize(h->stream));
    return MPM_OK;
}

int mpm_read_grid(mpm_handle *h, int field, double *out, int ptr_location)
{
    if (!h || !out) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    if (ptr_location != MPM_HOST && ptr_location != MPM_DEVICE) return fail(h, MPM_E_ARG, "mpm_read_grid: bad ptr_location");
    const GridDesc &gd = h->gd;
    const size_t Nn = (size_t)gd.Nn;
    int rc = MPM_OK;
    if (field == MPM_G_RHO_GRID || field == MPM_G_E_GRID) {      // diagnostics of the current particle state (A18), off the hot path
        if (!h->pbuf[0].m) return fail(h, MPM_E_STATE, "mpm_read_grid: no particles loaded");
        if (gd.quadratic) return fail(h, MPM_E_ARG, "mpm_read_grid: RHO_GRID / E_GRID are offered for the Q1 basis");
        double *num = nullptr;
        if (!dev_alloc_t(h, &num, 2 * Nn)) return fail(h, MPM_E_OOM, "mpm_read_grid: out of device memory");
        MPM_CUDA(h, cudaMemsetAsync(num, 0, sizeof(double) * 2 * Nn, h->stream));
        const PArr &p = h->pbuf[h->cur];
        const bool tiled = h->variant == MPM_VARIANT_TILED;
        launch_grid_diagnostic(gd, p, field == MPM_G_RHO_GRID ? p.rho : p.e, num, num + Nn, h->n,
                               SortedMap{ tiled && h->n > 0 ? h->groups : nullptr, h->n_groups }, h->max_groups, h->stream);
        h->launches += 2;
        rc = copy_out(h, out, num, gd.Nn, ptr_location);
        cudaError_t e = cudaStreamSynchronize(h->stream);
        dev_free(h, num);
        if (rc != MPM_OK) return rc;
        MPM_CUDA(h, e);
        return MPM_OK;
    }
    // TILED: the last completed step used the accumulator set that is no longer current
    GArr gl = (h->variant == MPM_VARIANT_TILED) ? tiled_acc(h, h->steps_done > 0 ? h->acur ^ 1 : h->acur) : h->g;
    if (gd.acc32) {
        // fp32 accumulators: widen the last step's sums into fp64 copies and replay the node conditions there
        if (!h->rg_m) {
            bool ok = dev_alloc_t(h, &h->rg_m, Nn);
            for (int a = 0; a < gd.dim && ok; ++a)
                ok = dev_alloc_t(h, &h->rg_mv[a], Nn) && dev_alloc_t(h, &h->rg_f[a], Nn) && dev_alloc_t(h, &h->rg_mv2[a], Nn);
            if (!ok) return fail(h, MPM_E_OOM, "mpm_read_grid: out of device memory");
            h->grid_final = false;
        }
        GArr gw = gl;
        gw.m = h->rg_m;
        for (int a = 0; a < gd.dim; ++a) { gw.mv[a] = h->rg_mv[a]; gw.f[a] = h->rg_f[a]; gw.mv2[a] = h->rg_mv2[a]; }
        if (!h->grid_final) {
            launch_widen(gd, gl, gw, h->stream);      // node-major fp32 -> component-major fp64
            if (h->steps_done > 0) { launch_node1(gd, gw, h->sc, h->stream, false); launch_node2(gd, gw, h->stream); }
            h->grid_final = true;
            h->launches += 3;
        }
        gl = gw;
    } else if (h->variant == MPM_VARIANT_TILED && !h->grid_final && h->steps_done > 0) {
        // the step left the raw sums; l.4-5 and l.9 are replayed in place with the node kernels (dt of that step is
        // still in the device scalars).  That accumulator set is cleared before it is used again.
        launch_node1(gd, gl, h->sc, h->stream, false);
        launch_node2(gd, gl, h->stream);
        h->grid_final = true;
        h->launches += 2;
    }
    switch (field) {
    case MPM_G_MASS: rc = copy_out(h, out, gl.m, gd.Nn, ptr_location); break;
    case MPM_G_MOMENTUM: for (int a = 0; a < gd.dim && rc == MPM_OK; ++a) rc = copy_out(h, out + a * Nn, gl.mv[a], gd.Nn, ptr_location); break;
    case MPM_G_FORCE: for (int a = 0; a < gd.dim && rc == MPM_OK; ++a) rc = copy_out(h, out + a * Nn, gl.f[a], gd.Nn, ptr_location); break;
    case MPM_G_MOMENTUM2: for (int a = 0; a < gd.dim && rc == MPM_OK; ++a) rc = copy_out(h, out + a * Nn, gl.mv2[a], gd.Nn, ptr_location); break;
    case MPM_G_NORMAL:
    case MPM_G_FLAG: {
        const int nc = field == MPM_G_NORMAL ? gd.dim : 1;
        std::vector<double> host(Nn * nc, 0.0);
        if (gd.has_obstacle) {
            if (field == MPM_G_NORMAL) host = h->h_normal;
            else for (size_t i = 0; i < Nn; ++i) host[i] = h->h_flag[i] ? 1.0 : 0.0;
        }
        if (ptr_location == MPM_HOST) std::memcpy(out, host.data(), sizeof(double) * host.size());
        else {
            MPM_CUDA(h, cudaMemcpyAsync(out, host.data(), sizeof(double) * host.size(), cudaMemcpyHostToDevice, h->stream));
            MPM_CUDA(h, cudaStreamSynchronize(h->stream));
        }
        break;
    }
    default: return fail(h, MPM_E_ARG, "mpm_read_grid: unknown field");
    }
    if (rc != MPM_OK) return rc;
    MPM_CUDA(h, cudaStreamSynchronize(h->stream));
    return MPM_OK;
}

int mpm_get_stats(mpm_handle *h, mpm_stats *out)
{
    if (!h || !out) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    std::memset(out, 0, sizeof(*out));
    DevScalars host;
    if (h->pbuf[0].m) {
        if (h->variant == MPM_VARIANT_TILED && h->n > 0)
            launch_stats_reduce_groups(h->gd, h->pbuf[h->cur], h->sc, SortedMap{ h->groups, h->n_groups }, h->max_groups, h->stream);
        else
            launch_stats_reduce(h->gd, h->pbuf[h->cur], h->sc, h->n, h->stream);
        h->launches += 2;
    }
    MPM_CUDA(h, cudaMemcpyAsync(&host, h->sc, sizeof(host), cudaMemcpyDeviceToHost, h->stream));
    MPM_CUDA(h, cudaStreamSynchronize(h->stream));
    out->t = host.t; out->dt_last = host.dt; out->dt_next = host.dt_next; out->step = host.step;
    out->vmax = host.vmax; out->cmax = host.cmax;
    out->n_recycled = (int64_t)host.n_recycled; out->n_clamped = (int64_t)host.n_clamped;
    out->n_negjac = (int64_t)host.n_negjac; out->n_nonfinite = (int64_t)host.n_nonfinite;
    out->n_cell_changes = (int64_t)host.n_cell_changes; out->n_out_of_cell = (int64_t)host.n_out_of_cell;
    out->n_bad_dt = (int64_t)host.n_bad_dt; out->n_left_slab = (int64_t)host.n_left_slab;
    out->sum_mass = host.sum_mass; out->sum_energy = host.sum_energy;
    for (int a = 0; a < 3; ++a) { out->sum_momentum[a] = host.sum_mom[a]; out->nn[a] = h->gd.nn[a]; }
    out->num_particles = h->n; out->num_nodes = h->gd.Nn;
    out->variant = h->variant; out->launches = h->launches;
    drain_spans(h);
    for (int k = 0; k < MPM_K_COUNT; ++k) { out->kernel_ms[k] = h->kernel_ms[k]; out->kernel_calls[k] = h->kernel_calls[k]; }
    return MPM_OK;
}

int mpm_set_profiling(mpm_handle *h, int on)
{
    if (!h) return MPM_E_ARG;
    DeviceGuard guard(h->cfg.device);
    drain_spans(h);
    if (on) for (int k = 0; k < MPM_K_COUNT; ++k) { h->kernel_ms[k] = 0.0; h->kernel_calls[k] = 0; }
    h->profiling = on != 0;
    return MPM_OK;
}

}  // extern "C"
