/*
 * mpm_oracle.c -- CPU ORACLE (test infrastructure, NOT the product; see mpm_oracle.h).
 *
 * One function per line of Algorithm 1, written in the order and
 * notation of Section 3.  fp64 throughout.  Single
 * thread, particles visited in index order, no tiling / fusion / sorting ("optional
 * re-ordering", must not change results so the oracle has none).
 *
 * Readings of silent / ambiguous points are tagged (A#) and listed in DESIGN.md.
 */
#include "mpm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

struct oracle_s {
    oracle_config cfg;
    int d;
    int nc[3];          /* cells per axis (1 on unused axes) */
    int nn[3];          /* nodes per axis: n (periodic) or n+1 (A11) */
    int per[3];         /* axis periodic? */
    double h, inv_h;    /* A4, A19 */
    double L[3];        /* domain lengths */
    long long Nn, Nc;
    unsigned char *mask;     /* [Nc] or NULL */
    unsigned char *obst;     /* [Nn] node flag: 1 = obstacle node (A7) */
    double *normal;          /* [d][Nn] */
    /* grid fields */
    double *m, *mv, *f, *mv2; /* m[Nn]; mv,f,mv2 [d][Nn] */
    /* particles, SoA */
    long long Np;
    double *X, *V, *M, *rho, *E, *Q;   /* X,V [d][Np] */
    double *Vbar, *A, *D;              /* transients of the step */
    long long *id;
    /* time */
    oracle_stats st;
};

/* ---------------------------------------------------------------- helpers */

static long long node_index(const oracle_t *o, const int i[3])
{
    return (long long)i[0] + (long long)o->nn[0] * ((long long)i[1] + (long long)o->nn[1] * (long long)i[2]);
}

/* Q1 hat-function data of one particle: cell c, 1D weights w[a][0..1], 1D slopes g[a][0..1].
 * PAPER.md:254 (Q1 basis on a Cartesian tensor grid); A6 (clamp cell at the upper face);
 * A19 (xi = X*(1/h) - c). */
static void particle_cell(const oracle_t *o, const double *X, long long stride, int c[3],
                          double w[3][2], double g[3][2])
{
    for (int a = 0; a < 3; ++a) {
        c[a] = 0; w[a][0] = 1.0; w[a][1] = 0.0; g[a][0] = 0.0; g[a][1] = 0.0;
    }
    for (int a = 0; a < o->d; ++a) {
        double s = X[a * stride] * o->inv_h;
        int ci = (int)floor(s);
        if (ci < 0) ci = 0;
        if (ci > o->nc[a] - 1) ci = o->nc[a] - 1;
        double xi = s - (double)ci;
        c[a] = ci;
        w[a][0] = 1.0 - xi;
        w[a][1] = xi;
        g[a][0] = -o->inv_h;
        g[a][1] = +o->inv_h;
    }
}

/* global node of corner b of cell c, periodic wrap node n == node 0 (A11) */
static long long corner_node(const oracle_t *o, const int c[3], const int b[3])
{
    int i[3];
    for (int a = 0; a < 3; ++a) {
        i[a] = c[a] + b[a];
        if (o->per[a] && i[a] == o->nc[a]) i[a] = 0;
    }
    return node_index(o, i);
}

/* phi and grad phi of corner b: phi = prod_a w_a(b_a); d_a phi = g_a(b_a) prod_{a'!=a} w_a'(b_a') */
static void corner_weights(const oracle_t *o, double w[3][2], double g[3][2], const int b[3],
                           double *phi, double grad[3])
{
    double p = 1.0;
    for (int a = 0; a < o->d; ++a) p *= w[a][b[a]];
    *phi = p;
    for (int a = 0; a < 3; ++a) grad[a] = 0.0;
    for (int a = 0; a < o->d; ++a) {
        double q = g[a][b[a]];
        for (int a2 = 0; a2 < o->d; ++a2)
            if (a2 != a) q *= w[a2][b[a2]];
        grad[a] = q;
    }
}

void oracle_shape(const oracle_t *o, const double *X, long long *node, double *phi, double *grad)
{
    int c[3]; double w[3][2], g[3][2];
    particle_cell(o, X, 1, c, w, g);
    int nb = 1 << o->d;
    for (int ib = 0; ib < nb; ++ib) {
        int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
        double gr[3];
        node[ib] = corner_node(o, c, b);
        corner_weights(o, w, g, b, &phi[ib], gr);
        for (int a = 0; a < o->d; ++a) grad[ib * o->d + a] = gr[a];
    }
}

/* ---------------------------------------------------------------- quadratic B-spline basis (A20)
 * PAPER.md:721, :735-739 name quadratic B-splines [60, 19] as the next basis.  The standard MPM quadratic B-spline centred on
 * the grid nodes:  N(u) = 3/4 - u^2 (|u| < 1/2),  (3/2 - |u|)^2 / 2 (1/2 <= |u| < 3/2),  0 otherwise,  u = (x - x_i)/h;
 * phi_i(X) = prod_a N((X_a - x_{i,a})/h).  A particle sees 3 nodes per axis: b, b+1, b+2 with b = floor(X/h - 1/2);
 * with f = X/h - b in [1/2, 3/2):  w(0) = (3/2 - f)^2/2,  w(1) = 3/4 - (f - 1)^2,  w(2) = (f - 1/2)^2/2  and slopes
 * dN/dx:  -(3/2 - f)/h,  -2 (f - 1)/h,  (f - 1/2)/h.  Periodic axes only: node index modulo n. */
typedef struct {
    int n;                 /* 3^d */
    long long node[27];
    double phi[27];
    double grad[27][3];
} support_t;

static void support_quadratic(const oracle_t *o, const double *X, long long stride, support_t *s)
{
    int base[3] = { 0, 0, 0 }, ns[3] = { 1, 1, 1 };
    double w[3][3] = { { 1, 0, 0 }, { 1, 0, 0 }, { 1, 0, 0 } }, g[3][3] = { { 0, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
    for (int a = 0; a < o->d; ++a) {
        double sx = X[a * stride] * o->inv_h;
        int b = (int)floor(sx - 0.5);
        double f = sx - (double)b;
        base[a] = b; ns[a] = 3;
        w[a][0] = 0.5 * (1.5 - f) * (1.5 - f);
        w[a][1] = 0.75 - (f - 1.0) * (f - 1.0);
        w[a][2] = 0.5 * (f - 0.5) * (f - 0.5);
        g[a][0] = -(1.5 - f) * o->inv_h;
        g[a][1] = -2.0 * (f - 1.0) * o->inv_h;
        g[a][2] = (f - 0.5) * o->inv_h;
    }
    int q = 0;
    for (int iz = 0; iz < ns[2]; ++iz)
        for (int iy = 0; iy < ns[1]; ++iy)
            for (int ix = 0; ix < ns[0]; ++ix, ++q) {
                int j[3] = { ix, iy, iz }, i[3] = { 0, 0, 0 };
                for (int a = 0; a < o->d; ++a) {
                    int t = (base[a] + j[a]) % o->nc[a];
                    i[a] = t < 0 ? t + o->nc[a] : t;
                }
                s->node[q] = node_index(o, i);
                double phi = 1.0;
                for (int a = 0; a < o->d; ++a) phi *= w[a][j[a]];
                s->phi[q] = phi;
                for (int a = 0; a < 3; ++a) s->grad[q][a] = 0.0;
                for (int a = 0; a < o->d; ++a) {
                    double t = g[a][j[a]];
                    for (int a2 = 0; a2 < o->d; ++a2)
                        if (a2 != a) t *= w[a2][j[a2]];
                    s->grad[q][a] = t;
                }
            }
    s->n = q;
}

void oracle_shape_quadratic(const oracle_t *o, const double *X, long long *node, double *phi, double *grad)
{
    support_t s;
    support_quadratic(o, X, 1, &s);
    for (int q = 0; q < s.n; ++q) {
        node[q] = s.node[q];
        phi[q] = s.phi[q];
        for (int a = 0; a < o->d; ++a) grad[q * o->d + a] = s.grad[q][a];
    }
}

/* counter-based uniform in [0,1): the splitmix64 finaliser (Steele, Lea & Flood 2014) applied to
 * a counter built from (seed, id, step, j).  Restated independently in the CUDA path (A8). */
static unsigned long long mix64(unsigned long long z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
unsigned long long oracle_mix64(unsigned long long z) { return mix64(z); }
double oracle_recycle_uniform(unsigned long long seed, long long id, long long step, int j);
static double recycle_uniform(unsigned long long seed, long long id, long long step, int j)
{
    unsigned long long z = mix64(seed);
    z = mix64(z ^ (unsigned long long)id);
    z = mix64(z ^ (unsigned long long)step);
    z = mix64(z ^ (unsigned long long)j);
    return (double)(z >> 11) * (1.0 / 9007199254740992.0); /* 2^-53 */
}

double oracle_recycle_uniform(unsigned long long seed, long long id, long long step, int j)
{
    return recycle_uniform(seed, id, step, j);
}

/* ---------------------------------------------------------------- obstacle setup (A7) */

static int cell_masked(const oracle_t *o, int cx, int cy, int cz, int *inside)
{
    int c[3] = { cx, cy, cz };
    for (int a = 0; a < o->d; ++a) {
        if (o->per[a]) { c[a] %= o->nc[a]; if (c[a] < 0) c[a] += o->nc[a]; }
        else if (c[a] < 0 || c[a] >= o->nc[a]) { *inside = 0; return 0; }
    }
    *inside = 1;
    return o->mask[(long long)c[0] + (long long)o->nc[0] * ((long long)c[1] + (long long)o->nc[1] * c[2])] != 0;
}

#define ORC_SD_WINDOW 4
/* sd(node) = dist(nearest masked-cell centre) - dist(nearest unmasked-cell centre), both searched in a
 * window of +-ORC_SD_WINDOW cells; a class not found in the window counts as (W+1) h away.  Positive
 * in the fluid, so grad sd points out of the obstacle (reading A7). */
static double sd_node(const oracle_t *o, const int i[3])
{
    const int W = ORC_SD_WINDOW;
    double far = (double)(W + 1) * o->h;
    double best_m = far, best_f = far;
    int lo[3] = { 0, 0, 0 }, hi[3] = { 0, 0, 0 };
    for (int a = 0; a < o->d; ++a) { lo[a] = i[a] - W; hi[a] = i[a] + W - 1; }
    for (int cz = lo[2]; cz <= hi[2]; ++cz)
        for (int cy = lo[1]; cy <= hi[1]; ++cy)
            for (int cx = lo[0]; cx <= hi[0]; ++cx) {
                int inside;
                int mk = cell_masked(o, cx, cy, cz, &inside);
                if (!inside) continue;
                int c[3] = { cx, cy, cz };
                double r2 = 0.0;
                for (int a = 0; a < o->d; ++a) {
                    double dxa = ((double)c[a] + 0.5 - (double)i[a]) * o->h;
                    r2 += dxa * dxa;
                }
                double r = sqrt(r2);
                if (mk) { if (r < best_m) best_m = r; }
                else    { if (r < best_f) best_f = r; }
            }
    return best_m - best_f;
}

static void setup_obstacle(oracle_t *o)
{
    const oracle_config *cfg = &o->cfg;
    o->obst = (unsigned char *)calloc((size_t)o->Nn, 1);
    o->normal = (double *)calloc((size_t)(o->d * o->Nn), sizeof(double));
    if (!o->mask) return;
    /* node flagged if ANY adjacent cell is masked (A7) */
    for (int iz = 0; iz < o->nn[2]; ++iz)
        for (int iy = 0; iy < o->nn[1]; ++iy)
            for (int ix = 0; ix < o->nn[0]; ++ix) {
                int i[3] = { ix, iy, iz };
                int flagged = 0;
                int nadj = 1 << o->d;
                for (int ib = 0; ib < nadj && !flagged; ++ib) {
                    int c[3] = { ix - (ib & 1), iy - ((ib >> 1) & 1), iz - ((ib >> 2) & 1) };
                    if (o->d < 3) c[2] = 0;
                    int inside;
                    if (cell_masked(o, c[0], c[1], c[2], &inside)) flagged = 1;
                }
                o->obst[node_index(o, i)] = (unsigned char)flagged;
            }
    if (cfg->node_normals) {
        memcpy(o->normal, cfg->node_normals, sizeof(double) * (size_t)(o->d * o->Nn));
        return;
    }
    /* n = grad sd / |grad sd| by central differences of sd over +-1 node (eq. 24, A7) */
    for (int iz = 0; iz < o->nn[2]; ++iz)
        for (int iy = 0; iy < o->nn[1]; ++iy)
            for (int ix = 0; ix < o->nn[0]; ++ix) {
                int i[3] = { ix, iy, iz };
                long long I = node_index(o, i);
                if (!o->obst[I]) continue;
                double gsd[3] = { 0, 0, 0 }, nrm = 0.0;
                for (int a = 0; a < o->d; ++a) {
                    int ip[3] = { ix, iy, iz }, im[3] = { ix, iy, iz };
                    ip[a] += 1; im[a] -= 1;
                    gsd[a] = (sd_node(o, ip) - sd_node(o, im)) / (2.0 * o->h);
                    nrm += gsd[a] * gsd[a];
                }
                nrm = sqrt(nrm);
                for (int a = 0; a < o->d; ++a)
                    o->normal[a * o->Nn + I] = (nrm > 0.0) ? gsd[a] / nrm : 0.0;
            }
}

/* ---------------------------------------------------------------- create / destroy / load */

oracle_t *oracle_create(const oracle_config *cfg)
{
    if (!cfg || (cfg->dim != 2 && cfg->dim != 3) || !(cfg->dx > 0.0) || !(cfg->gamma > 1.0)) return NULL;
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    o->cfg = *cfg;
    o->d = cfg->dim;
    o->h = cfg->dx;
    o->inv_h = 1.0 / cfg->dx;
    o->Nn = 1; o->Nc = 1;
    for (int a = 0; a < 3; ++a) {
        if (a < o->d) {
            if (cfg->n[a] < 1) { free(o); return NULL; }
            int p0 = cfg->bc[a][0] == ORC_BC_PERIODIC, p1 = cfg->bc[a][1] == ORC_BC_PERIODIC;
            if (p0 != p1) { free(o); return NULL; }
            o->nc[a] = cfg->n[a];
            o->per[a] = p0;
            o->nn[a] = p0 ? cfg->n[a] : cfg->n[a] + 1;
            o->L[a] = (double)cfg->n[a] * cfg->dx;
        } else {
            o->nc[a] = 1; o->nn[a] = 1; o->per[a] = 0; o->L[a] = 0.0;
        }
        o->Nn *= o->nn[a];
        o->Nc *= o->nc[a];
    }
    if (cfg->basis != ORC_BASIS_Q1) {      /* A20: quadratic B-splines on fully periodic grids of >= 3 cells per axis */
        int ok = cfg->basis == ORC_BASIS_QUADRATIC && !cfg->obstacle_mask;
        for (int a = 0; a < o->d; ++a) ok = ok && o->per[a] && o->nc[a] >= 3;
        if (!ok) { free(o); return NULL; }
    }
    if (cfg->obstacle_mask) {
        o->mask = (unsigned char *)malloc((size_t)o->Nc);
        memcpy(o->mask, cfg->obstacle_mask, (size_t)o->Nc);
    }
    setup_obstacle(o);
    o->cfg.obstacle_mask = NULL; o->cfg.node_normals = NULL;
    o->m = (double *)calloc((size_t)o->Nn, sizeof(double));
    o->mv = (double *)calloc((size_t)(o->d * o->Nn), sizeof(double));
    o->f = (double *)calloc((size_t)(o->d * o->Nn), sizeof(double));
    o->mv2 = (double *)calloc((size_t)(o->d * o->Nn), sizeof(double));
    return o;
}

static void free_particles(oracle_t *o)
{
    free(o->X); free(o->V); free(o->M); free(o->rho); free(o->E); free(o->Q);
    free(o->Vbar); free(o->A); free(o->D); free(o->id);
    o->X = o->V = o->M = o->rho = o->E = o->Q = o->Vbar = o->A = o->D = NULL; o->id = NULL;
    o->Np = 0;
}

void oracle_destroy(oracle_t *o)
{
    if (!o) return;
    free_particles(o);
    free(o->mask); free(o->obst); free(o->normal);
    free(o->m); free(o->mv); free(o->f); free(o->mv2);
    free(o);
}

long long oracle_num_nodes(const oracle_t *o, int nn[3])
{
    if (nn) for (int a = 0; a < 3; ++a) nn[a] = o->nn[a];
    return o->Nn;
}
long long oracle_num_particles(const oracle_t *o) { return o->Np; }

/* speed of sound of eq. (25)/(29) text: sqrt(gamma p / rho) with p = (gamma-1) rho e (eq. 3) */
static double sound_speed(const oracle_t *o, double rho, double e)
{
    double P = (o->cfg.gamma - 1.0) * rho * e;
    return sqrt(o->cfg.gamma * P / rho);
}

int oracle_load_particles(oracle_t *o, long long n, const double *x, const double *v,
                          const double *mass, const double *rho, const double *e, const double *q)
{
    return oracle_load_particles_ex(o, n, x, v, mass, rho, e, q, NULL, 0);
}

/* ids: persistent ids chosen by the caller (NULL = the load index); keep_time: time, step, maxima and counters survive
 * (a slab of a decomposed domain replacing its particle set, tests/slab_oracle_engine.py) */
int oracle_load_particles_ex(oracle_t *o, long long n, const double *x, const double *v,
                             const double *mass, const double *rho, const double *e, const double *q,
                             const long long *ids, int keep_time)
{
    if (!o || n < 0) return -1;
    free_particles(o);
    o->Np = n;
    size_t N = (size_t)(n > 0 ? n : 1);
    o->X = (double *)calloc(N * o->d, sizeof(double));
    o->V = (double *)calloc(N * o->d, sizeof(double));
    o->Vbar = (double *)calloc(N * o->d, sizeof(double));
    o->A = (double *)calloc(N * o->d, sizeof(double));
    o->M = (double *)calloc(N, sizeof(double));
    o->rho = (double *)calloc(N, sizeof(double));
    o->E = (double *)calloc(N, sizeof(double));
    o->Q = (double *)calloc(N, sizeof(double));
    o->D = (double *)calloc(N, sizeof(double));
    o->id = (long long *)calloc(N, sizeof(long long));
    memcpy(o->X, x, sizeof(double) * (size_t)(n * o->d));
    memcpy(o->V, v, sizeof(double) * (size_t)(n * o->d));
    memcpy(o->M, mass, sizeof(double) * (size_t)n);
    memcpy(o->rho, rho, sizeof(double) * (size_t)n);
    memcpy(o->E, e, sizeof(double) * (size_t)n);
    if (q) memcpy(o->Q, q, sizeof(double) * (size_t)n);
    for (long long k = 0; k < n; ++k) o->id[k] = ids ? ids[k] : k;
    if (keep_time) return 0;
    memset(&o->st, 0, sizeof(o->st));
    /* first CFL reduction from the loaded state, ||V|| only (A13) */
    double vmax = 0.0, cmax = 0.0;
    for (long long k = 0; k < n; ++k) {
        double v2 = 0.0;
        for (int a = 0; a < o->d; ++a) v2 += o->V[a * n + k] * o->V[a * n + k];
        double vn = sqrt(v2), cs = sound_speed(o, o->rho[k], o->E[k]);
        if (vn > vmax) vmax = vn;
        if (cs > cmax) cmax = cs;
    }
    o->st.vmax = vmax; o->st.cmax = cmax;
    return 0;
}

/* ---------------------------------------------------------------- Algorithm 1 */

/* l.2 Grid reset: m = mv = f = 0; flags and normals are static. */
void oracle_grid_reset(oracle_t *o)
{
    memset(o->m, 0, sizeof(double) * (size_t)o->Nn);
    memset(o->mv, 0, sizeof(double) * (size_t)(o->d * o->Nn));
    memset(o->f, 0, sizeof(double) * (size_t)(o->d * o->Nn));
}

/* l.3 Mass, momentum and force P2G (eqs. 13, 14, 16, 18):
 *   m_i += M_k phi_i(X_k);  mv_i += M_k V_k phi_i(X_k);  f_i += (P_k+Q_k) M_k/rho_k grad phi_i(X_k)
 * with P_k = (gamma-1) rho_k E_k (eq. 3, A15). */
void oracle_p2g1(oracle_t *o)
{
    const long long n = o->Np, Nn = o->Nn;
    const int nb = 1 << o->d;
    for (long long k = 0; k < n; ++k) {
        int c[3]; double w[3][2], g[3][2];
        double P = (o->cfg.gamma - 1.0) * o->rho[k] * o->E[k];
        double S = (P + o->Q[k]) * o->M[k] / o->rho[k];
        if (o->cfg.basis == ORC_BASIS_QUADRATIC) {   /* the same three sums over the 3^d nodes of the B-spline support */
            support_t s;
            support_quadratic(o, &o->X[k], n, &s);
            for (int q = 0; q < s.n; ++q) {
                long long i = s.node[q];
                o->m[i] += o->M[k] * s.phi[q];
                for (int a = 0; a < o->d; ++a) {
                    o->mv[a * Nn + i] += o->M[k] * o->V[a * n + k] * s.phi[q];
                    o->f[a * Nn + i] += S * s.grad[q][a];
                }
            }
            continue;
        }
        particle_cell(o, &o->X[k], n, c, w, g);
        for (int ib = 0; ib < nb; ++ib) {
            int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
            double phi, grad[3];
            long long i = corner_node(o, c, b);
            corner_weights(o, w, g, b, &phi, grad);
            o->m[i] += o->M[k] * phi;
            for (int a = 0; a < o->d; ++a) {
                o->mv[a * Nn + i] += o->M[k] * o->V[a * n + k] * phi;
                o->f[a * Nn + i] += S * grad[a];
            }
        }
    }
}

/* Boundary conditions on one vector node field pair.  Order: x faces, y faces, z faces, obstacle
 * (A9, A14).  REFLECT: normal component of mv and f -> 0 (eq. 30).  INFLOW: mv = m v_in,
 * f = 0.  OUTFLOW: normal component of f -> 0 (A10).  Obstacle: eqs. (21),(22), which are algebraically
 * w - min(w.n, 0) n.  `f` may be NULL (second application). */
static void apply_bc(oracle_t *o, double *mv, double *f)
{
    const long long Nn = o->Nn;
    for (int iz = 0; iz < o->nn[2]; ++iz)
        for (int iy = 0; iy < o->nn[1]; ++iy)
            for (int ix = 0; ix < o->nn[0]; ++ix) {
                int i[3] = { ix, iy, iz };
                long long I = node_index(o, i);
                for (int a = 0; a < o->d; ++a) {
                    if (o->per[a]) continue;
                    for (int s = 0; s < 2; ++s) {
                        int on_face = (s == 0) ? (i[a] == 0) : (i[a] == o->nn[a] - 1);
                        if (!on_face) continue;
                        int bc = o->cfg.bc[a][s];
                        if (bc == ORC_BC_REFLECT) {
                            mv[a * Nn + I] = 0.0;
                            if (f) f[a * Nn + I] = 0.0;
                        } else if (bc == ORC_BC_INFLOW) {
                            for (int a2 = 0; a2 < o->d; ++a2) {
                                mv[a2 * Nn + I] = o->m[I] * o->cfg.inflow_v[a2];
                                if (f) f[a2 * Nn + I] = 0.0;
                            }
                        } else if (bc == ORC_BC_OUTFLOW) {
                            if (f) f[a * Nn + I] = 0.0;
                        }
                    }
                }
                if (o->obst[I]) {
                    /* eq. (21): mv' = mv - ((mv.n - |mv.n|)/2) n */
                    double dot = 0.0;
                    for (int a = 0; a < o->d; ++a) dot += mv[a * Nn + I] * o->normal[a * Nn + I];
                    double half = (dot - fabs(dot)) / 2.0;
                    for (int a = 0; a < o->d; ++a) mv[a * Nn + I] -= half * o->normal[a * Nn + I];
                    if (f) { /* eq. (22) */
                        double dotf = 0.0;
                        for (int a = 0; a < o->d; ++a) dotf += f[a * Nn + I] * o->normal[a * Nn + I];
                        double halff = (dotf - fabs(dotf)) / 2.0;
                        for (int a = 0; a < o->d; ++a) f[a * Nn + I] -= halff * o->normal[a * Nn + I];
                    }
                }
            }
}

/* l.4 BC on mv, f and obstacle treatment */
void oracle_grid_bc(oracle_t *o) { apply_bc(o, o->mv, o->f); }

/* l.5 (mv)' = mv + dt f */
void oracle_grid_advance(oracle_t *o, double dt)
{
    for (long long j = 0; j < o->d * o->Nn; ++j) o->mv[j] = o->mv[j] + dt * o->f[j];
}

/* l.6-7 G2P (eq. 17 with theta(x,y)=x/y): Vbar = G2P(mv'/m), A = G2P(f/m);
 * x/m := 0 where m = 0 (A5);  V' = V + dt A; Vbar is NOT used to update V. */
void oracle_g2p_velocity(oracle_t *o, double dt)
{
    const long long n = o->Np, Nn = o->Nn;
    const int nb = 1 << o->d;
    for (long long k = 0; k < n; ++k) {
        int c[3]; double w[3][2], g[3][2];
        double vb[3] = { 0, 0, 0 }, ac[3] = { 0, 0, 0 };
        if (o->cfg.basis == ORC_BASIS_QUADRATIC) {
            support_t s;
            support_quadratic(o, &o->X[k], n, &s);
            for (int q = 0; q < s.n; ++q) {
                long long i = s.node[q];
                double mi = o->m[i];
                for (int a = 0; a < o->d; ++a) {
                    double vel = (mi != 0.0) ? o->mv[a * Nn + i] / mi : 0.0;
                    double acc = (mi != 0.0) ? o->f[a * Nn + i] / mi : 0.0;
                    vb[a] += s.phi[q] * vel;
                    ac[a] += s.phi[q] * acc;
                }
            }
        } else {
        particle_cell(o, &o->X[k], n, c, w, g);
        for (int ib = 0; ib < nb; ++ib) {
            int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
            double phi, grad[3];
            long long i = corner_node(o, c, b);
            corner_weights(o, w, g, b, &phi, grad);
            double mi = o->m[i];
            for (int a = 0; a < o->d; ++a) {
                double vel = (mi != 0.0) ? o->mv[a * Nn + i] / mi : 0.0;
                double acc = (mi != 0.0) ? o->f[a * Nn + i] / mi : 0.0;
                vb[a] += phi * vel;
                ac[a] += phi * acc;
            }
        }
        }
        for (int a = 0; a < o->d; ++a) {
            o->Vbar[a * n + k] = vb[a];
            o->A[a * n + k] = ac[a];
            o->V[a * n + k] = o->V[a * n + k] + dt * ac[a];
        }
    }
}

/* l.8 Momentum P2G: mv2_i = sum_k M_k V'_k phi_i(X_k), same positions */
void oracle_p2g2(oracle_t *o)
{
    const long long n = o->Np, Nn = o->Nn;
    const int nb = 1 << o->d;
    memset(o->mv2, 0, sizeof(double) * (size_t)(o->d * Nn));
    for (long long k = 0; k < n; ++k) {
        int c[3]; double w[3][2], g[3][2];
        if (o->cfg.basis == ORC_BASIS_QUADRATIC) {
            support_t s;
            support_quadratic(o, &o->X[k], n, &s);
            for (int q = 0; q < s.n; ++q)
                for (int a = 0; a < o->d; ++a) o->mv2[a * Nn + s.node[q]] += o->M[k] * o->V[a * n + k] * s.phi[q];
            continue;
        }
        particle_cell(o, &o->X[k], n, c, w, g);
        for (int ib = 0; ib < nb; ++ib) {
            int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
            double phi, grad[3];
            long long i = corner_node(o, c, b);
            corner_weights(o, w, g, b, &phi, grad);
            for (int a = 0; a < o->d; ++a) o->mv2[a * Nn + i] += o->M[k] * o->V[a * n + k] * phi;
        }
    }
}

/* l.9 BC on the updated grid momentum */
void oracle_grid_bc2(oracle_t *o) { apply_bc(o, o->mv2, NULL); }

/* l.10 Particle properties update (eq. 4 at :125; A2, A3):
 *   grad V = G2PD(mv2/m), D = trace;
 *   Q from eq. (4) with the D just gathered and the current (un-primed) rho, P: eqs. (5a),(5b)
 *   use ONE div v for q and for the energy equation, so q is always dissipative (-(q) D >= 0);
 *   E' = E - dt (P+Q)/rho D;  rho' = rho/(1 + dt D);  P' = (gamma-1) rho' E' (implicit, A15).
 *   Q is stored and enters the next step's force. */
void oracle_particle_update(oracle_t *o, double dt)
{
    const long long n = o->Np, Nn = o->Nn;
    const int nb = 1 << o->d;
    const double gam = o->cfg.gamma;
    long long nonfinite = 0;
    for (long long k = 0; k < n; ++k) {
        int c[3]; double w[3][2], g[3][2];
        double D = 0.0;
        if (o->cfg.basis == ORC_BASIS_QUADRATIC) {
            support_t s;
            support_quadratic(o, &o->X[k], n, &s);
            for (int q = 0; q < s.n; ++q) {
                double mi = o->m[s.node[q]];
                for (int a = 0; a < o->d; ++a) {
                    double vel = (mi != 0.0) ? o->mv2[a * Nn + s.node[q]] / mi : 0.0;
                    D += vel * s.grad[q][a];
                }
            }
        } else {
        particle_cell(o, &o->X[k], n, c, w, g);
        for (int ib = 0; ib < nb; ++ib) {
            int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
            double phi, grad[3];
            long long i = corner_node(o, c, b);
            corner_weights(o, w, g, b, &phi, grad);
            double mi = o->m[i];
            for (int a = 0; a < o->d; ++a) {
                double vel = (mi != 0.0) ? o->mv2[a * Nn + i] / mi : 0.0;
                D += vel * grad[a];
            }
        }
        }
        o->D[k] = D;
        double rho = o->rho[k], E = o->E[k];
        double P = (gam - 1.0) * rho * E;
        double Q = 0.0;
        if (D < 0.0) {
            double cs = sqrt(gam * P / rho);
            if (o->cfg.visc_form == ORC_VISC_STANDARD)
                Q = rho * (o->cfg.c0 * o->h * o->h * D * D - o->cfg.c1 * o->h * cs * D);
            else
                Q = o->cfg.c0 * (rho * o->h * D) * (rho * o->h * D) - o->cfg.c1 * o->h * cs * D;
        }
        double En = E + dt * (-(P + Q) / rho) * D;
        double jac = 1.0 + dt * D;
        if (jac <= 0.0) o->st.n_negjac++;
        double rhon = rho / jac;
        double Qn = Q;
        o->E[k] = En; o->rho[k] = rhon; o->Q[k] = Qn;
        if (!isfinite(En) || !isfinite(rhon)) nonfinite++;
    }
    o->st.n_nonfinite = nonfinite;
}

/* l.11 Particles moving X' = X + dt Vbar; periodic wrap (A11); recycling of particles
 * that pass an OUTFLOW face (A8); clamp to the domain on non-periodic axes. */
void oracle_advect(oracle_t *o, double dt)
{
    const long long n = o->Np;
    const oracle_config *cfg = &o->cfg;
    /* the inflow face used for recycling: the first INFLOW face in the order x-lo, x-hi, y-lo, ... */
    int in_axis = -1, in_side = 0;
    for (int a = 0; a < o->d && in_axis < 0; ++a)
        for (int s = 0; s < 2; ++s)
            if (cfg->bc[a][s] == ORC_BC_INFLOW) { in_axis = a; in_side = s; break; }
    for (long long k = 0; k < n; ++k) {
        int recycle = 0;
        double Xn[3] = { 0, 0, 0 };
        for (int a = 0; a < o->d; ++a) {
            double x = o->X[a * n + k] + dt * o->Vbar[a * n + k];
            if (o->per[a]) {
                x = x - o->L[a] * floor(x / o->L[a]);
                if (x >= o->L[a]) x = 0.0; /* rounding guard: keep x in [0, L) */
            } else {
                if (x < 0.0 && cfg->bc[a][0] == ORC_BC_OUTFLOW) recycle = 1;
                if (x > o->L[a] && cfg->bc[a][1] == ORC_BC_OUTFLOW) recycle = 1;
            }
            Xn[a] = x;
        }
        if (recycle && in_axis >= 0) {
            long long id = o->id[k];
            int j = 0;
            double u0 = recycle_uniform(cfg->recycle_seed, id, o->st.step, j++);
            for (int a = 0; a < o->d; ++a) {
                if (a == in_axis) {
                    Xn[a] = (in_side == 0) ? u0 * o->h : o->L[a] - u0 * o->h;
                } else {
                    double u1 = recycle_uniform(cfg->recycle_seed, id, o->st.step, j++);
                    double u2 = recycle_uniform(cfg->recycle_seed, id, o->st.step, j++);
                    /* a slab of a larger domain (last axis): the inflow face is the global one, the cell index slab-local */
                    int slab = cfg->slab_global_n > 0 && a == o->d - 1;
                    int na = slab ? cfg->slab_global_n : o->nc[a];
                    int cell = (int)floor(u1 * (double)na);
                    if (cell > na - 1) cell = na - 1;
                    if (slab) cell -= cfg->slab_offset;
                    Xn[a] = ((double)cell + u2) * o->h;
                }
                o->V[a * n + k] = cfg->inflow_v[a];
            }
            o->rho[k] = cfg->inflow_rho;
            o->E[k] = cfg->inflow_p / ((cfg->gamma - 1.0) * cfg->inflow_rho);
            o->Q[k] = 0.0;
            double vol = 1.0;
            for (int a = 0; a < o->d; ++a) vol *= o->h;
            o->M[k] = cfg->inflow_rho * vol / cfg->ppc_inflow;
            o->st.n_recycled++;
        }
        for (int a = 0; a < o->d; ++a) {
            if (!o->per[a]) {   /* an OPEN face is an interface to a neighbouring slab: the particle leaves, unclamped */
                if (Xn[a] < 0.0 && cfg->bc[a][0] != ORC_BC_OPEN) { Xn[a] = 0.0; o->st.n_clamped++; }
                if (Xn[a] > o->L[a] && cfg->bc[a][1] != ORC_BC_OPEN) { Xn[a] = o->L[a]; o->st.n_clamped++; }
            }
            o->X[a * n + k] = Xn[a];
        }
    }
}

/* l.13 CFL (eq. 25 in the enforced form eq. 29; A12, A13):
 *   vmax = max_k max(|V'_k|, |Vbar_k|), cmax = max_k sqrt(gamma P'_k/rho'_k), dt_next = alpha h/(vmax+cmax).
 * Called BEFORE advection/recycling changes V, rho, E (so it sees V', Vbar, rho', E' of this step). */
void oracle_cfl(oracle_t *o, double alpha)
{
    const long long n = o->Np;
    double vmax = 0.0, cmax = 0.0;
    for (long long k = 0; k < n; ++k) {
        double v2 = 0.0, vb2 = 0.0;
        for (int a = 0; a < o->d; ++a) {
            v2 += o->V[a * n + k] * o->V[a * n + k];
            vb2 += o->Vbar[a * n + k] * o->Vbar[a * n + k];
        }
        double vn = sqrt(v2), vbn = sqrt(vb2);
        double cs = sound_speed(o, o->rho[k], o->E[k]);
        if (vn > vmax) vmax = vn;
        if (vbn > vmax) vmax = vbn;
        if (cs > cmax) cmax = cs;
    }
    o->st.vmax = vmax; o->st.cmax = cmax;
    o->st.dt_next = alpha * o->h / (vmax + cmax);
}

/* l.13 time advance for a caller that drives Algorithm 1 line by line (oracle_step does the same inline) */
void oracle_advance_time(oracle_t *o, double dt)
{
    o->st.t += dt;
    o->st.dt_last = dt;
    o->st.step += 1;
}

int oracle_step(oracle_t *o, double dt_fixed, double alpha, int nsteps, double *dt_last)
{
    if (!o) return -1;
    for (int s = 0; s < nsteps; ++s) {
        double dt = (dt_fixed > 0.0) ? dt_fixed : alpha * o->h / (o->st.vmax + o->st.cmax);
        oracle_grid_reset(o);            /* l.2  */
        oracle_p2g1(o);                  /* l.3  */
        oracle_grid_bc(o);               /* l.4  */
        oracle_grid_advance(o, dt);      /* l.5  */
        oracle_g2p_velocity(o, dt);      /* l.6-7 */
        oracle_p2g2(o);                  /* l.8  */
        oracle_grid_bc2(o);              /* l.9  */
        oracle_particle_update(o, dt);   /* l.10 */
        oracle_cfl(o, alpha);            /* l.13, evaluated on V', Vbar, rho', E' before recycling */
        oracle_advect(o, dt);            /* l.11 */
        o->st.t += dt;                   /* l.13 time advance */
        o->st.dt_last = dt;
        o->st.step += 1;
    }
    if (dt_last) *dt_last = o->st.dt_last;
    return 0;
}

/* Node plane `side` (0 low, 1 high) of the last axis of a slab: which = 0: m, mv[d], f[d]; 1: mv2[d].  op 0: buf <- plane,
 * op 1: plane += buf (the halo sum-exchange of a decomposed domain).  buf: [channels][plane nodes]. */
int oracle_halo(oracle_t *o, int which, int side, int op, double *buf)
{
    if (!o || !buf || (which != 0 && which != 1) || (side != 0 && side != 1) || (op != 0 && op != 1)) return -1;
    const int last = o->d - 1;
    const long long plane = o->Nn / o->nn[last], at = side ? (long long)(o->nn[last] - 1) * plane : 0;
    double *ch[7]; int nch = 0;
    if (which == 0) {
        ch[nch++] = o->m;
        for (int a = 0; a < o->d; ++a) ch[nch++] = o->mv + a * o->Nn;
        for (int a = 0; a < o->d; ++a) ch[nch++] = o->f + a * o->Nn;
    } else for (int a = 0; a < o->d; ++a) ch[nch++] = o->mv2 + a * o->Nn;
    for (int c = 0; c < nch; ++c)
        for (long long j = 0; j < plane; ++j) {
            if (op == 0) buf[c * plane + j] = ch[c][at + j];
            else ch[c][at + j] += buf[c * plane + j];
        }
    return 0;
}

/* Diagnostic only (reading A18; the "interpolated on the grid" curve of Fig. 5): mass-weighted nodal mean
 * of a particle field, out_i = sum_k M_k a_k phi_i(X_k) / sum_k M_k phi_i(X_k) with a = rho (which 0) or E (which 1), 0 where
 * the node has no mass.  Q1 basis.  Not part of Algorithm 1; touches none of its arrays. */
int oracle_grid_diagnostic(const oracle_t *o, int which, double *out)
{
    if (!o || !out || (which != 0 && which != 1) || o->cfg.basis != ORC_BASIS_Q1) return -1;
    const long long n = o->Np, Nn = o->Nn;
    const int nb = 1 << o->d;
    double *den = (double *)calloc((size_t)Nn, sizeof(double));
    for (long long i = 0; i < Nn; ++i) out[i] = 0.0;
    for (long long k = 0; k < n; ++k) {
        int c[3]; double w[3][2], g[3][2];
        particle_cell(o, &o->X[k], n, c, w, g);
        double a = which == 0 ? o->rho[k] : o->E[k];
        for (int ib = 0; ib < nb; ++ib) {
            int b[3] = { ib & 1, (ib >> 1) & 1, (ib >> 2) & 1 };
            double phi, grad[3];
            long long i = corner_node(o, c, b);
            corner_weights(o, w, g, b, &phi, grad);
            out[i] += o->M[k] * a * phi;
            den[i] += o->M[k] * phi;
        }
    }
    for (long long i = 0; i < Nn; ++i) out[i] = (den[i] != 0.0) ? out[i] / den[i] : 0.0;
    free(den);
    return 0;
}

/* ---------------------------------------------------------------- read-back */

int oracle_read_particles(const oracle_t *o, int field, double *out)
{
    const long long n = o->Np;
    const double *src = NULL; int nc = 1;
    switch (field) {
    case ORC_P_X: src = o->X; nc = o->d; break;
    case ORC_P_V: src = o->V; nc = o->d; break;
    case ORC_P_M: src = o->M; break;
    case ORC_P_RHO: src = o->rho; break;
    case ORC_P_E: src = o->E; break;
    case ORC_P_Q: src = o->Q; break;
    case ORC_P_VBAR: src = o->Vbar; nc = o->d; break;
    case ORC_P_ACC: src = o->A; nc = o->d; break;
    case ORC_P_DIV: src = o->D; break;
    default: return -1;
    }
    memcpy(out, src, sizeof(double) * (size_t)(nc * n));
    return 0;
}

int oracle_read_grid(const oracle_t *o, int field, double *out)
{
    const long long Nn = o->Nn;
    switch (field) {
    case ORC_G_MASS: memcpy(out, o->m, sizeof(double) * (size_t)Nn); return 0;
    case ORC_G_MOM: memcpy(out, o->mv, sizeof(double) * (size_t)(o->d * Nn)); return 0;
    case ORC_G_FORCE: memcpy(out, o->f, sizeof(double) * (size_t)(o->d * Nn)); return 0;
    case ORC_G_MOM2: memcpy(out, o->mv2, sizeof(double) * (size_t)(o->d * Nn)); return 0;
    case ORC_G_NORMAL: memcpy(out, o->normal, sizeof(double) * (size_t)(o->d * Nn)); return 0;
    case ORC_G_FLAG: for (long long i = 0; i < Nn; ++i) out[i] = (double)o->obst[i]; return 0;
    default: return -1;
    }
}

void oracle_get_stats(const oracle_t *o, oracle_stats *s) { *s = o->st; }
