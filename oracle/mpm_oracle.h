/*
 * mpm_oracle.h -- CPU ORACLE for the compressible-flow MPM particle-grid cycle.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, link, import or run
 * anything under oracle/.  It shares no code with the CUDA path (include/, paper_2404_17057_b200/).
 *
 * Plain, slow, single-threaded fp64 C written from /root/reference/PAPER.md
 * (arXiv 2404.17057): Section 3 steps (i)-(xiv) and Algorithm 1
 * (PAPER.md:757-796), in the paper's order and notation, no blocking, fusion or
 * reordering.  Points where the paper is silent are resolved by the readings
 * A1..A19 listed in DESIGN.md (taken from SURVEY.md section 8(c)); each function in
 * mpm_oracle.c cites the passage and the reading it follows.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"): partition of unity, brute-force
 * evaluation of eqs. (16)-(19) with global hat functions, affine reproduction, mass /
 * momentum / work-identity conservation, steady states, uniform compression closed form,
 * obstacle rule, CFL identity, mirror symmetry, exact Riemann solution of the Sod tube.
 * Unpinned against the AUTHORS' code (no numbers are printed in the paper): the timing of
 * Q (A2), normals derived from a cell mask (A7), outflow treatment (A10) -- "parity
 * unpinned" versus the authors for those three readings; they are pinned internally.
 */
#ifndef MPM_ORACLE_H
#define MPM_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* boundary-condition codes per face, bc[axis][side] (side 0 = low, 1 = high) */
enum { ORC_BC_PERIODIC = 0, ORC_BC_REFLECT = 1, ORC_BC_INFLOW = 2, ORC_BC_OUTFLOW = 3,
       ORC_BC_OPEN = 4 /* interface to a neighbouring slab of a decomposed domain: no nodal condition, no clamp */ };
/* artificial-viscosity form (reading A3): eq. (4) as printed, or the textbook vNR+Landshoff */
enum { ORC_VISC_PRINTED = 0, ORC_VISC_STANDARD = 1 };

/* shape functions: the paper's Q1 hats, or the quadratic B-splines it names as the next basis
 * (the standard MPM quadratic B-spline of its refs. [60, 19]).  The quadratic basis is offered on
 * fully periodic grids only: the paper does not say how a spline whose support leaves the grid is to be modified at a
 * wall (reading A20). */
enum { ORC_BASIS_Q1 = 0, ORC_BASIS_QUADRATIC = 1 };

/* grid fields for oracle_read_grid (content = whatever the last sub-step left there) */
enum { ORC_G_MASS = 0, ORC_G_MOM = 1, ORC_G_FORCE = 2, ORC_G_MOM2 = 3, ORC_G_NORMAL = 4, ORC_G_FLAG = 5 };
/* particle fields for oracle_read_particles */
enum { ORC_P_X = 0, ORC_P_V = 1, ORC_P_M = 2, ORC_P_RHO = 3, ORC_P_E = 4, ORC_P_Q = 5,
       ORC_P_VBAR = 6, ORC_P_ACC = 7, ORC_P_DIV = 8 };

typedef struct {
    int dim;                 /* 2 or 3 */
    int n[3];                /* cells per axis */
    double dx;               /* h (reading A4: h = dx, cubic cells) */
    double gamma;            /* eq. (3) */
    double c0, c1;           /* eq. (4) */
    int visc_form;           /* ORC_VISC_* (A3) */
    int bc[3][2];            /* ORC_BC_* */
    double inflow_rho, inflow_p, inflow_v[3];
    const unsigned char *obstacle_mask; /* one byte per cell, x fastest, NULL = none (copied) */
    const double *node_normals;         /* [dim][N_n] component-major, NULL = derive (A7) (copied) */
    unsigned long long recycle_seed;    /* A8 */
    double ppc_inflow;                  /* A8: recycled mass = rho_in h^d / ppc_inflow */
    int basis;                          /* ORC_BASIS_* (A20) */
    int slab_global_n, slab_offset;     /* > 0: this grid is cells [offset, offset + n[last]) of slab_global_n along the last
                                           axis (recycled particles are placed on the GLOBAL inflow face) */
} oracle_config;

typedef struct {
    double t, dt_last, dt_next;
    long long step;
    double vmax, cmax;             /* maxima of the last CFL reduction (A12) */
    long long n_recycled;          /* cumulative */
    long long n_clamped;           /* cumulative */
    long long n_negjac;            /* cumulative count of 1 + dt*D <= 0 (A13) */
    long long n_nonfinite;         /* particles with a non-finite rho/E/X after the last step */
} oracle_stats;

typedef struct oracle_s oracle_t;

oracle_t *oracle_create(const oracle_config *cfg);
void oracle_destroy(oracle_t *o);
long long oracle_num_nodes(const oracle_t *o, int nn[3]);
long long oracle_num_particles(const oracle_t *o);

/* arrays are component-major: x[a*n + k]; q may be NULL (-> 0).  Copies everything.
 * Also performs the first CFL reduction from the loaded state (A13). */
int oracle_load_particles(oracle_t *o, long long n, const double *x, const double *v,
                          const double *mass, const double *rho, const double *e, const double *q);

int oracle_load_particles_ex(oracle_t *o, long long n, const double *x, const double *v,
                             const double *mass, const double *rho, const double *e, const double *q,
                             const long long *ids, int keep_time);
int oracle_halo(oracle_t *o, int which, int side, int op, double *buf);
void oracle_advance_time(oracle_t *o, double dt);

/* Q1 shape functions at a point (3D by :729-733): node[2^d], phi[2^d], grad[2^d*d] */
void oracle_shape(const oracle_t *o, const double *X, long long *node, double *phi, double *grad);

/* quadratic B-spline shape functions at a point: node[3^d], phi[3^d], grad[3^d*d] (x fastest) */
void oracle_shape_quadratic(const oracle_t *o, const double *X, long long *node, double *phi, double *grad);

/* counter-based generator of reading A8, exported so that the tests can pin it to the published
 * splitmix64 test vector: oracle_mix64(z) = output function applied to state z + golden gamma */
unsigned long long oracle_mix64(unsigned long long z);
double oracle_recycle_uniform(unsigned long long seed, long long id, long long step, int j);

/* Algorithm 1, line by line.  oracle_step = the sequence below, nsteps times. */
void oracle_grid_reset(oracle_t *o);                 /* l.2  */
void oracle_p2g1(oracle_t *o);                       /* l.3  */
void oracle_grid_bc(oracle_t *o);                    /* l.4  */
void oracle_grid_advance(oracle_t *o, double dt);    /* l.5  */
void oracle_g2p_velocity(oracle_t *o, double dt);    /* l.6-7 */
void oracle_p2g2(oracle_t *o);                       /* l.8  */
void oracle_grid_bc2(oracle_t *o);                   /* l.9  */
void oracle_particle_update(oracle_t *o, double dt); /* l.10 */
void oracle_advect(oracle_t *o, double dt);          /* l.11 (+ wrap / recycle / clamp) */
void oracle_cfl(oracle_t *o, double alpha);          /* l.13 */

/* dt > 0: fixed step; dt <= 0: dt = alpha*h/(vmax+cmax) from the latest reduction (eq. 25/29) */
int oracle_step(oracle_t *o, double dt, double alpha, int nsteps, double *dt_last);

/* diagnostic nodal mean of rho (which 0) or E (which 1), reading A18: out[N_n] */
int oracle_grid_diagnostic(const oracle_t *o, int which, double *out);
int oracle_read_particles(const oracle_t *o, int field, double *out); /* [ncomp][n] */
int oracle_read_grid(const oracle_t *o, int field, double *out);      /* [ncomp][N_n] */
void oracle_get_stats(const oracle_t *o, oracle_stats *s);

#ifdef __cplusplus
}
#endif
#endif
