// mpm_node_bc.cuh -- the boundary and obstacle conditions of one grid node (Alg. 1 l.4 and l.9), shared by the node
// kernels (mpm_kernels_grid.cu) and by the tile kernels, which apply them while staging a tile (mpm_kernels_tiled.cu).
#pragma once
#include "mpm_internal.cuh"

namespace mpm {

// Domain-face and obstacle conditions on one node's (mv, f) pair, in the order x, y, z faces then obstacle (A9, A14).
// WITH_F = false is the second application (momentum only).
template <int DIM, bool WITH_F>
__device__ __forceinline__ void apply_bc(const GridDesc &gd, const GArr &g, long long i, const int idx[DIM], double m,
                                         double mv[DIM], double f[DIM])
{
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        if (gd.per[a]) continue;
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const bool on_face = (s == 0) ? (idx[a] == 0) : (idx[a] == gd.nn[a] - 1);
            if (!on_face) continue;
            const int bc = gd.bc[a][s];
            if (bc == MPM_BC_REFLECT) {            // eq. (30): v.n = 0
                mv[a] = 0.0;
                if (WITH_F) f[a] = 0.0;
            } else if (bc == MPM_BC_INFLOW) {      // Dirichlet inflow
#pragma unroll
                for (int a2 = 0; a2 < DIM; ++a2) {
                    mv[a2] = m * gd.inflow_v[a2];
                    if (WITH_F) f[a2] = 0.0;
                }
            } else if (bc == MPM_BC_OUTFLOW) {     // A10
                if (WITH_F) f[a] = 0.0;
            }
        }
    }
    if (gd.has_obstacle && g.flag[i]) {
        double nrm[DIM], dot = 0.0, dotf = 0.0;
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            nrm[a] = g.normal[a][i];
            dot += mv[a] * nrm[a];
            if (WITH_F) dotf += f[a] * nrm[a];
        }
        const double half = (dot - fabs(dot)) / 2.0;       // eq. (21)
        const double halff = (dotf - fabs(dotf)) / 2.0;    // eq. (22)
#pragma unroll
        for (int a = 0; a < DIM; ++a) {
            mv[a] -= half * nrm[a];
            if (WITH_F) f[a] -= halff * nrm[a];
        }
    }
}

}  // namespace mpm
