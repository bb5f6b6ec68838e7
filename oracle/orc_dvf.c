/* oracle/orc_dvf.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Construction of the full deformation vector field from the minimal grid information of a DICOM deformable
 * spatial registration, PAPER.md:251-259 (App. B, Eq. 7-8; Sec. 2.D.1: "calculate the full DVF based on
 * the stored minimal-grid information ... one-thread-per-deformation-grid-voxel ... to calculate r_f for all voxels").
 * For grid voxel (i, j, k), i along the row direction U, j along the column direction V, k along W = U x V:
 *   Eq. 8   r_0 = start + i dX U + j dY V + k dZ W
 *   Eq. 7   r_f = M_Post ( M_Pre [r_0; 1] + [Delta; 0] )
 * All arithmetic in double, in the order written below (each product/sum rounded once, no fused multiply-add);
 * outputs: r_f and the displacement r_f - r_0, both rounded to fp32.  Arrays are [3][k][j][i], i fastest. */
#include "orc.h"
#include <stddef.h>

static void mat4_apply(const double* M /* row-major 4x4 */, const double v[4], double out[4])
{
    for (int r = 0; r < 4; ++r) {
        double s = M[4 * r + 0] * v[0];
        s = s + M[4 * r + 1] * v[1];
        s = s + M[4 * r + 2] * v[2];
        s = s + M[4 * r + 3] * v[3];
        out[r] = s;
    }
}

int orc_build_dvf(const orc_dicom_dvf* g, const float* delta, float* rf, float* disp)
{
    if (!g || !delta || g->nx <= 0 || g->ny <= 0 || g->nz <= 0) return -1;
    const double* U = g->row_cos; const double* V = g->col_cos;
    const double W[3] = { U[1] * V[2] - U[2] * V[1], U[2] * V[0] - U[0] * V[2], U[0] * V[1] - U[1] * V[0] };
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    #pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
    for (int j = 0; j < g->ny; ++j)
    for (int i = 0; i < g->nx; ++i) {
        const size_t v = ((size_t)k * g->ny + j) * g->nx + i;
        double r0[4], a[4], b[4];
        for (int c = 0; c < 3; ++c) {                                   /* Eq. 8 */
            double s = U[c] * g->delta[0] * (double)i;
            s = s + V[c] * g->delta[1] * (double)j;
            s = s + W[c] * g->delta[2] * (double)k;
            r0[c] = s + g->start[c];
        }
        r0[3] = 1.0;
        mat4_apply(g->pre, r0, a);                                      /* Eq. 7 */
        for (int c = 0; c < 3; ++c) a[c] = a[c] + (double)delta[(size_t)c * n + v];
        mat4_apply(g->post, a, b);
        for (int c = 0; c < 3; ++c) {
            if (rf)   rf[(size_t)c * n + v]   = (float)b[c];
            if (disp) disp[(size_t)c * n + v] = (float)(b[c] - r0[c]);
        }
    }
    return 0;
}
