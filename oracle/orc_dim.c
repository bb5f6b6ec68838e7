/* oracle/orc_dim.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Dose-interpolation method (DIM) of dose accumulation, PAPER.md:95-100 (Sec. 2.D.2, Eq. 3):
 *   "For each source phase S: each voxel on I_R was split into n x n x n subvoxels, the central location of each
 *    subvoxel r_ik was mapped to I_S giving T^{R->S}(r_ik), the trilinearly-interpolated dose at this location
 *    D~^S[T^{R->S}(r_ik)] was computed and the final D_i^S was then  D_i^S = n^-3 sum_k D~^S[T^{R->S}(r_ik)]".
 * Steps (DESIGN.md "DIM steps" P1-P5; arithmetic as for the EMTM oracle: strict IEEE fp32, one rounding per
 * operation, no fused multiply-add; the sum over subvoxels in double, in (b, a, c) loop order -- c, the z index,
 * innermost: Eq. 3 is a plain mean, the paper fixes no order, and this one lets an implementation walk a subvoxel
 * column along z, where consecutive subvoxels share the x/y-interpolated DVF values (reading D4)):
 *   P1  subvoxel centre on the reference grid            p = o + ((float)i + (a + 0.5f)/ns) * h      (as A2)
 *   P2  displacement T^{R->S} at p by trilinear interpolation between DVF-grid centres (as A3);
 *       a centre outside the DVF grid's voxel extent contributes nothing
 *   P3  q = p + u                                                                                      (Eq. 1)
 *   P4  D~^S(q): trilinear interpolation between the centres of the source dose grid, clamp-to-edge inside the
 *       grid's voxel extent, 0 outside it (4 lerps in x, 2 in y, 1 in z; lerp(A,B,w) = A + w*(B-A))
 *   P5  D_i^S = (sum_k (double)D~^S) / (double)(nsx*nsy*nsz)                                            (Eq. 3)
 * Final sum (Eq. 2) and mask as for the EMTM: out = (float)((double)D^R + sum_S D_i^S) in ascending
 * phase order, 0 where the voxel centre is outside any DVF's extent. */
#include "orc.h"
#include <math.h>
#include <stddef.h>

static float centre_of(float o, float h, int i, int a, int ns)
{
    float f = ((float)a + 0.5f) / (float)ns;
    float c = (float)i + f;
    float m = c * h;
    return o + m;
}

/* continuous index of coordinate p between the centres of a grid axis; 0 if p is outside the voxel extent */
static int cell_of(float p, float o, float h, int n, int* i0, int* i1, float* w)
{
    float d = p - o;
    float q = d / h;
    float g = q - 0.5f;
    if (!(g >= -0.5f) || !(g < (float)n - 0.5f)) return 0;
    if (g < 0.0f) g = 0.0f;
    if (g > (float)(n - 1)) g = (float)(n - 1);
    int k = (int)floorf(g);
    if (k > n - 2) k = n - 2;
    if (k < 0) k = 0;
    *i0 = k;
    *i1 = (k + 1 < n) ? k + 1 : n - 1;
    *w  = g - (float)k;
    return 1;
}

static float mix(float A, float B, float w)
{
    float d = B - A;
    float m = w * d;
    return A + m;
}

static float trilinear(const float* f, const orc_grid* G, int x0, int x1, int y0, int y1, int z0, int z1,
                       float wx, float wy, float wz)
{
    #define AT(zz, yy, xx) f[((size_t)(zz) * G->ny + (yy)) * G->nx + (xx)]
    float c00 = mix(AT(z0, y0, x0), AT(z0, y0, x1), wx);
    float c01 = mix(AT(z0, y1, x0), AT(z0, y1, x1), wx);
    float c10 = mix(AT(z1, y0, x0), AT(z1, y0, x1), wx);
    float c11 = mix(AT(z1, y1, x0), AT(z1, y1, x1), wx);
    #undef AT
    float c0 = mix(c00, c01, wy);
    float c1 = mix(c10, c11, wy);
    return mix(c0, c1, wz);
}

int orc_dim_pull(const orc_grid* R, int32_t nsx, int32_t nsy, int32_t nsz,
                 const orc_grid* Dg, const float* disp /* T^{R->S}, [3][z][y][x] on Dg, reference frame */,
                 const orc_grid* S, const float* dose_src, double* dose_pulled /* [R voxels], D_i^S */,
                 orc_acc_stats* stats)
{
    if (!R || !Dg || !disp || !S || !dose_src || !dose_pulled || nsx < 1 || nsy < 1 || nsz < 1) return -1;
    const size_t plane = (size_t)Dg->nx * Dg->ny * Dg->nz;
    const float* U[3] = { disp, disp + plane, disp + 2 * plane };
    const double n_sub_vox = (double)nsx * (double)nsy * (double)nsz;
    uint64_t n_sub = 0, n_src = 0, n_dvf = 0;

    #pragma omp parallel for schedule(dynamic, 1) reduction(+:n_sub,n_src,n_dvf)
    for (int k = 0; k < R->nz; ++k)
    for (int j = 0; j < R->ny; ++j)
    for (int i = 0; i < R->nx; ++i) {
        double sum = 0.0;
        for (int b = 0; b < nsy; ++b)
        for (int a = 0; a < nsx; ++a)
        for (int c = 0; c < nsz; ++c) {
            n_sub += 1;
            /* P1 */
            float p[3] = { centre_of(R->ox, R->hx, i, a, nsx), centre_of(R->oy, R->hy, j, b, nsy),
                           centre_of(R->oz, R->hz, k, c, nsz) };
            /* P2 */
            int x0, x1, y0, y1, z0, z1; float wx, wy, wz;
            if (!cell_of(p[0], Dg->ox, Dg->hx, Dg->nx, &x0, &x1, &wx) ||
                !cell_of(p[1], Dg->oy, Dg->hy, Dg->ny, &y0, &y1, &wy) ||
                !cell_of(p[2], Dg->oz, Dg->hz, Dg->nz, &z0, &z1, &wz)) { n_dvf += 1; continue; }
            float q[3];
            for (int comp = 0; comp < 3; ++comp)
                q[comp] = p[comp] + trilinear(U[comp], Dg, x0, x1, y0, y1, z0, z1, wx, wy, wz);      /* P3 */
            /* P4 */
            if (!cell_of(q[0], S->ox, S->hx, S->nx, &x0, &x1, &wx) ||
                !cell_of(q[1], S->oy, S->hy, S->ny, &y0, &y1, &wy) ||
                !cell_of(q[2], S->oz, S->hz, S->nz, &z0, &z1, &wz)) { n_src += 1; continue; }
            sum += (double)trilinear(dose_src, S, x0, x1, y0, y1, z0, z1, wx, wy, wz);
        }
        dose_pulled[((size_t)k * R->ny + j) * R->nx + i] = sum / n_sub_vox;                            /* P5 */
    }
    if (stats) { stats->subvoxels = n_sub; stats->dropped_outside_ref = n_src; stats->dropped_outside_dvf = n_dvf; }
    return 0;
}

int orc_dim_finalize(const orc_grid* R, const float* dose_ref, int32_t n_src, const double* pulled /* [n_src][R] */,
                     const orc_grid* dg, float* out)
{
    if (!R || !dose_ref || n_src < 0 || (n_src && (!pulled || !dg)) || !out) return -1;
    const size_t nv = (size_t)R->nx * R->ny * R->nz;
    #pragma omp parallel for schedule(static)
    for (int k = 0; k < R->nz; ++k)
    for (int j = 0; j < R->ny; ++j)
    for (int i = 0; i < R->nx; ++i) {
        size_t v = ((size_t)k * R->ny + j) * R->nx + i;
        float p[3] = { centre_of(R->ox, R->hx, i, 0, 1), centre_of(R->oy, R->hy, j, 0, 1), centre_of(R->oz, R->hz, k, 0, 1) };
        int covered = 1;
        for (int s = 0; s < n_src && covered; ++s) {
            int a0, a1; float w;
            covered = cell_of(p[0], dg[s].ox, dg[s].hx, dg[s].nx, &a0, &a1, &w) &&
                      cell_of(p[1], dg[s].oy, dg[s].hy, dg[s].ny, &a0, &a1, &w) &&
                      cell_of(p[2], dg[s].oz, dg[s].hz, dg[s].nz, &a0, &a1, &w);
        }
        if (!covered) { out[v] = 0.0f; continue; }
        double D = (double)dose_ref[v];                                                    /* Eq. 2 */
        for (int s = 0; s < n_src; ++s) D += pulled[(size_t)s * nv + v];
        out[v] = (float)D;
    }
    return 0;
}
