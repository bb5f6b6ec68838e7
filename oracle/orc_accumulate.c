/* oracle/orc_accumulate.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Energy-/mass-transfer subvoxel dose accumulation, SURVEY 8(c) steps A1-A6.
 * PAPER.md:106-124 (Sec. 2.D.2, Eq. 4-6): every source voxel j is split into n x n x n subvoxels, M = rho_j v_k,
 * E = M D_j (Eq. 4); the subvoxel centre is mapped by the trilinearly interpolated DVF T^{S->R} (Eq. 1, App. B
 * PAPER.md:259) and E, M are summed into the reference voxel that contains the image (Eq. 6); D_i^S = sum E / sum M
 * (Eq. 5); D_i = D_i^R + sum_S D_i^S (Eq. 2); mask to the volume covered by all DVFs.
 * Arithmetic: strict IEEE fp32, one rounding per operation, NO fused multiply-add (build with
 * -ffp-contract=off), integers for the sums -- there is exactly one correct result. */
#include "orc.h"
#include <math.h>
#include <stddef.h>

/* A2: centre of subvoxel a (of ns) of voxel i on an axis */
static float sub_centre(float o, float h, int i, int a, int ns)
{
    float f = ((float)a + 0.5f) / (float)ns;
    float c = (float)i + f;
    float m = c * h;
    return o + m;
}

/* A3: continuous DVF-grid index; returns 0 if outside the DVF grid's voxel extent */
static int dvf_coord(float p, float od, float hd, int nd, int* i0, int* i1, float* w)
{
    float d = p - od;
    float q = d / hd;
    float g = q - 0.5f;
    if (!(g >= -0.5f) || !(g < (float)nd - 0.5f)) return 0;
    if (g < 0.0f) g = 0.0f;
    if (g > (float)(nd - 1)) g = (float)(nd - 1);
    int k = (int)floorf(g);
    if (k > nd - 2) k = nd - 2;
    if (k < 0) k = 0;
    *i0 = k;
    *i1 = (k + 1 < nd) ? k + 1 : nd - 1;
    *w  = g - (float)k;
    return 1;
}

static float lerp(float A, float B, float w)
{
    float d = B - A;
    float m = w * d;
    return A + m;
}

/* A4: destination index on an axis; returns 0 if outside [0, n) */
static int dest_index(float q, float o, float h, int n, int* ix)
{
    float d = q - o;
    float v = d / h;
    float fl = floorf(v);
    if (!(fl >= 0.0f) || !(fl < (float)n)) return 0;
    *ix = (int)fl;
    return 1;
}

int orc_emtm_push(const orc_grid* S, const float* dose, const float* rho,
                  const orc_grid* Dg, const float* disp,
                  const orc_grid* R, int32_t nsx, int32_t nsy, int32_t nsz,
                  int64_t* E, int64_t* M, orc_acc_stats* stats)
{
    if (!S || !dose || !rho || !Dg || !disp || !R || !E || !M || nsx < 1 || nsy < 1 || nsz < 1) return -1;
    const size_t plane = (size_t)Dg->nx * Dg->ny * Dg->nz;
    const float* U[3] = { disp, disp + plane, disp + 2 * plane };
    uint64_t n_sub = 0, n_ref = 0, n_dvf = 0;

    #pragma omp parallel for schedule(dynamic, 1) reduction(+:n_sub,n_ref,n_dvf)
    for (int k = 0; k < S->nz; ++k)
    for (int j = 0; j < S->ny; ++j)
    for (int i = 0; i < S->nx; ++i) {
        size_t v = ((size_t)k * S->ny + j) * S->nx + i;
        /* A1 (Eq. 4; the common subvoxel volume v_k cancels in Eq. 5) */
        int64_t m_q = llrint((double)rho[v] * 16777216.0);
        int64_t e_q = llrint((double)rho[v] * (double)dose[v] * 4294967296.0);
        for (int c = 0; c < nsz; ++c)
        for (int b = 0; b < nsy; ++b)
        for (int a = 0; a < nsx; ++a) {
            n_sub += 1;
            float p[3] = { sub_centre(S->ox, S->hx, i, a, nsx),
                           sub_centre(S->oy, S->hy, j, b, nsy),
                           sub_centre(S->oz, S->hz, k, c, nsz) };
            int x0, x1, y0, y1, z0, z1; float wx, wy, wz;
            if (!dvf_coord(p[0], Dg->ox, Dg->hx, Dg->nx, &x0, &x1, &wx) ||
                !dvf_coord(p[1], Dg->oy, Dg->hy, Dg->ny, &y0, &y1, &wy) ||
                !dvf_coord(p[2], Dg->oz, Dg->hz, Dg->nz, &z0, &z1, &wz)) { n_dvf += 1; continue; }
            float q[3];
            for (int comp = 0; comp < 3; ++comp) {
                const float* u = U[comp];
                #define DV(zz, yy, xx) u[((size_t)(zz) * Dg->ny + (yy)) * Dg->nx + (xx)]
                float c00 = lerp(DV(z0, y0, x0), DV(z0, y0, x1), wx);
                float c01 = lerp(DV(z0, y1, x0), DV(z0, y1, x1), wx);
                float c10 = lerp(DV(z1, y0, x0), DV(z1, y0, x1), wx);
                float c11 = lerp(DV(z1, y1, x0), DV(z1, y1, x1), wx);
                #undef DV
                float c0 = lerp(c00, c01, wy);
                float c1 = lerp(c10, c11, wy);
                float uu = lerp(c0, c1, wz);
                q[comp] = p[comp] + uu;                      /* Eq. 1 / Eq. 7 with identity pre/post matrices */
            }
            int ix, iy, iz;
            if (!dest_index(q[0], R->ox, R->hx, R->nx, &ix) ||
                !dest_index(q[1], R->oy, R->hy, R->ny, &iy) ||
                !dest_index(q[2], R->oz, R->hz, R->nz, &iz)) { n_ref += 1; continue; }
            size_t dst = ((size_t)iz * R->ny + iy) * R->nx + ix;
            #pragma omp atomic
            E[dst] += e_q;                                   /* A5 */
            #pragma omp atomic
            M[dst] += m_q;
        }
    }
    if (stats) { stats->subvoxels = n_sub; stats->dropped_outside_ref = n_ref; stats->dropped_outside_dvf = n_dvf; }
    return 0;
}

int orc_emtm_finalize(const orc_grid* R, const float* dose_ref, int32_t n_src,
                      const int64_t* E, const int64_t* M, const orc_grid* dg, float* out)
{
    if (!R || !dose_ref || n_src < 0 || (n_src && (!E || !M || !dg)) || !out) return -1;
    const size_t nv = (size_t)R->nx * R->ny * R->nz;
    #pragma omp parallel for schedule(static)
    for (int k = 0; k < R->nz; ++k)
    for (int j = 0; j < R->ny; ++j)
    for (int i = 0; i < R->nx; ++i) {
        size_t v = ((size_t)k * R->ny + j) * R->nx + i;
        /* mask: voxel centre must lie inside every source DVF's extent */
        float p[3] = { sub_centre(R->ox, R->hx, i, 0, 1), sub_centre(R->oy, R->hy, j, 0, 1), sub_centre(R->oz, R->hz, k, 0, 1) };
        int covered = 1;
        for (int s = 0; s < n_src && covered; ++s) {
            int a0, a1; float w;
            covered = dvf_coord(p[0], dg[s].ox, dg[s].hx, dg[s].nx, &a0, &a1, &w) &&
                      dvf_coord(p[1], dg[s].oy, dg[s].hy, dg[s].ny, &a0, &a1, &w) &&
                      dvf_coord(p[2], dg[s].oz, dg[s].hz, dg[s].nz, &a0, &a1, &w);
        }
        if (!covered) { out[v] = 0.0f; continue; }
        double D = (double)dose_ref[v];                      /* Eq. 2 */
        for (int s = 0; s < n_src; ++s) {
            int64_t m = M[(size_t)s * nv + v];
            if (m != 0) D += (double)E[(size_t)s * nv + v] / (double)m * (1.0 / 256.0);   /* Eq. 5 */
        }
        out[v] = (float)D;
    }
    return 0;
}
