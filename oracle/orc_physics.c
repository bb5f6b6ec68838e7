/* oracle/orc_physics.c -- CPU ORACLE (test infrastructure only; see orc.h).
 * Philox4x32-10 and the closed forms of T5, T8, T9 in double precision.
 * Model statement: BASELINE.json north_star + config 1 ("Bethe-Bloch CSDA energy loss, Highland
 * multiple-Coulomb-scattering deflection and Bohr straggling", water I = 75 eV); PAPER.md:69 gives no physics. */
#include "orc.h"
#include <math.h>
#include <stdlib.h>

/* ---------------- T1: Philox4x32-10 ---------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;   /* M0 * c0 */
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;   /* M1 * c2 */
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;                          /* Weyl key schedule, bumped between rounds */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ---------------- constants (SURVEY section 8 header) ---------------- */
static const double K_BETHE = 0.307075;        /* MeV cm2/mol */
static const double ME      = 0.51099895;      /* MeV */
static const double MP      = 938.27208816;    /* MeV */
static const double ZA      = 10.0 / 18.01528; /* water Z/A */
static const double I_MEV   = 75.0e-6;         /* BASELINE.json config 1: I = 75 eV */
static const double X0      = 36.08;           /* g/cm2, water */
static const double ES      = 13.6;            /* MeV, Highland */
static const double E_CUT   = 0.5;             /* MeV, BASELINE.json config 1 */

static void kin(double E, double* beta2, double* gamma, double* tmax)
{
    double g  = 1.0 + E / MP;
    double b2 = 1.0 - 1.0 / (g * g);
    double r  = ME / MP;
    *gamma = g; *beta2 = b2;
    *tmax  = 2.0 * ME * b2 * g * g / (1.0 + 2.0 * g * r + r * r);
}

/* T5: S(E) = K (Z/A) / beta^2 [ 1/2 ln(2 me c2 beta2 gamma2 Tmax / I^2) - beta2 ] */
double orc_bethe_S(double E)
{
    double b2, g, tm;
    kin(E, &b2, &g, &tm);
    double arg = 2.0 * ME * b2 * g * g * tm / (I_MEV * I_MEV);
    return K_BETHE * ZA / b2 * (0.5 * log(arg) - b2);
}

/* T8: Bohr variance per mass thickness: 1/2 K (Z/A) / beta2 * Tmax * (1 - beta2/2) */
double orc_bohr_var_per_t(double E)
{
    double b2, g, tm;
    kin(E, &b2, &g, &tm);
    return 0.5 * K_BETHE * ZA / b2 * tm * (1.0 - 0.5 * b2);
}

/* T9: theta0^2 / t = (Es/pv)^2 / X0, pv = (E^2 + 2 E Mp)/(E + Mp); no logarithmic term (reading A8) */
double orc_theta0_sq_per_t(double E)
{
    double pv = (E * E + 2.0 * E * MP) / (E + MP);
    double a  = ES / pv;
    return a * a / X0;
}

/* ---------------- T5: CSDA range table ----------------
 * R_w(E) = R_c + int_{Ec}^{E} dE'/S(E'),  R_c = Ec/S(Ec)  (reading A6).
 * NTAB log-spaced nodes on [Ec, EMAX]; each interval integrated with 4-point Gauss-Legendre in ln E. */
#define NTAB 32768
static const double EMAX = 400.0;
static double* g_lnR = 0;   /* ln R_w at nodes */
static double  g_dl;        /* node spacing in ln E */

static void build_table(void)
{
    static const double gx[4] = { -0.8611363115940526, -0.3399810435848563, 0.3399810435848563, 0.8611363115940526 };
    static const double gw[4] = {  0.3478548451374538,  0.6521451548625461, 0.6521451548625461, 0.3478548451374538 };
    double* t = (double*)malloc(sizeof(double) * NTAB);
    double l0 = log(E_CUT);
    g_dl = (log(EMAX) - l0) / (NTAB - 1);
    double R = E_CUT / orc_bethe_S(E_CUT);
    t[0] = log(R);
    for (int i = 1; i < NTAB; ++i) {
        double la = l0 + (i - 1) * g_dl, lb = l0 + i * g_dl;
        double mid = 0.5 * (la + lb), half = 0.5 * (lb - la), acc = 0.0;
        for (int q = 0; q < 4; ++q) {
            double E = exp(mid + half * gx[q]);
            acc += gw[q] * E / orc_bethe_S(E);      /* dE/S = E dlnE / S */
        }
        R += acc * half;
        t[i] = log(R);
    }
    g_lnR = t;
}

double orc_range_water(double E)
{
    if (!g_lnR) {
        #pragma omp critical(orc_range_table)
        { if (!g_lnR) build_table(); }
    }
    if (E <= E_CUT) return E / orc_bethe_S(E_CUT) ;  /* below the cutoff: linear closure (never used by T-steps) */
    double x = (log(E) - log(E_CUT)) / g_dl;
    int i = (int)floor(x);
    if (i > NTAB - 2) i = NTAB - 2;
    double f = x - i;
    return exp(g_lnR[i] + f * (g_lnR[i + 1] - g_lnR[i]));
}
