// Host construction of the per-energy physics table of the transport kernel (physics_tables.h).
//   S(E)   Bethe mass stopping power of water, I = 75 eV, exact T_max, no shell/density corrections
//          (reading A2; BASELINE.json config 1)
//   R_w(E) = R_c + int_{Ec}^{E} dE'/S(E'),  R_c = Ec / S(Ec),  Ec = 0.5 MeV (reading A6); composite Simpson rule,
//          32 panels per table interval, long double accumulation
//   V(E)   = 1/2 K Z/A beta^-2 T_max (1 - beta^2/2)                      (Bohr, T8)
//   T(E)   = (E_s / pv)^2 / X0,  pv = (E^2 + 2 E M_p) / (E + M_p)         (Highland without log term, T9)
#include "physics_tables.h"

#include <cmath>
#include <cstring>

namespace pbs4d {

namespace {
constexpr long double Mp = 938.27208816L, me = 0.51099895L, K = 0.307075L, ZA = 10.0L / 18.01528L, Iex = 75.0e-6L;
constexpr long double X0 = 36.08L, Es = 13.6L, kLn2 = 0.693147180559945309417232121458L;

struct Kin { long double beta2, bg2, gam, tmax; };
Kin kin(long double E)
{
    Kin k;
    const long double tau = E / Mp, q = me / Mp;
    k.bg2 = tau * (tau + 2.0L); k.gam = 1.0L + tau; k.beta2 = k.bg2 / (k.gam * k.gam);
    k.tmax = 2.0L * me * k.bg2 / (1.0L + 2.0L * k.gam * q + q * q);
    return k;
}
long double stopping_power(long double E)
{
    const Kin k = kin(E);
    return K * ZA / k.beta2 * (0.5L * std::log(2.0L * me * k.bg2 * k.tmax / (Iex * Iex)) - k.beta2);
}
long double node_energy(int i)
{
    const uint32_t b = kTabBits0 + ((uint32_t)i << 16);
    float f; std::memcpy(&f, &b, 4);
    return (long double)f;
}
long double inv_S_integral(long double a, long double b)     // int_a^b dE / S(E), b > a
{
    const int panels = 32;
    const long double h = (b - a) / (2 * panels);
    long double sum = 1.0L / stopping_power(a) + 1.0L / stopping_power(b);
    for (int j = 1; j < 2 * panels; ++j) sum += ((j & 1) ? 4.0L : 2.0L) / stopping_power(a + j * h);
    return sum * h / 3.0L;
}
}  // namespace

void build_physics_table(TabNode* nodes)
{
    const int i_cut = 128;                                   // node at exactly 0.5 MeV
    static long double R[kTabNodes];
    R[i_cut] = 0.5L / stopping_power(0.5L);
    for (int i = i_cut + 1; i < kTabNodes; ++i) R[i] = R[i - 1] + inv_S_integral(node_energy(i - 1), node_energy(i));
    for (int i = i_cut - 1; i >= 0; --i)        R[i] = R[i + 1] - inv_S_integral(node_energy(i), node_energy(i + 1));
    for (int i = 0; i < kTabNodes; ++i) {
        const long double E = node_energy(i);
        const Kin k = kin(E);
        const long double pv = (E * E + 2.0L * E * Mp) / (E + Mp);
        nodes[i].rs = (float)(0.2L * R[i]);
        nodes[i].S  = (float)stopping_power(E);
        nodes[i].V2 = (float)(2.0L * kLn2 * 0.5L * K * ZA / k.beta2 * k.tmax * (1.0L - 0.5L * k.beta2));
        nodes[i].T2 = (float)(2.0L * kLn2 * (Es / pv) * (Es / pv) / X0);
    }
}

// untyped entry for api.cu (which does not see the node layout): fills physics_table_bytes() bytes
void build_physics_table_host(void* nodes) { build_physics_table(static_cast<TabNode*>(nodes)); }

}  // namespace pbs4d
