// Host construction of the water CSDA range table used by the transport kernel:
//   R_w(E) = R_c + int_{Ec}^{E} dE'/S(E'),  R_c = Ec / S(Ec),  Ec = 0.5 MeV,
// S = Bethe mass stopping power of water with I = 75 eV (BASELINE.json config 1), no shell/density corrections.
// Composite Simpson rule in E, 16 panels per table interval, long double accumulation.
#include "physics_tables.h"

#include <cmath>

namespace pbs4d {

namespace {
long double stopping_power(long double E)
{
    const long double Mp = 938.27208816L, me = 0.51099895L, K = 0.307075L, ZA = 10.0L / 18.01528L, I = 75.0e-6L;
    const long double tau = E / Mp, bg2 = tau * (tau + 2.0L), gam = 1.0L + tau, beta2 = bg2 / (gam * gam);
    const long double q = me / Mp;
    const long double tmax = 2.0L * me * bg2 / (1.0L + 2.0L * gam * q + q * q);
    return K * ZA / beta2 * (0.5L * std::log(2.0L * me * bg2 * tmax / (I * I)) - beta2);
}
}  // namespace

void build_range_table(float* log2_range)
{
    const long double Ec = 0.5L;
    long double R = Ec / stopping_power(Ec);
    long double E_prev = std::exp2((long double)kRangeLog2E0);
    log2_range[0] = (float)std::log2(R);
    for (int i = 1; i < kRangeNodes; ++i) {
        const long double E_next = std::exp2((long double)kRangeLog2E0 + (long double)i / (long double)kRangeInvStep);
        const int panels = 16;
        const long double hstep = (E_next - E_prev) / (2 * panels);
        long double sum = 1.0L / stopping_power(E_prev) + 1.0L / stopping_power(E_next);
        for (int j = 1; j < 2 * panels; ++j)
            sum += ((j & 1) ? 4.0L : 2.0L) / stopping_power(E_prev + j * hstep);
        R += sum * hstep / 3.0L;
        log2_range[i] = (float)std::log2(R);
        E_prev = E_next;
    }
}

}  // namespace pbs4d
