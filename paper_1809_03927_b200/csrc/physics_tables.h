// Per-energy physics table shared by the host builder (tables.cpp) and the transport kernel (transport.cu).
//
// Grid: node i sits at the energy whose IEEE-754 bit pattern is kTabBits0 + (i << 16), i.e. 128 nodes per octave,
// equally spaced in E inside each octave, from 0.25 MeV (below the 0.5 MeV transport cutoff, so the midpoint
// energy of the last step is still inside) to 512 MeV.  The kernel finds the interval of an energy E with integer
// operations on its bit pattern (no logarithm) and interpolates linearly in E; with 128 nodes per octave the
// relative interpolation error of a power-law-like function E^p is <= p(p-1)/8 * 2^-14 ~ 1e-5.
//
// Each node holds four quantities of water at kinetic energy E (BASELINE.json config 1):
//   x: 0.2 * R_w(E)         2 % of the CSDA range, as mm * g/cm3 (divide by the density to get the step limit in mm)
//   y: S(E)                 Bethe mass stopping power, MeV cm2/g
//   z: 2 ln2 * V(E)         V = Bohr straggling variance per mass thickness, MeV2 cm2/g (relativistic form)
//   w: 2 ln2 * T(E)         T = Highland theta0^2 per mass thickness (no log term), (E_s/pv)^2 / X0, cm2/g
// The factor 2 ln2 turns -log2(u) into the -2 ln(u) of Box-Muller.
#pragma once
#include <cstdint>
namespace pbs4d {
constexpr uint32_t kTabBits0 = 0x3E800000u;                 // 0.25f
constexpr int      kTabOctaves = 11;                        // 0.25 .. 512 MeV
constexpr int      kTabNodes = kTabOctaves * 128 + 1;       // 1409 nodes, 22.5 KB as float4
struct TabNode { float rs, S, V2, T2; };
void build_physics_table(TabNode* nodes /*[kTabNodes]*/);
}  // namespace pbs4d
