// CSDA range table geometry shared by the host builder (tables.cpp) and the transport kernel.
// Nodes are equally spaced in log2(E): E_i = 2^(kRangeLog2E0 + i / kRangeInvStep), i = 0 .. kRangeNodes-1,
// covering 0.5 MeV (the transport cutoff, BASELINE.json config 1) to 512 MeV; the table holds log2(R_w [g/cm2]).
#pragma once
namespace pbs4d {
constexpr int   kRangeNodes   = 1281;
constexpr float kRangeLog2E0  = -1.0f;
constexpr float kRangeInvStep = 128.0f;
void build_range_table(float* log2_range /*[kRangeNodes]*/);
}  // namespace pbs4d
