// trig_kernel.cuh -- trigonometric averages at an arbitrary list of frequencies: the two systems
// (19) and (20) of PAPER.md:242-262 (section 5), the paper's own GPU kernels K1 / K2.
#pragma once
#include "common.cuh"

namespace fredec {

constexpr int kTrigCols = 10;  // <c> <s> <tc> <ts> <xc> <xs> <xtc> <xts> <t^2 c> <t^2 s>

// out [M][kTrigCols]; t, x, w [N] and freqs [M] in device memory.  One CTA per frequency, per-pair
// sincos of the exactly reduced phase (the frequencies are not on a grid: no recurrence applies),
// fixed-order sums.
cudaError_t launch_trig_averages(const double* t, const double* x, const double* w, int64_t N, const double* freqs,
                                 int64_t M, double* out, cudaStream_t stream);

}  // namespace fredec
