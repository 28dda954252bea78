// pm_fast.cuh -- specialised deposit / return kernels for the shapes the BASELINE configs use:
//   pm_sn_fast.cuh    supernova deposit, kernel half-width 3 with 4 sub-samples per axis
//   pm_sink_fast.cuh  sink deposit and return, kernel half-width 4
// Same arithmetic contract as the generic kernels in pm_b200.cu: every integer decision (host cell, membership,
// omega count) is evaluated by the same fp64 expressions in the same order; value arithmetic may differ by a few ulp
// (no per-cell divisions, explicit fma, separable Gaussian), far inside the parity tolerances of DESIGN.md.
#pragma once
#include "pm_sn_fast.cuh"
#include "pm_sink_fast.cuh"
