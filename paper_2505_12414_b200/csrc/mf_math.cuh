// mf_math.cuh — fp64 device math used inside the per-event bodies (S3).
//
// fp64 exp / log have no hardware unit: they are DFMA polynomials plus integer exponent
// handling, so they ARE the per-event cost of the mass model (SURVEY.md §7 "issue-slot
// pressure").  Arguments on this path are restricted: exp() sees finite arguments <= 700,
// log() sees the positive PDF value.  Events outside those ranges are flagged (P <= 0)
// and their results discarded, so the special-case handling of the general library
// routines is not needed inside the loop.
#pragma once

namespace mf {

__device__ __forceinline__ double mf_rcp(double x) { return __drcp_rn(x); }
__device__ __forceinline__ double mf_exp(double x) { return exp(x); }
__device__ __forceinline__ double mf_log(double x) { return log(x); }

}  // namespace mf
