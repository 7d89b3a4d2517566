// arc_divide.cuh -- the tracer's division (DESIGN.md 6.2 step 1; contract C3 demands the IEEE quotient).
// Shared by arc_trace_kernel.cuh (the march) and arc_trace.cu (arc_selftest_division, which hammers it against
// __ddiv_rn).  Nothing here is shared with oracle/.
#pragma once

// a / b rounded to nearest, bit-identical to IEEE division, given y = RN(1 / b) (one true division per ray and axis):
// q0 = RN(a y) is within 1.5 ulp of a/b; one residual correction q1 = RN(q0 + (a - b q0) y) makes it faithful, and
// for a faithful q1 and a correctly rounded y the second correction returns RN(a / b) (Markstein 1990, the closing
// step of the IA-64 division sequences).  The residuals are exact (FMA).  No overflow / underflow here: |a| <= 2N,
// 2^-40 < |b| <= 1.  Five FP64 instructions instead of the ~17 of the generic division.
__device__ __forceinline__ double arc_div_by_recip(double a, double b, double y)
{
    const double q0 = __dmul_rn(a, y);
    const double q1 = __fma_rn(__fma_rn(-b, q0, a), y, q0);
    return __fma_rn(__fma_rn(-b, q1, a), y, q1);
}
