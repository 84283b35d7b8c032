// Small device helpers shared by the kernels.
#pragma once
#include "oci_internal.h"

namespace oci {

// Early exit for launches queued after the step has converged: the previous
// iteration's norms are final when this kernel starts (stream order).
__device__ __forceinline__ bool step_done(const unsigned long long* __restrict__ norms, int prev_slot,
                                          double tol)
{
    if (prev_slot < 0) return false;
    double d = __longlong_as_double((long long)norms[2 * prev_slot + 0]);
    double r = __longlong_as_double((long long)norms[2 * prev_slot + 1]);
    return converged(tol, d, r);
}

// max over non-negative doubles through their (order-preserving) bit patterns: exact and
// independent of the reduction order, so host and device agree on the iteration count.
__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v)
{
    // same-address atomics serialise in L2 (about 25 ns each with thousands of CTAs): skip the ones
    // that cannot raise the maximum (the plain read may be stale low, never high: max only grows)
    const unsigned long long bits = (unsigned long long)__double_as_longlong(v);
    if (bits > __ldcg(addr)) atomicMax(addr, bits);
}

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// D(8x8) += A(8x4, row) * B(4x8, col), fp64 tensor pipe (SASS DMMA.8x8x4).
// a: A[lane/4][lane%4]; b: B[lane%4][lane/4]; c0,c1: C[lane/4][2*(lane%4) + {0,1}].
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

}  // namespace oci
