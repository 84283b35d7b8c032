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
    double d = __longlong_as_double((long long)__ldcg(norms + 2 * prev_slot + 0));
    double r = __longlong_as_double((long long)__ldcg(norms + 2 * prev_slot + 1));
    return converged(tol, d, r);
}

// FIX pass of the reduced step (first kernel of every oci_step in that form): CTA 0 also clears the norm slots
// and the grid-barrier counter the iteration launches of this step will use (saves two memsets per step).
__device__ __forceinline__ void clear_step_state(const DevView& V)
{
    if (blockIdx.x == 0) {
        for (int i = threadIdx.x; i < 2 * kNormSlots; i += blockDim.x) V.norms[i] = 0ull;
        if (threadIdx.x == 0) V.flags[8] = 0;
    }
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

// ---- packed interface layout of the reduced step (oci_reduced.cu has the definition)
// q < N  (mu < 0, leaves through the left face):  q = h*(N/2) + mm          (k run, then k+1/2 run)
// q >= N (mu > 0, leaves through the right face): q = N + (1-h)*(N/2) + mm  (k+1/2 run, then k run)
// so that the k+1/2 entries of a row are the single run [N/2, 3N/2).
__device__ __forceinline__ void unpack_q(int q, int N, int& half, int& h, int& mm)
{
    const int N2 = N >> 1;
    half = q >= N;
    const int r = q - half * N;
    const int second = r >= N2;
    mm = r - second * N2;
    h = half ? 1 - second : second;
}

__device__ __forceinline__ int pack_q(int half, int h, int mm, int N)
{
    const int N2 = N >> 1;
    return half * N + (half ? 1 - h : h) * N2 + mm;
}

__device__ __forceinline__ int o_row(int q, int N)   // full index 4m+s of packed outgoing row q
{
    int half, h, mm;
    unpack_q(q, N, half, h, mm);
    return 4 * (half * (N >> 1) + mm) + (half ? 2 * h + 1 : 2 * h);
}

// packed index of the mirror image (m -> N-1-m) of packed row q, same time slot
__device__ __forceinline__ int mirror_q(int q, int N)
{
    int half, h, mm;
    unpack_q(q, N, half, h, mm);
    return pack_q(1 - half, h, (N >> 1) - 1 - mm, N);
}

// First iteration index (1-based) whose norms satisfy the stopping rule, 0 if none of the `cnt` queued
// iterations did.  Slots past the last executed iteration are still zero from the memset, and
// converged(tol, 0, 0) holds for tol >= 0, so the scan must stop at the first hit.
__device__ __forceinline__ int first_converged(const unsigned long long* __restrict__ norms, int cnt, double tol)
{
    for (int i = 0; i < cnt; ++i) {
        const double d = __longlong_as_double((long long)__ldcg(norms + 2 * i + 0));
        const double r = __longlong_as_double((long long)__ldcg(norms + 2 * i + 1));
        if (converged(tol, d, r)) return i + 1;
    }
    return 0;
}

}  // namespace oci
