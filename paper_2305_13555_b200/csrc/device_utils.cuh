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
    return stop_now(tol, d, r);
}

// FIX pass of the reduced step (first kernel of every oci_step in that form): CTA 0 also clears the norm slots
// and the grid-barrier counter the iteration launches of this step will use (saves two memsets per step).
__device__ __forceinline__ void clear_step_state(const DevView& V)
{
    if (blockIdx.x == 0) {
        for (int i = threadIdx.x; i < 2 * kNormSlots; i += blockDim.x) V.norms[i] = 0ull;
        if (threadIdx.x == 0) {
            V.flags[8] = 0;                            // arrival counter of the grid-wide barrier
            V.flags[12] = 0;                           // ticket counter of the fused loops that hand out work dynamically
        }
    }
}

// a7, the host's side of a fused iteration loop: one thread of the grid calls this when the loop ends (converged, or all
// `cnt` iterations run) with the number of iterations run and the norms of the last one.  The values land in mapped host
// memory, the launch's sequence number last (system-scope fence in between), so the host learns the iteration count by
// polling a word instead of queueing a copy and synchronising a stream.
__device__ __forceinline__ void publish_step(const DevView& V, int iterations, int last_slot)
{
    if (V.host_pub == nullptr) return;
    volatile unsigned long long* h = V.host_pub;
    h[1] = (unsigned long long)iterations;
    h[2] = __ldcg(V.norms + 2 * last_slot + 0);
    h[3] = __ldcg(V.norms + 2 * last_slot + 1);
    __threadfence_system();
    h[0] = V.pub_seq;
}

// ---- shared-memory / mbarrier / TMA wrappers (one PTX instruction each), used by every TMA-fed kernel
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// non-blocking test of a phase (the predicate is consumed later, so the latency of the test overlaps other work)
__device__ __forceinline__ uint32_t mbar_test(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok;
}
// 1-D bulk TMA global -> shared, completion on an mbarrier (SASS UBLKCP)
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tma_load_1d_hint(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
                 : "memory");
}
// 2-D tensor-map TMA box global -> shared (SASS UTMALDG); c0 = column (inner), c1 = row of the box origin
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
// the same with an L2 cache policy (createpolicy): which operand should stay in L2 and which should stream
__device__ __forceinline__ void tma_load_2d_hint(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar, uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
            smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_last()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// 16-byte global load / store / L2 prefetch with an L2 eviction policy
__device__ __forceinline__ double2 ldg2_hint(const double* p, uint64_t policy)
{
    double2 r;
    asm volatile("ld.global.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(r.x), "=d"(r.y) : "l"(p), "l"(policy));
    return r;
}
__device__ __forceinline__ void stg2_hint(double* p, double2 v, uint64_t policy)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" ::"l"(p), "d"(v.x), "d"(v.y), "l"(policy) : "memory");
}
__device__ __forceinline__ void prefetch_l2_evict_last(const void* p) { asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(p)); }
// generic-proxy accesses of shared memory (LDS / STS) ordered before async-proxy ones (the TMA unit)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
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

// max of two values that are each non-negative (fabs applied) or NaN, taken on the bit patterns as integers:
// the pattern of a non-negative double is monotone in its value, +inf sorts above every finite number and NaN
// (0x7ff8...) above +inf, so a non-finite scalar flux reaches the host instead of being dropped the way fmax
// drops a NaN.  Integer compare + select also keeps these off the fp64 pipe the DMMAs run on.
__device__ __forceinline__ double nanmax(double a, double b)
{
    return __longlong_as_double(max(__double_as_longlong(a), __double_as_longlong(b)));
}

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
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

// The same under a warp-uniform predicate, and a predicated 8-byte shared-memory load: work that only some tiles
// need (the scalar-flux rows) without a branch, so that the surrounding DMMA stream stays one basic block and the
// compiler can software-pipeline the fragment loads across k-steps.
__device__ __forceinline__ void dmma_if(double& c0, double& c1, double a, double b, int pred)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.s32 p, %4, 0;\n"
        "@p mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
        "}\n"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b), "r"(pred));
}
__device__ __forceinline__ void lds_if(double& v, uint32_t saddr, int pred)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.s32 p, %2, 0;\n"
        "@p ld.shared.f64 %0, [%1];\n"
        "}\n"
        : "+d"(v)
        : "r"(saddr), "r"(pred));
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
        if (stop_now(tol, d, r)) return i + 1;
    }
    return 0;
}

}  // namespace oci
