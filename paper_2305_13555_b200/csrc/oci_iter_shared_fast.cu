// Kernel (b)+(c), shared-block fast path for block sizes n = 4N in {64, 128} ("resident" form).
//
// Psi^(l+1)[j] = B^{-1} c[j] for all cells is the dense contraction [J x n] = [J x n].[n x n]^T
// (eq. 19, one inverse for the whole slab).  On sm_100a the fp64 tensor pipe is reached only
// by mma.sync DMMA.8x8x4 (tcgen05 has no f64 kind), one instruction per 16 clk per SM sub-partition,
// so the issue slots are nearly free and the design goal is to keep that pipe fed:
//
//   * one persistent CTA per SM, 8 MMA warps + 4 auxiliary warps; MMA warp w owns output rows [n/8*w, n/8*(w+1)) and keeps its
//     slice of B^{-1} as DMMA B-fragments IN REGISTERS for the whole kernel (n=128: 64 doubles per
//     thread) - the inverse is read from L2 once per CTA per launch and never touches shared memory;
//   * cell tiles of 32 stream through a 2-stage shared-memory ring filled by 1-D bulk TMA
//     (cp.async.bulk + mbarrier complete_tx): per cell the c_fix row and the two neighbour half-rows
//     the RHS needs (rows a3: first half of Psi^(l)[j+1], second half of Psi^(l)[j-1]; ghost rows make
//     the domain edges look like neighbours);
//   * the RHS (row a4) is assembled in place in shared memory, c = c_fix + coef * psi_nbr[k^1], only on
//     the 2N rows that take an incident flux; rows are padded to stride = 4 (mod 16) doubles so the
//     A-fragment loads are bank-conflict free;
//   * epilogue: accumulators -> global Psi^(l+1) (16-byte stores), the scalar flux (eq. 18) reduced
//     across lanes by shuffle and across warps through shared memory, the two max-norms by atomicMax
//     (row a6), and the reflecting ghost rows (reading S4) - no second pass over Psi.
#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int TM = 32;        // cells per tile
constexpr int STAGES = 2;

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
// 1-D bulk TMA global -> shared, completion on an mbarrier (SASS UBLKCP)
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

template <int NT>
struct Cfg {
    static constexpr int LD = NT + 4;                 // padded row (doubles): LD = 4 (mod 16)
    static constexpr int KS = NT / 4;                 // k-steps of 4
    static constexpr int NB = NT / 64;                // n8 blocks per warp (8 warps)
    static constexpr int STAGE_DOUBLES = 2 * TM * LD; // c_fix tile + neighbour tile
    static constexpr size_t SMEM = sizeof(double) * (STAGES * STAGE_DOUBLES + STAGES * 8 * TM * 4) + 3 * STAGES * 8 + 64;
};

}  // namespace

// Warp roles: warps 0..7 = MMA warps (two warpgroups, 224 registers each after setmaxnreg);
// warps 8..11 = auxiliary warpgroup (56 registers): TMA issue, RHS assembly, phi / norms / ghost rows.
// Hand-offs are mbarriers only (no __syncthreads in the steady state):
//   full[s]   TMA bytes of stage s have landed            (1 arrival + tx bytes)   aux waits
//   cready[s] RHS of stage s assembled                    (128 aux arrivals)       MMA warps wait
//   freeb[s]  MMA warps are done with stage s: RHS read, Psi^(l+1) stored, phi partials written
//                                                         (8 arrivals, one per MMA warp)  aux waits
template <int NT>
__global__ void __launch_bounds__(384, 1)
oci_iter_resident_kernel(DevView V, int src, int slot, int prev_slot, double tol)
{
    using C = Cfg<NT>;
    if (step_done(V.norms, prev_slot, tol)) return;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* stage_base = reinterpret_cast<double*>(smem_raw);
    double* phi_part = stage_base + STAGES * C::STAGE_DOUBLES;                     // [STAGES][8 warps][TM][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(phi_part + STAGES * 8 * TM * 4);  // [STAGES]
    uint64_t* cready = full + STAGES;
    uint64_t* freeb = cready + STAGES;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int N = NT / 4, HALF = NT / 2;
    const int64_t J = V.J;
    const double* __restrict__ Pold = V.psi[src];
    double* __restrict__ Pnew = V.psi[src ^ 1];
    const int64_t ntiles = (J + TM - 1) / TM;
    const int my_tiles = (int)((ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x);   // >= 1

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&cready[s], 128);
            mbar_init(&freeb[s], 8);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= 8) {
        // =========================== auxiliary warpgroup ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        const int atid = tid - 256;
        const double* __restrict__ cfix = V.cfix;
        auto issue = [&](int it) {   // warp 8 only: one cell row per lane
            const int st = it % STAGES;
            const int64_t j0 = ((int64_t)blockIdx.x + (int64_t)it * gridDim.x) * TM;
            const int rows = (int)((J - j0 < TM) ? (J - j0) : TM);
            double* cs = stage_base + st * C::STAGE_DOUBLES;
            double* ps = cs + TM * C::LD;
            if (lane == 0) mbar_expect_tx(&full[st], (uint32_t)rows * NT * 16u);
            __syncwarp();
            if (lane < rows) {
                const int64_t j = j0 + lane;
                tma_load_1d(cs + lane * C::LD, cfix + j * NT, NT * 8, &full[st]);
                tma_load_1d(ps + lane * C::LD, Pold + (j + 1) * NT, HALF * 8, &full[st]);                // k < n/2: from j+1
                tma_load_1d(ps + lane * C::LD + HALF, Pold + (j - 1) * NT + HALF, HALF * 8, &full[st]);  // k >= n/2: from j-1
            }
        };
        if (warp == 8)
            for (int it = 0; it < STAGES && it < my_tiles; ++it) issue(it);

        // this thread always patches the same RHS row k_a (one of the 2N rows that take an incident flux)
        const int a_idx = atid & (HALF - 1);
        const int a_m = a_idx >> 1;
        const int k_a = 4 * a_m + ((a_m < N / 2) ? 1 + 2 * (a_idx & 1) : 2 * (a_idx & 1));
        const double coef_a = V.coef[k_a];
        constexpr int ROWS_PER_PASS = 128 / HALF;
        const int r_a = atid / HALF;
        double dmax = 0.0, rmax = 0.0;

        // phi (eq. 18), max-norms, ghost rows for the tile of CTA-iteration `it` (after the MMA warps released it)
        auto finalize = [&](int it) {
            const int st = it % STAGES;
            const int64_t tile = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
            const int64_t j0 = tile * TM;
            const int rows = (int)((J - j0 < TM) ? (J - j0) : TM);
            const int r = atid >> 2;
            if (r < rows) {
                const double* pp = phi_part + (size_t)st * 8 * TM * 4;
                double s = 0.0;
#pragma unroll
                for (int w8 = 0; w8 < 8; ++w8) s += pp[(w8 * TM + r) * 4 + (atid & 3)];
                const int64_t idx = (j0 + r) * 4 + (atid & 3);
                const double old = V.phi[idx];
                V.phi[idx] = s;
                dmax = fmax(dmax, fabs(s - old));
                rmax = fmax(rmax, fabs(s));
            }
            if (tile == 0 && V.bcL == OCI_BC_REFLECTING) {
                for (int idx = atid; idx < NT; idx += 128) {
                    const int m = idx >> 2, s = idx & 3;
                    if (m >= N / 2 && (s & 1)) Pnew[-(int64_t)NT + idx] = __ldcg(Pnew + 4 * (N - 1 - m) + (s - 1));
                }
            }
            if (tile == ntiles - 1 && V.bcR == OCI_BC_REFLECTING) {
                for (int idx = atid; idx < NT; idx += 128) {
                    const int m = idx >> 2, s = idx & 3;
                    if (m < N / 2 && !(s & 1)) Pnew[J * NT + idx] = __ldcg(Pnew + (J - 1) * NT + 4 * (N - 1 - m) + (s + 1));
                }
            }
        };

        for (int it = 0; it < my_tiles; ++it) {
            const int st = it % STAGES;
            const uint32_t parity = (it / STAGES) & 1;
            const int64_t j0 = ((int64_t)blockIdx.x + (int64_t)it * gridDim.x) * TM;
            const int rows = (int)((J - j0 < TM) ? (J - j0) : TM);
            double* cs = stage_base + st * C::STAGE_DOUBLES;
            double* ps = cs + TM * C::LD;
            mbar_wait(&full[st], parity);
            // a4: c = c_fix + coef * psi_nbr[k^1], in place
#pragma unroll 4
            for (int r = r_a; r < TM; r += ROWS_PER_PASS)
                if (r < rows) cs[r * C::LD + k_a] = fma(coef_a, ps[r * C::LD + (k_a ^ 1)], cs[r * C::LD + k_a]);
            mbar_arrive(&cready[st]);
            // previous tile: release its stage to the TMA, then reduce its scalar flux
            if (it >= 1) {
                const int sp = (it - 1) % STAGES;
                mbar_wait(&freeb[sp], ((it - 1) / STAGES) & 1);
                if (warp == 8 && it - 1 + STAGES < my_tiles) {
                    fence_proxy_async();
                    issue(it - 1 + STAGES);
                }
                finalize(it - 1);
            }
        }
        mbar_wait(&freeb[(my_tiles - 1) % STAGES], ((my_tiles - 1) / STAGES) & 1);
        finalize(my_tiles - 1);
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) {
            atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
        }
    } else {
        // =========================== MMA warps ===========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
        const int g4 = lane >> 2, t4 = lane & 3;
        // this warp's slice of B^{-1} as B-fragments: b[ks][t] = Binv[warp*8*NB + 8t + g4][4ks + t4]
        double bfr[C::KS][C::NB];
        {
            const double* __restrict__ Bw = V.binv + (size_t)(warp * 8 * C::NB + g4) * NT + t4;
#pragma unroll
            for (int ks = 0; ks < C::KS; ++ks)
#pragma unroll
                for (int t = 0; t < C::NB; ++t) bfr[ks][t] = __ldg(Bw + (size_t)(8 * t) * NT + 4 * ks);
        }
        double wq[C::NB];   // quadrature weights of the angles this lane's accumulators belong to
#pragma unroll
        for (int t = 0; t < C::NB; ++t) wq[t] = V.w[(warp * 8 * C::NB + 8 * t + 2 * t4) >> 2];

        for (int it = 0; it < my_tiles; ++it) {
            const int st = it % STAGES;
            const uint32_t parity = (it / STAGES) & 1;
            const int64_t j0 = ((int64_t)blockIdx.x + (int64_t)it * gridDim.x) * TM;
            const int rows = (int)((J - j0 < TM) ? (J - j0) : TM);
            const double* cs = stage_base + st * C::STAGE_DOUBLES;
            double* pp = phi_part + (size_t)st * 8 * TM * 4;
            mbar_wait(&cready[st], parity);

            // a5: D[cell][i] += c[cell][k] * Binv[i][k]
            double acc[4][C::NB][2];
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int t = 0; t < C::NB; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;
            const double* arow = cs + g4 * C::LD + t4;
#pragma unroll
            for (int ks = 0; ks < C::KS; ++ks) {
                double a[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) a[g] = arow[(8 * g) * C::LD + 4 * ks];
#pragma unroll
                for (int g = 0; g < 4; ++g)
#pragma unroll
                    for (int t = 0; t < C::NB; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], bfr[ks][t]);
            }
            // epilogue: Psi^(l+1) and this warp's partial scalar flux
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                const int r = 8 * g + g4;
                double p0 = 0.0, p1 = 0.0;
#pragma unroll
                for (int t = 0; t < C::NB; ++t) {
                    if (r < rows)
                        *reinterpret_cast<double2*>(Pnew + (j0 + r) * NT + warp * 8 * C::NB + 8 * t + 2 * t4) =
                            make_double2(acc[g][t][0], acc[g][t][1]);
                    p0 = fma(wq[t], acc[g][t][0], p0);
                    p1 = fma(wq[t], acc[g][t][1], p1);
                }
                // lanes t4 and t4^2 hold the same slots (s = 2*(t4&1) + {0,1}) of neighbouring angles
                p0 += __shfl_xor_sync(0xffffffffu, p0, 2);
                p1 += __shfl_xor_sync(0xffffffffu, p1, 2);
                if (t4 < 2) {
                    pp[(warp * TM + r) * 4 + 2 * t4 + 0] = p0;
                    pp[(warp * TM + r) * 4 + 2 * t4 + 1] = p1;
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&freeb[st]);
        }
    }
}

bool oci_shared_fast_supported(const DevView& V) { return V.nblk == 1 && (V.n == 128 || V.n == 64); }

int launch_oci_shared_fast(const DevView& V, int src, int slot, int prev_slot, double tol, cudaStream_t s)
{
    static int sm_count = 0;
    if (sm_count == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
    }
    const int64_t ntiles = (V.J + TM - 1) / TM;
    const unsigned grid = (unsigned)(ntiles < sm_count ? ntiles : sm_count);
    if (V.n == 128) {
        static bool attr = false;
        if (!attr) {
            cudaFuncSetAttribute(oci_iter_resident_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<128>::SMEM);
            attr = true;
        }
        oci_iter_resident_kernel<128><<<grid, 384, Cfg<128>::SMEM, s>>>(V, src, slot, prev_slot, tol);
    } else {
        static bool attr = false;
        if (!attr) {
            cudaFuncSetAttribute(oci_iter_resident_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg<64>::SMEM);
            attr = true;
        }
        oci_iter_resident_kernel<64><<<grid, 384, Cfg<64>::SMEM, s>>>(V, src, slot, prev_slot, tol);
    }
    return 1;
}

}  // namespace oci
