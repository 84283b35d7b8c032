// Interface-reduced OCI step (oci_reduced.cu has the derivation), shared block, K2 = 2N in {32, 64}
// (n = 64, 128: configs 2 and 3): the fp64 tensor-core form of the three passes.
//
//   FIX  :  [yfix | phifix][j], ifix[j] = X [psi_{k-1/2}[j]; Q[j]]                      two row groups of X, K = K2+4
//   ITER :  [y^(l+1) | phi^(l+1)][j] = [yfix | phifix][j] + [G; H] inc^(l)[j]           (K2+8) x K2, rows padded
//   FINAL:  z[j] = ifix[j] + F inc^(L-1)[j]                                            K2 x K2
//
// At config 3 one iteration is 1.2 GFLOP against 0.2 GB of HBM traffic: the fp64 tensor pipe and HBM are
// equally loaded (arithmetic intensity 5.7 flop/B = the machine balance), so the design keeps both busy
// with the least synchronisation possible:
//
//   * one persistent CTA per SM, 8 warps, and EVERY WARP IS AN INDEPENDENT WORKER on tiles of 16 cells:
//     it owns all output rows of its cells, so there is no cross-warp reduction and no CTA barrier after
//     start-up (the scalar-flux rows are just one more n8 block of the same warp);
//   * the operator (39 KB for ITER, 74 KB for FIX at K2 = 64) lives in shared memory, rows padded to K2+4
//     doubles so that the DMMA fragment loads are bank-conflict free; per k-step a warp loads 2 A fragments
//     (cells) and NB B fragments (operator) for 2*NB DMMA.8x8x4;
//   * the input vectors need NO assembly: inc[j] = [y[j+1][0:N] | y[j-1][N:2N]] (|mu| is folded into the
//     operator) and psi_{k-1/2}[j] = four runs of N/2 doubles of y[j], z[j] (alpha folded into X), so each
//     lane issues 1-D bulk TMA copies (cp.async.bulk) straight into the warp's private two-stage ring; the
//     next tile is requested before the current one is computed;
//   * yfix / ifix / phifix / old phi are read straight from global memory in accumulator layout at the
//     start of the tile and only consumed in the epilogue (added to the accumulators, 16-byte stores).
#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int RT_M = 16;       // cells per warp tile
constexpr int RT_WARPS = 8;
constexpr int RT_STAGES = 2;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}


template <int K2, int PASS>
struct RCfg {
    static constexpr int KIN = PASS == PASS_FIX ? K2 + 4 : K2;          // operator columns (k extent)
    static constexpr int LD = K2 + 4;                                    // padded row (doubles): LD = 4 (mod 16)
    static constexpr int NB0 = PASS == PASS_FINAL ? K2 / 8 : K2 / 8 + 1; // n8 blocks of row group 0 (last = scalar flux)
    static constexpr int NB1 = PASS == PASS_FIX ? K2 / 8 : 0;            // row group 1 (FIX only: the I rows)
    static constexpr int KS = KIN / 4;
    static constexpr int OP_DOUBLES = (NB0 + NB1) * 8 * LD;
    static constexpr int STAGE_DOUBLES = RT_M * LD;
    static constexpr size_t SMEM = sizeof(double) * (OP_DOUBLES + RT_WARPS * RT_STAGES * STAGE_DOUBLES) +
                                   RT_WARPS * RT_STAGES * 8 + 16;
};

// acc[g][t] += A(cells 8g..8g+7) . Op(rows 8t..8t+7)^T over KS k-steps
template <int NB, int KS, int LD>
__device__ __forceinline__ void tile_dmma(double (&acc)[2][NB][2], const double* __restrict__ arow, const double* __restrict__ brow)
{
#pragma unroll 4
    for (int ks = 0; ks < KS; ++ks) {
        double a[2], b[NB];
#pragma unroll
        for (int g = 0; g < 2; ++g) a[g] = arow[(8 * g) * LD + 4 * ks];
#pragma unroll
        for (int t = 0; t < NB; ++t) b[t] = brow[(8 * t) * LD + 4 * ks];
#pragma unroll
        for (int g = 0; g < 2; ++g)
#pragma unroll
            for (int t = 0; t < NB; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
    }
}

}  // namespace

template <int K2, int PASS>
__global__ void __launch_bounds__(RT_WARPS * 32, 1)
oci_red_resident_kernel(DevView V, int ybase, int slot, int prev_slot, double tol, int cnt, int force)
{
    using C = RCfg<K2, PASS>;
    int ysrc = ybase;
    if (PASS == PASS_ITER) {
        if (step_done(V.norms, prev_slot, tol)) return;
    } else if (PASS == PASS_FINAL) {
        int L = first_converged(V.norms, cnt, tol);
        if (L == 0) {
            if (!force) return;
            L = cnt;
        }
        ysrc = (ybase + L - 1) & 1;
    }
    extern __shared__ __align__(128) unsigned char smem_raw[];
    double* op_s = reinterpret_cast<double*>(smem_raw);                         // [(NB0+NB1)*8][LD]
    double* ring = op_s + C::OP_DOUBLES;                                        // [warps][stages][RT_M][LD]
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + RT_WARPS * RT_STAGES * C::STAGE_DOUBLES);

    constexpr int N = K2 / 2, N2 = K2 / 4;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g4 = lane >> 2, t4 = lane & 3;
    const int64_t J = V.J;
    const double* __restrict__ Ys = V.y[ysrc];
    double* __restrict__ Yd = V.y[ysrc ^ 1];

    // operator -> shared memory.  FIX: X rows [O | I | phi] are regrouped as [O | phi | I]
    {
        const double* __restrict__ src = PASS == PASS_FIX ? V.xop : PASS == PASS_ITER ? V.rop : V.fop;
        constexpr int GLD = PASS == PASS_FIX ? K2 + 16 : K2;
        constexpr int C2 = C::KIN / 2;
        for (int e = tid; e < (C::NB0 + C::NB1) * 8 * C2; e += RT_WARPS * 32) {
            const int r = e / C2, c2 = e - r * C2;
            int gr = r;
            if (PASS == PASS_FIX) gr = r < K2 ? r : (r < K2 + 8 ? r + K2 : r - 8);
            *reinterpret_cast<double2*>(op_s + r * C::LD + 2 * c2) = *reinterpret_cast<const double2*>(src + (size_t)gr * GLD + 2 * c2);
        }
    }
    if (lane == 0) {
        for (int s = 0; s < RT_STAGES; ++s) mbar_init(&full[warp * RT_STAGES + s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int64_t ntiles = (J + RT_M - 1) / RT_M;
    const int64_t wid = (int64_t)blockIdx.x * RT_WARPS + warp, nw = (int64_t)gridDim.x * RT_WARPS;
    const int my_tiles = wid < ntiles ? (int)((ntiles - wid + nw - 1) / nw) : 0;
    double* my_ring = ring + warp * RT_STAGES * C::STAGE_DOUBLES;
    uint64_t* my_full = full + warp * RT_STAGES;

    // bulk copies, one per lane and round.  ITER / FINAL: lanes 0..15 the first half of y[j+1] (mu<0 leaves
    // cell j+1 through its left face), lanes 16..31 the second half of y[j-1].  FIX: the four h = 1 runs of
    // y[j], z[j] and Q[j]
    auto prefetch = [&](int it) {
        const int s = it & 1;
        const int64_t j0 = (wid + (int64_t)it * nw) * RT_M;
        const int rows = (int)((J - j0 < RT_M) ? (J - j0) : RT_M);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        if (lane == 0) mbar_expect_tx(&my_full[s], (uint32_t)rows * C::KIN * 8);
        __syncwarp();
        double* st = my_ring + s * C::STAGE_DOUBLES;
        if (PASS == PASS_FIX) {
            for (int idx = lane; idx < 5 * RT_M; idx += 32) {
                const int row = idx & (RT_M - 1), seg = idx / RT_M;
                if (row < rows) {
                    const int64_t j = j0 + row;
                    const double* src = seg == 0   ? Ys + j * K2 + N2
                                        : seg == 1 ? Ys + j * K2 + N + N2
                                        : seg == 2 ? V.z + j * K2 + N2
                                        : seg == 3 ? V.z + j * K2 + N + N2
                                                   : V.Q + j * 4;
                    tma_load_1d(st + row * C::LD + seg * N2, src, seg == 4 ? 32 : N2 * 8, &my_full[s]);
                }
            }
        } else {
            const int row = lane & 15, half = lane >> 4;
            if (row < rows) {
                const int64_t j = j0 + row;
                const double* src = half ? Ys + (j - 1) * K2 + N : Ys + (j + 1) * K2;
                tma_load_1d(st + row * C::LD + half * N, src, N * 8, &my_full[s]);
            }
        }
    };

    double dmax = 0.0, rmax = 0.0;
    if (my_tiles > 0) prefetch(0);

    for (int it = 0; it < my_tiles; ++it) {
        const int s = it & 1;
        const int64_t j0 = (wid + (int64_t)it * nw) * RT_M;
        const int rows = (int)((J - j0 < RT_M) ? (J - j0) : RT_M);
        if (it + 1 < my_tiles) prefetch(it + 1);

        // ---- global operands of the epilogue, requested now, consumed after the DMMAs
        double2 fx[2][PASS == PASS_FIX ? 1 : K2 / 8];
        double2 pf[2], po[2];
        if (PASS != PASS_FIX) {
            const double* __restrict__ fixp = PASS == PASS_FINAL ? V.ifix : V.yfix;
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                const int r = 8 * g + g4;
                const int64_t j = (r < rows) ? j0 + r : j0;             // clamped: unconditional loads
#pragma unroll
                for (int t = 0; t < K2 / 8; ++t) fx[g][t] = *reinterpret_cast<const double2*>(fixp + j * K2 + 8 * t + 2 * t4);
                if (PASS == PASS_ITER) {
                    pf[g] = *reinterpret_cast<const double2*>(V.phifix + j * 4 + 2 * (t4 & 1));
                    po[g] = *reinterpret_cast<const double2*>(V.phi + j * 4 + 2 * (t4 & 1));
                }
            }
        }

        double acc[2][C::NB0][2];
#pragma unroll
        for (int g = 0; g < 2; ++g)
#pragma unroll
            for (int t = 0; t < C::NB0; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;

        mbar_wait(&my_full[s], (it >> 1) & 1);
        const double* arow = my_ring + s * C::STAGE_DOUBLES + g4 * C::LD + t4;
        const double* brow = op_s + g4 * C::LD + t4;
        tile_dmma<C::NB0, C::KS, C::LD>(acc, arow, brow);

        // ---- epilogue of row group 0
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            const int r = 8 * g + g4;
            const int64_t j = j0 + r;
            if (r < rows) {
                if (PASS == PASS_ITER) {
#pragma unroll
                    for (int t = 0; t < K2 / 8; ++t)
                        *reinterpret_cast<double2*>(Yd + j * K2 + 8 * t + 2 * t4) =
                            make_double2(fx[g][t].x + acc[g][t][0], fx[g][t].y + acc[g][t][1]);
                    if (t4 < 2) {                                   // phi rows: columns 0..3 of the last block
                        const double p0 = pf[g].x + acc[g][C::NB0 - 1][0], p1 = pf[g].y + acc[g][C::NB0 - 1][1];
                        *reinterpret_cast<double2*>(V.phi + j * 4 + 2 * t4) = make_double2(p0, p1);
                        dmax = fmax(dmax, fmax(fabs(p0 - po[g].x), fabs(p1 - po[g].y)));
                        rmax = fmax(rmax, fmax(fabs(p0), fabs(p1)));
                    }
                } else if (PASS == PASS_FINAL) {
#pragma unroll
                    for (int t = 0; t < K2 / 8; ++t)
                        *reinterpret_cast<double2*>(V.z + j * K2 + 8 * t + 2 * t4) =
                            make_double2(fx[g][t].x + acc[g][t][0], fx[g][t].y + acc[g][t][1]);
                } else {
#pragma unroll
                    for (int t = 0; t < K2 / 8; ++t)
                        *reinterpret_cast<double2*>(V.yfix + j * K2 + 8 * t + 2 * t4) = make_double2(acc[g][t][0], acc[g][t][1]);
                    if (t4 < 2)
                        *reinterpret_cast<double2*>(V.phifix + j * 4 + 2 * t4) =
                            make_double2(acc[g][C::NB0 - 1][0], acc[g][C::NB0 - 1][1]);
                }
            }
        }
        if (PASS == PASS_FIX) {
            // ---- row group 1: the I rows of Psi_fix from the same input tile
            double acc1[2][C::NB1 > 0 ? C::NB1 : 1][2];
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int t = 0; t < C::NB1; ++t) acc1[g][t][0] = acc1[g][t][1] = 0.0;
            tile_dmma<(C::NB1 > 0 ? C::NB1 : 1), C::KS, C::LD>(acc1, arow, brow + C::NB0 * 8 * C::LD);
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                const int r = 8 * g + g4;
                const int64_t j = j0 + r;
                if (r < rows) {
#pragma unroll
                    for (int t = 0; t < C::NB1; ++t)
                        *reinterpret_cast<double2*>(V.ifix + j * K2 + 8 * t + 2 * t4) = make_double2(acc1[g][t][0], acc1[g][t][1]);
                }
            }
        }
        __syncwarp();
        // ---- reflecting ghost rows of y (reading S4) by the warp that owns the edge cell
        if (PASS == PASS_ITER) {
            const bool gl = j0 == 0 && V.bcL == OCI_BC_REFLECTING;
            const bool gr = j0 + rows == J && V.bcR == OCI_BC_REFLECTING;
            if (gl || gr) {
                __threadfence_block();
                for (int q = lane; q < K2; q += 32) {
                    const int mir = mirror_q(q, N);
                    if (gl && q >= N) Yd[-(int64_t)K2 + q] = __ldcg(Yd + mir);
                    if (gr && q < N) Yd[J * K2 + q] = __ldcg(Yd + (J - 1) * K2 + mir);
                }
                __syncwarp();
            }
        }
    }
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0 && my_tiles > 0) {
            atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
        }
    }
}

bool oci_red_resident_supported(const DevView& V) { return V.nblk == 1 && (V.n == 128 || V.n == 64); }

namespace {
template <int K2, int PASS>
void launch_rr(const DevView& V, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    static int sm_count = 0;
    static bool attr = false;
    if (sm_count == 0) {
        int dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
    }
    if (!attr) {
        cudaFuncSetAttribute(oci_red_resident_kernel<K2, PASS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)RCfg<K2, PASS>::SMEM);
        attr = true;
    }
    const int64_t ntiles = (V.J + RT_M - 1) / RT_M;
    const int64_t ctas = (ntiles + RT_WARPS - 1) / RT_WARPS;
    const unsigned grid = (unsigned)(ctas < sm_count ? ctas : sm_count);
    oci_red_resident_kernel<K2, PASS><<<grid, RT_WARPS * 32, RCfg<K2, PASS>::SMEM, s>>>(V, ybase, slot, prev_slot, tol, cnt, force);
}

template <int K2>
void launch_rr_pass(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    if (pass == PASS_FIX) launch_rr<K2, PASS_FIX>(V, ybase, 0, -1, tol, 0, 0, s);
    else if (pass == PASS_ITER) launch_rr<K2, PASS_ITER>(V, ybase, slot, prev_slot, tol, 0, 0, s);
    else launch_rr<K2, PASS_FINAL>(V, ybase, 0, -1, tol, cnt, force, s);
}
}  // namespace

int launch_red_resident(const DevView& V, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                        cudaStream_t s)
{
    if (V.n == 128) launch_rr_pass<64>(V, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    else launch_rr_pass<32>(V, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    return 1;
}

}  // namespace oci
