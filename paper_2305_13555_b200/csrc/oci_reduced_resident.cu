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
//     start-up (the scalar-flux rows are just one more n8 block of the same warp); the warps of a CTA claim its
//     tiles from a counter in shared memory, so that a warp whose tiles run slow takes fewer of them;
//   * the operator (39 KB for ITER, 74 KB for FIX at K2 = 64) lives in shared memory, rows padded to K2+4
//     doubles so that the DMMA fragment loads are bank-conflict free; per k-step a warp loads 2 A fragments
//     (cells) and NB B fragments (operator) for 2*NB DMMA.8x8x4;
//   * the input vectors need NO assembly (|mu|, alpha, h/4 are folded into the operators) and arrive as
//     tensor-map TMA boxes issued by one lane into the warp's private two-stage ring, the next tile
//     requested before the current one is computed.  ITER / FINAL: inc[j] = [y[j+1][0:N] | y[j-1][N:2N]], so
//     a tile of 16 cells is ONE box of the 18 whole rows j0-1 .. j0+16 of y; the box is 4 columns wider than
//     the array (zero filled), which gives the padded, bank-conflict-free row pitch for free.  FIX:
//     psi_{k-1/2}[j] = the k+1/2 runs y[j][N/2:3N/2], z[j][N/2:3N/2]: two boxes of N+4 columns, plus Q;
//   * yfix / ifix / phifix / old phi are read straight from global memory in accumulator layout at the
//     start of the tile and only consumed in the epilogue (added to the accumulators, 16-byte stores).
#include <cuda.h>

#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int RT_M = 16;       // cells per warp tile
constexpr int RT_WARPS = 8;
constexpr int RT_STAGES = 2;

template <int K2, int PASS>
struct RCfg {
    static constexpr int N = K2 / 2;
    static constexpr int LD = K2 + 4;                                    // operator row pitch (doubles): LD = 4 (mod 16)
    static constexpr int LDH = N + 4;                                    // FIX: pitch of the y / z half-row boxes
    static constexpr int NSL = K2 / 8;                                   // n8 output blocks ("slices") of y / z / yfix / ifix
    static constexpr int NB0 = PASS == PASS_FINAL ? NSL : NSL + 1;       // blocks of row group 0 (last = scalar flux)
    static constexpr int NB1 = PASS == PASS_FIX ? NSL : 0;               // row group 1 (FIX only: the I rows)
    static constexpr int KIN = PASS == PASS_FIX ? K2 + 4 : K2;           // operator columns
    static constexpr int KS = KIN / 4;                                   // k-steps of one phase
    static constexpr int DIST = K2 / 16;                                 // pipelined epilogue: load-to-use distance (k-steps)
    static constexpr int OP_DOUBLES = (NB0 + NB1) * 8 * LD;
    // stage: ITER / FINAL [18][LD] (rows j0-1 .. j0+16 of y); FIX [16][LDH] y | [16][LDH] z | [16][4] Q
    static constexpr int STAGE_BYTES_RAW = PASS == PASS_FIX ? (2 * RT_M * LDH + RT_M * 4) * 8 : (RT_M + 2) * LD * 8;
    static constexpr int STAGE_BYTES = (STAGE_BYTES_RAW + 127) / 128 * 128;
    static constexpr int TX_BYTES = STAGE_BYTES_RAW;                     // a box always delivers all its bytes (zero fill)
    static constexpr size_t SMEM = 128 + sizeof(double) * OP_DOUBLES + (size_t)RT_WARPS * RT_STAGES * STAGE_BYTES +
                                   (RT_WARPS * RT_STAGES + 1) * 8 + 16;
    static_assert((OP_DOUBLES * 8) % 128 == 0, "ring must stay 128-byte aligned");
};

// what a finished accumulator tile still owes: its epilogue, drained during the NEXT phase's DMMA stream
enum { PK_ITER = 0, PK_FINAL = 1, PK_FIX0 = 2, PK_FIX1 = 3 };

// A-fragment element of k-step ks, cell block g, for this lane (pa = stage + lane offset; see the kernel)
template <int K2, int PASS>
__device__ __forceinline__ double a_frag(const double* __restrict__ pa, const double* __restrict__ pq, int ks, int g)
{
    using C = RCfg<K2, PASS>;
    constexpr int N = K2 / 2;
    if (PASS == PASS_FIX) {
        if (ks < N / 4) return pa[(8 * g) * C::LDH + 4 * ks];                            // y half rows
        if (ks < N / 2) return pa[(RT_M + 8 * g) * C::LDH + 4 * (ks - N / 4)];           // z half rows
        return pq[(8 * g) * 4];                                                          // Q
    }
    // cell r of the tile: k < N from y row r+2 (cell j+1), k >= N from y row r (cell j-1)
    return pa[(8 * g + (ks < N / 4 ? 2 : 0)) * C::LD + 4 * ks];
}

// Where a pending epilogue reads and writes (per kernel launch).
struct EpiCtx {
    const double* __restrict__ fixp;   // additive operand (yfix for ITER, ifix for FINAL)
    double* __restrict__ out;          // y[dst] (ITER), z (FINAL), yfix (FIX0), ifix (FIX1)
    const double* __restrict__ phifix;
    double* __restrict__ phi;
    double* __restrict__ phifix_out;
    uint64_t pol_keep;                 // L2 policy of the additive operand (re-read every iteration: evict_last)
    uint64_t pol_out;                  // L2 policy of the FIX pass's stores (yfix: evict_last, ifix: evict_first)
};

// One phase = all k-steps of one row group of one tile (NBC n8 blocks, accumulators acc) with the epilogue of
// the PREVIOUS phase (pend, NBP blocks, cells pj0 .. pj0+prows-1) drained between the DMMAs one slice per
// k-step: its loads are issued DIST k-steps before they are needed and its 16-byte stores are spread out, so
// the warp never leaves the DMMA stream for a burst of memory instructions.  MMA = false: drain only.
template <int K2, int PASS, int NBC, int NBP, int PK, bool MMA>
__device__ __forceinline__ void phase(double (&acc)[2][NBC][2], const double* __restrict__ pa, const double* __restrict__ pq,
                                      const double* __restrict__ brow, const double (&pend)[2][NBP][2], int64_t pj0, int prows,
                                      const EpiCtx& E, int g4, int t4, double& dmax, double& rmax)
{
    using C = RCfg<K2, PASS>;
    constexpr int NSL = C::NSL, KS = C::KS;
    constexpr bool LOADS = PK == PK_ITER || PK == PK_FINAL;
    constexpr int DIST = LOADS ? C::DIST : 0;
    double2 fxw[NSL][2];
    double2 pf[2], po[2];
    int64_t pj[2];
    bool ok[2];
#pragma unroll
    for (int g = 0; g < 2; ++g) {
        const int r = 8 * g + g4;
        ok[g] = r < prows;
        pj[g] = pj0 + (ok[g] ? r : 0);                     // clamped: unconditional loads
    }
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
        if (MMA) {
            double a[2], b[NBC];
#pragma unroll
            for (int g = 0; g < 2; ++g) a[g] = a_frag<K2, PASS>(pa, pq, ks, g);
#pragma unroll
            for (int t = 0; t < NBC; ++t) b[t] = brow[(8 * t) * C::LD + 4 * ks];
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int t = 0; t < NBC; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
        }
        // ---- pending epilogue: loads of slice ks
        if (LOADS && ks < NSL) {
#pragma unroll
            for (int g = 0; g < 2; ++g) fxw[ks][g] = ldg2_hint(E.fixp + pj[g] * K2 + 8 * ks + 2 * t4, E.pol_keep);
        }
        // (requested at the first k-step, together with slice 0: measured 5 % faster at config 3 than requesting them
        // after the last slice - fewer groups of loads in flight at a time for the six scoreboards)
        if (PK == PK_ITER && ks == 0) {
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                pf[g] = *reinterpret_cast<const double2*>(E.phifix + pj[g] * 4 + 2 * (t4 & 1));
                po[g] = __ldcg(reinterpret_cast<const double2*>(E.phi + pj[g] * 4 + 2 * (t4 & 1)));   // rewritten every iteration: L2
            }
        }
        // ---- pending epilogue: slice ks - DIST is added and stored
        const int t = ks - DIST;
        if (t >= 0 && t < NSL) {
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                double2 v = make_double2(pend[g][t][0], pend[g][t][1]);
                if (LOADS) { v.x += fxw[t][g].x; v.y += fxw[t][g].y; }
                if (ok[g]) {
                    if (LOADS) *reinterpret_cast<double2*>(E.out + pj[g] * K2 + 8 * t + 2 * t4) = v;
                    else stg2_hint(E.out + pj[g] * K2 + 8 * t + 2 * t4, v, E.pol_out);
                }
            }
        }
        if ((PK == PK_ITER || PK == PK_FIX0) && ks == NSL + DIST) {     // scalar-flux block: columns 0..3 of block NSL
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                if (ok[g] && t4 < 2) {
                    if (PK == PK_ITER) {
                        const double p0 = pf[g].x + pend[g][NBP - 1][0], p1 = pf[g].y + pend[g][NBP - 1][1];
                        *reinterpret_cast<double2*>(E.phi + pj[g] * 4 + 2 * t4) = make_double2(p0, p1);
                        dmax = nanmax(dmax, nanmax(fabs(p0 - po[g].x), fabs(p1 - po[g].y)));
                        rmax = nanmax(rmax, nanmax(fabs(p0), fabs(p1)));
                    } else {
                        *reinterpret_cast<double2*>(E.phifix_out + pj[g] * 4 + 2 * t4) = make_double2(pend[g][NBP - 1][0], pend[g][NBP - 1][1]);
                    }
                }
            }
        }
    }
}

}  // namespace

template <int K2, int PASS>
__global__ void __launch_bounds__(RT_WARPS * 32, 1)
oci_red_resident_kernel(DevView V, const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_a_alt,
                        const __grid_constant__ CUtensorMap map_z, const __grid_constant__ CUtensorMap map_q,
                        const __grid_constant__ CUtensorMap map_op, const __grid_constant__ CUtensorMap map_op2, int ybase, int slot,
                        int prev_slot, double tol, int cnt, int force)
{
    // map_a: tensor map of y[ybase] (whole-row boxes for ITER / FINAL, half-row boxes for FIX), map_a_alt: of
    // y[ybase ^ 1]; map_op (+ map_op2 for the scalar-flux rows of X): the operator as boxes of padded rows
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
    // ITER: `cnt` iterations run inside this one (cooperative) launch, separated by a grid-wide barrier; iteration l
    // reads y[(ybase + l) & 1], reports its norms in slot `slot + l`, and the loop ends at the first converged one
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;
    if (PASS == PASS_FIX) clear_step_state(V);

    extern __shared__ unsigned char smem_raw[];
    // aligned up inside the shared window (pointer arithmetic on the array keeps the LDS/STS address space)
    unsigned char* sbase = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    double* op_s = reinterpret_cast<double*>(sbase);                            // [(NB0+NB1)*8][LD]
    unsigned char* ring = sbase + sizeof(double) * C::OP_DOUBLES;               // [warps][stages][STAGE_BYTES]
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + (size_t)RT_WARPS * RT_STAGES * C::STAGE_BYTES);
    uint64_t* op_bar = full + RT_WARPS * RT_STAGES;

    constexpr int N = K2 / 2, N2 = K2 / 4;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int g4 = lane >> 2, t4 = lane & 3;
    const int64_t J = V.J;

    const int64_t ntiles = (J + RT_M - 1) / RT_M;
    // CTA b owns the tiles b, b + grid, b + 2 grid, ... (a small problem spreads over all SMs, and the grid sweeps the
    // slab front to back); its warps CLAIM them one at a time from a counter in shared memory, one tile ahead of the one
    // they compute: the time a tile takes varies by +-10 % between the warps of an SM (measured), and with a fixed
    // seven tiles per warp an iteration lasts as long as its unluckiest warp
    __shared__ int tile_ctr;
    const int Mcta = (int64_t)blockIdx.x < ntiles ? (int)((ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0;
    unsigned char* my_ring = ring + (size_t)warp * RT_STAGES * C::STAGE_BYTES;
    uint64_t* my_full = full + warp * RT_STAGES;

    if (tid == 0) {
        tile_ctr = 0;
        for (int s = 0; s < RT_WARPS * RT_STAGES; ++s) mbar_init(&full[s], 1);
        mbar_init(op_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // the operator: one to three boxes of padded rows.  FIX: X rows [O | I | phi] land regrouped as [O | phi | I]
    if (tid == 0) {
        mbar_expect_tx(op_bar, C::OP_DOUBLES * 8);
        if (PASS == PASS_FIX) {
            tma_load_2d(op_s, &map_op, 0, 0, op_bar);
            tma_load_2d(op_s + K2 * C::LD, &map_op2, 0, 2 * K2, op_bar);
            tma_load_2d(op_s + (K2 + 8) * C::LD, &map_op, 0, K2, op_bar);
        } else {
            tma_load_2d(op_s, &map_op, 0, 0, op_bar);
        }
    }

    // L2 residency (126 MB): the additive operand (yfix: J x 2N doubles, 64 MB at config 3) is re-read by every
    // iteration of the step and is asked to stay (evict_last); the iterate streams: a row of y is dead once its tile
    // and the two neighbouring tiles have read it (evict_first), and y^(l+1) is written with the default priority so
    // that its most recently written part is still in L2 when iteration l+1 reads it - which is why odd iterations
    // walk the tiles in the opposite order (`rev`).  ifix is only read by the FINAL pass: written evict_first.
    const uint64_t pol_last = l2_policy_evict_last(), pol_first = l2_policy_evict_first();
    bool rev = false;                    // this iteration walks the CTA's tiles from the last one down
    auto tile_at = [&](int m) -> int64_t { return blockIdx.x + (int64_t)(rev ? Mcta - 1 - m : m) * gridDim.x; };
    auto claim = [&]() -> int {
        int m = 0;
        if (lane == 0) m = atomicAdd(&tile_ctr, 1);
        return __shfl_sync(0xffffffffu, m, 0);
    };

    // one lane requests a tile: tensor-map boxes straight into the warp's private ring
    const CUtensorMap* my = nullptr;     // tensor map of this iteration's source y
    int tc = 0;                          // tiles this warp has consumed so far (ring position)
    auto prefetch = [&](int m, int tcm) {   // tile m of the CTA into the stage of the warp's tcm-th tile
        if (lane == 0) {
            const int s = tcm & 1;
            const int j0 = (int)(tile_at(m) * RT_M);
            unsigned char* st = my_ring + (size_t)s * C::STAGE_BYTES;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&my_full[s], C::TX_BYTES);
            if (PASS == PASS_FIX) {
                tma_load_2d(st, my, N2, j0 + 1, &my_full[s]);                                     // y map row = cell + 1
                tma_load_2d(st + RT_M * C::LDH * 8, &map_z, N2, j0, &my_full[s]);
                tma_load_2d(st + 2 * RT_M * C::LDH * 8, &map_q, 0, j0, &my_full[s]);
            } else {
                tma_load_2d_hint(st, my, 0, j0, &my_full[s], pol_first);                          // rows j0-1 .. j0+16
            }
        }
        __syncwarp();
    };

    EpiCtx E;
    E.fixp = PASS == PASS_FINAL ? V.ifix : V.yfix;
    E.out = PASS == PASS_FINAL ? V.z : V.yfix;          // ITER: set per iteration
    E.phifix = V.phifix;
    E.phi = V.phi;
    E.phifix_out = V.phifix;
    E.pol_keep = pol_last;
    E.pol_out = pol_last;          // FIX: yfix stays for the iterations
    EpiCtx E1 = E;                 // FIX: the pending I rows go to ifix
    E1.out = V.ifix;
    E1.pol_out = pol_first;

    double* Yd = nullptr;
    const double* brow = op_s + g4 * C::LD + t4;
    constexpr int NBP = PASS == PASS_FIX ? C::NB1 : C::NB0;      // blocks of the epilogue carried from tile to tile
    mbar_wait(op_bar, 0);

    // reflecting ghost rows of y (reading S4) by the warp that owns the edge cell, once its stores are out
    auto ghost_rows = [&](int64_t j0, int rows) {
        if (PASS != PASS_ITER || rows == 0) return;
        const bool gl = j0 == 0 && V.bcL == OCI_BC_REFLECTING;
        const bool gr = j0 + rows == J && V.bcR == OCI_BC_REFLECTING;
        if (gl || gr) {
            __syncwarp();
            __threadfence_block();
            for (int q = lane; q < K2; q += 32) {
                const int mir = mirror_q(q, N);
                if (gl && q >= N) Yd[-(int64_t)K2 + q] = __ldcg(Yd + mir);
                if (gr && q < N) Yd[J * K2 + q] = __ldcg(Yd + (J - 1) * K2 + mir);
            }
            __syncwarp();
        }
    };

  for (int l = 0; l < nloop; ++l) {
    const int ysrc_l = PASS == PASS_ITER ? (ybase + l) & 1 : ysrc;
    my = (ysrc_l == ybase) ? &map_a : &map_a_alt;
    Yd = V.y[ysrc_l ^ 1];
    if (PASS == PASS_ITER) E.out = Yd;
    rev = PASS == PASS_ITER && ((slot + l) & 1);
    int m_cur = claim();
    if (m_cur < Mcta) prefetch(m_cur, tc);
    double dmax = 0.0, rmax = 0.0;
    double pend[2][NBP][2];
#pragma unroll
    for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int t = 0; t < NBP; ++t) pend[g][t][0] = pend[g][t][1] = 0.0;
    int64_t pj0 = m_cur < Mcta ? tile_at(m_cur) * RT_M : 0;
    int prows = 0;                                                 // nothing pending yet: loads clamped, stores off
    bool worked = false;

    for (; m_cur < Mcta; ++tc) {
        const int s = tc & 1;
        const int64_t j0 = tile_at(m_cur) * RT_M;
        const int rows = (int)((J - j0 < RT_M) ? (J - j0) : RT_M);
        m_cur = claim();                                           // the NEXT tile, requested before this one is computed
        if (m_cur < Mcta) prefetch(m_cur, tc + 1);
        worked = true;
        // the additive operands of THIS tile's epilogue (drained during the next phase) -> L2, so that the loads
        // issued DIST k-steps ahead of their use see an L2 hit instead of a DRAM round trip
        if (PASS != PASS_FIX) {
            const char* f0 = reinterpret_cast<const char*>(E.fixp + j0 * K2);
            const int bytes = rows * K2 * 8;
            for (int o = lane * 128; o < bytes; o += 32 * 128) prefetch_l2_evict_last(f0 + o);
            if (PASS == PASS_ITER && lane < 8) {
                const char* p0 = reinterpret_cast<const char*>((lane < 4 ? E.phifix : E.phi) + j0 * 4);
                const int o = (lane & 3) * 128;
                if (o < rows * 32) asm volatile("prefetch.global.L2 [%0];" ::"l"(p0 + o));
            }
        }

        double acc[2][C::NB0][2];
#pragma unroll
        for (int g = 0; g < 2; ++g)
#pragma unroll
            for (int t = 0; t < C::NB0; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;

        mbar_wait(&my_full[s], (tc >> 1) & 1);
        const double* st = reinterpret_cast<const double*>(my_ring + (size_t)s * C::STAGE_BYTES);
        if (PASS == PASS_FIX) {
            const double* pa = st + g4 * C::LDH + t4;
            const double* pq = st + 2 * RT_M * C::LDH + g4 * 4 + t4;
            // row group 0 (O rows + scalar flux) while the previous tile's I rows are stored
            phase<K2, PASS, C::NB0, NBP, PK_FIX1, true>(acc, pa, pq, brow, pend, pj0, prows, E1, g4, t4, dmax, rmax);
            // row group 1 (I rows) while this tile's O rows and scalar flux are stored
            constexpr int NB1 = C::NB1 > 0 ? C::NB1 : 1;
            double acc1[2][NB1][2];
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int t = 0; t < NB1; ++t) acc1[g][t][0] = acc1[g][t][1] = 0.0;
            phase<K2, PASS, NB1, C::NB0, PK_FIX0, true>(acc1, pa, pq, brow + C::NB0 * 8 * C::LD, acc, j0, rows, E, g4, t4, dmax, rmax);
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int t = 0; t < NBP; ++t) { pend[g][t][0] = acc1[g][t < NB1 ? t : 0][0]; pend[g][t][1] = acc1[g][t < NB1 ? t : 0][1]; }
        } else {
            const double* pa = st + g4 * C::LD + t4;
            phase<K2, PASS, C::NB0, NBP, PASS == PASS_ITER ? PK_ITER : PK_FINAL, true>(acc, pa, pa, brow, pend, pj0, prows, E, g4, t4,
                                                                                       dmax, rmax);
            ghost_rows(pj0, prows);
#pragma unroll
            for (int g = 0; g < 2; ++g)
#pragma unroll
                for (int t = 0; t < NBP; ++t) { pend[g][t][0] = acc[g][t][0]; pend[g][t][1] = acc[g][t][1]; }
        }
        pj0 = j0;
        prows = rows;
    }
    // ---- drain the last pending epilogue
    if (prows > 0) {
        double dummy[2][1][2];
        if (PASS == PASS_FIX) phase<K2, PASS, 1, NBP, PK_FIX1, false>(dummy, nullptr, nullptr, nullptr, pend, pj0, prows, E1, g4, t4, dmax, rmax);
        else
            phase<K2, PASS, 1, NBP, PASS == PASS_ITER ? PK_ITER : PK_FINAL, false>(dummy, nullptr, nullptr, nullptr, pend, pj0, prows, E,
                                                                                   g4, t4, dmax, rmax);
        ghost_rows(pj0, prows);
    }
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0 && worked) {
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 1], rmax);
        }
        if (nloop > 1) {
            // ---- grid-wide barrier (cooperative launch: all CTAs are resident), then the stopping rule (a7)
            // on the now final norms of this iteration: every CTA takes the same decision
            __threadfence();
            __syncthreads();
            if (tid == 0) {
                unsigned int* bar = reinterpret_cast<unsigned int*>(V.flags) + 8;
                atomicAdd(bar, 1u);
                const unsigned int target = (unsigned int)(l + 1) * gridDim.x;
                unsigned int seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
                } while (seen < target);
                // the y rows other CTAs have just stored are read next through the async proxy (TMA)
                asm volatile("fence.proxy.async;" ::: "memory");
                tile_ctr = 0;                                      // every warp of the CTA has made its last claim
            }
            __syncthreads();
            const bool stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;
            if (stop && blockIdx.x == 0 && tid == 0) publish_step(V, l + 1, slot + l);
            if (stop) break;
        }
    }
  }
}

bool oci_red_resident_supported(const DevView& V) { return V.nblk == 1 && (V.n == 128 || V.n == 64) && V.J + 18 < (int64_t)1 << 31; }

bool oci_red_resident_prepare(const DevView& V, RedResidentMaps* M)
{
    const uint64_t K2 = (uint64_t)V.n / 2, N = (uint64_t)V.N, J = (uint64_t)V.J;
    const uint32_t LD = (uint32_t)K2 + 4;
    for (int b = 0; b < 2; ++b)
        if (!oci_encode_2d(&M->y_rows[b], V.y[b] - K2, J + 2, K2, RT_M + 2, LD, false) ||
            !oci_encode_2d(&M->y_half[b], V.y[b] - K2, J + 2, K2, RT_M, (uint32_t)N + 4, false))
            return false;
    return oci_encode_2d(&M->z_half, V.z, J, K2, RT_M, (uint32_t)N + 4, false) && oci_encode_2d(&M->q, V.Q, J, 4, RT_M, 4, false) &&
           oci_encode_2d(&M->rop, V.rop, K2 + 8, K2, (uint32_t)K2 + 8, LD, false) &&
           oci_encode_2d(&M->fop, V.fop, K2, K2, (uint32_t)K2, LD, false) &&
           oci_encode_2d(&M->xop_rows, V.xop, 2 * K2 + 8, K2 + 16, (uint32_t)K2, LD, false) &&
           oci_encode_2d(&M->xop_phi, V.xop, 2 * K2 + 8, K2 + 16, 8, LD, false);
}

namespace {
template <int K2, int PASS>
void launch_rr(const DevView& V, const RedResidentMaps& M, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
               cudaStream_t s)
{
    const int sm_count = V.sm_count;
    const int64_t ntiles = (V.J + RT_M - 1) / RT_M;
    const unsigned grid = (unsigned)(ntiles < sm_count ? ntiles : sm_count);
    const int b = ybase & 1;
    const CUtensorMap& ya = PASS == PASS_FIX ? M.y_half[b] : M.y_rows[b];
    const CUtensorMap& yb = PASS == PASS_FIX ? M.y_half[b ^ 1] : M.y_rows[b ^ 1];
    const CUtensorMap& op = PASS == PASS_FIX ? M.xop_rows : PASS == PASS_ITER ? M.rop : M.fop;
    if (PASS == PASS_ITER && cnt > 1) {
        // `cnt` iterations in one launch with a grid-wide barrier between them: every CTA must be resident
        DevView Vv = V;
        CUtensorMap a0 = ya, a1 = yb, a2 = M.z_half, a3 = M.q, a4 = op, a5 = M.xop_phi;
        void* args[] = {&Vv, &a0, &a1, &a2, &a3, &a4, &a5, &ybase, &slot, &prev_slot, &tol, &cnt, &force};
        cudaLaunchCooperativeKernel((const void*)oci_red_resident_kernel<K2, PASS>, dim3(grid), dim3(RT_WARPS * 32), args,
                                    RCfg<K2, PASS>::SMEM, s);     // a refused launch is picked up by launched()
        return;
    }
    oci_red_resident_kernel<K2, PASS><<<grid, RT_WARPS * 32, RCfg<K2, PASS>::SMEM, s>>>(V, ya, yb, M.z_half, M.q, op, M.xop_phi, ybase,
                                                                                        slot, prev_slot, tol, cnt, force);
}

template <int K2>
void launch_rr_pass(const DevView& V, const RedResidentMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt,
                    int force, cudaStream_t s)
{
    if (pass == PASS_FIX) launch_rr<K2, PASS_FIX>(V, M, ybase, 0, -1, tol, 0, 0, s);
    else if (pass == PASS_ITER) launch_rr<K2, PASS_ITER>(V, M, ybase, slot, prev_slot, tol, cnt, 0, s);   // cnt > 1: in-kernel loop
    else launch_rr<K2, PASS_FINAL>(V, M, ybase, 0, -1, tol, cnt, force, s);
}
}  // namespace

int launch_red_resident(const DevView& V, const RedResidentMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt,
                        int force, cudaStream_t s)
{
    if (V.n == 128) launch_rr_pass<64>(V, M, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    else launch_rr_pass<32>(V, M, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    return launched(1);
}

namespace {
template <int K2, int PASS>
cudaError_t opt_in_rr()
{
    return cudaFuncSetAttribute(oci_red_resident_kernel<K2, PASS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RCfg<K2, PASS>::SMEM);
}
}  // namespace

cudaError_t oci_red_resident_opt_in()
{
    cudaError_t e = cudaSuccess;
    if ((e = opt_in_rr<64, PASS_FIX>()) != cudaSuccess || (e = opt_in_rr<64, PASS_ITER>()) != cudaSuccess ||
        (e = opt_in_rr<64, PASS_FINAL>()) != cudaSuccess || (e = opt_in_rr<32, PASS_FIX>()) != cudaSuccess ||
        (e = opt_in_rr<32, PASS_ITER>()) != cudaSuccess || (e = opt_in_rr<32, PASS_FINAL>()) != cudaSuccess)
        return e;
    return e;
}

}  // namespace oci
