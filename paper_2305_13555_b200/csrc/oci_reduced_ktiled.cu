// Interface-reduced OCI step (oci_reduced.cu has the derivation), shared block or a handful of blocks, N a
// multiple of 16 (config 4: N = 128, K2 = 2N = 256; the last 128-row item of a cell tile is partial when K2 is
// not a multiple of 128): the K-tiled fp64 tensor-core
// form of the three passes.  Each pass is a "gathered GEMM"
//     out[j][i] = add[j][i] + sum_k Op[i][k] in_j[k]
// whose input vector is a concatenation of row segments of arrays that already sit in HBM in the packed
// layout (no assembly, |mu| / alpha / h/4 folded into the operator):
//     ITER, FINAL:  in_j = [ y[j+1][0:N] | y[j-1][N:2N] ]
//     FIX        :  in_j = [ y[j][N/2:3N/2] | z[j][N/2:3N/2] | Q16[j] ]
// so every K chunk of the A operand is ONE 2-D tensor-map TMA box (64 cells x 16 k) from some (array,
// column, row shift), and every chunk of the B operand one box (128 operator rows x 16 k).  The operator
// (0.5 - 1.1 MB) stays in L2.
//
//   * persistent CTAs, one per SM; work item = 64 cells x 128 operator rows, full K; the items of one
//     cell tile run on neighbouring SMs at the same time (the input tile is read from HBM once);
//   * 8 MMA warps (2 x 4, each 32 cells x 32 rows, 16 DMMA.8x8x4 accumulators; 224 registers after
//     setmaxnreg) + an auxiliary warpgroup (56 registers) one thread of which issues the TMA,
//     8-stage ring of 26 KB stages, full / empty mbarriers;
//   * shared memory is dense under the hardware 128-byte swizzle; one DMMA consumes the k-set
//     {2s, 2s+1, 2s+8, 2s+9} of the chunk, which makes every fragment load bank-conflict free;
//   * the four scalar-flux rows (H of ITER, W B^{-1} rows of FIX) ride along with item 0 of each cell tile
//     as one more 8-row operator box; MMA warp (wm, wn) takes their k-step ks = wn of every chunk (one
//     extra DMMA per four), the four partial sums meet in shared memory in the epilogue;
//   * epilogue from registers: + yfix / ifix (requested at the start of the item), 16-byte stores, the
//     reflecting ghost rows of y, phi and the two max-norms;
//   * a handful of materials (Reed-type slabs): the operators of all blocks are one tall
//     matrix, so a block is a row offset of the same tensor map; the host lists (cell tile, block, mask of the
//     tile's cells that have this block) groups, a tile that straddles an interface appears once per block it
//     contains and stores only the masked cells.
#include <cuda.h>

#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int RK_M = 64;      // cells per work item
constexpr int RK_N = 128;     // operator rows per work item
constexpr int RK_K = 16;      // k per chunk = one 128-byte swizzle row
constexpr int RK_STAGES = 8;
constexpr int RK_A_BYTES = RK_M * RK_K * 8;   // 8 KB
constexpr int RK_B_BYTES = RK_N * RK_K * 8;   // 16 KB
constexpr int RK_P_BYTES = 8 * RK_K * 8;      // 1 KB: the scalar-flux rows (4 used)
constexpr int RK_STAGE_BYTES = RK_A_BYTES + RK_B_BYTES + RK_P_BYTES + 1024;   // keeps every stage 2 KB-aligned
constexpr size_t RK_SMEM = 1024 /*alignment slack*/ + (size_t)RK_STAGES * RK_STAGE_BYTES + 2 * 4 * RK_M * 4 * 8 /*phi_s, 2 buffers*/ +
                           2 * RK_STAGES * 8 + 16 /*iter_bar, go*/ + 64;

}  // namespace

template <int PASS>
__global__ void __launch_bounds__(384, 1)
oci_red_ktiled_kernel(DevView V, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_y_alt,
                      const __grid_constant__ CUtensorMap map_z, const __grid_constant__ CUtensorMap map_q,
                      const __grid_constant__ CUtensorMap map_op, const __grid_constant__ CUtensorMap map_op8, int ybase, int slot,
                      int prev_slot, double tol, int cnt, int force)
{
    // map_y = tensor map of y[ybase], map_y_alt = of y[ybase ^ 1]
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
    // ITER: `cnt` > 1 iterations run inside this one (cooperative) launch, separated by a grid-wide barrier; iteration l
    // reads y[(ybase + l) & 1], reports its norms in slot `slot + l`, and the loop ends at the first converged one
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;
    if (PASS == PASS_FIX) clear_step_state(V);

    extern __shared__ unsigned char smem_raw[];
    // aligned up inside the shared window (pointer arithmetic on the array keeps the LDS/STS address space)
    unsigned char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char* stages = base;                                                    // [S][A 8K | B 16K | P 1K | pad]
    double* phi_s2 = reinterpret_cast<double*>(base + (size_t)RK_STAGES * RK_STAGE_BYTES);  // [2][4 wn][64][4]
    uint64_t* full = reinterpret_cast<uint64_t*>(phi_s2 + 2 * 4 * RK_M * 4);
    uint64_t* empty = full + RK_STAGES;
    uint64_t* iter_bar = empty + RK_STAGES;   // MMA warps -> producer: "the grid barrier after iteration l has been passed"
    volatile int* go_s = reinterpret_cast<volatile int*>(iter_bar + 1);   // ... and whether another iteration follows

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = V.N, K2 = V.n >> 1, N2 = N >> 1;
    const int64_t J = V.J;
    const int K = PASS == PASS_FIX ? K2 + RK_K : K2;
    const int kch = K / RK_K;                                         // chunks per item
    const int orows = PASS == PASS_FIX ? 2 * K2 : K2;                 // output rows (without the scalar-flux block)
    const int ntn = (orows + RK_N - 1) / RK_N;                        // items per cell tile (the last one may be partial)
    const int prow = PASS == PASS_FIX ? 2 * K2 : K2;                  // operator row of the scalar-flux block
    const int rpb = PASS == PASS_FIX ? 2 * K2 + 8 : PASS == PASS_ITER ? K2 + 8 : K2;   // operator rows per block
    const int64_t nct = (J + RK_M - 1) / RK_M;
    const int64_t ngroups = V.gitems ? V.ngroups : nct;              // (cell tile, block) groups
    const int64_t nitems = ngroups * ntn;
    // item -> (cell tile, output tile, block, mask of the tile's cells that have this block)
    auto decode = [&](int64_t item, int64_t& ct, int& nt, int& blk, unsigned& m0, unsigned& m1) {
        const int64_t g = item / ntn;
        nt = (int)(item - g * ntn);
        if (V.gitems) {
            const int4 e = __ldg(reinterpret_cast<const int4*>(V.gitems) + g);
            ct = e.x; blk = e.y; m0 = (unsigned)e.z; m1 = (unsigned)e.w;
        } else {
            ct = g; blk = 0; m0 = m1 = 0xffffffffu;
        }
    };
    const int my_items = (int)((nitems - blockIdx.x + gridDim.x - 1) / gridDim.x);

    if (tid == 0) {
        for (int s = 0; s < RK_STAGES; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 8);
        }
        mbar_init(iter_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= 8) {
        // =========================== TMA producer (one thread of the auxiliary warpgroup) ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp == 8 && lane == 0) {
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_y)) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_y_alt)) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_op)) : "memory");
            if (PASS != PASS_FINAL) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_op8)) : "memory");
            if (PASS == PASS_FIX) {
                asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_z)) : "memory");
                asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_q)) : "memory");
            }
            int q = 0;
          for (int l = 0; l < nloop; ++l) {
            const int ysrc_l = PASS == PASS_ITER ? (ybase + l) & 1 : ysrc;
            const CUtensorMap* my = (ysrc_l == ybase) ? &map_y : &map_y_alt;
            if (PASS == PASS_ITER && l > 0) {
                // the rows other CTAs stored in iteration l-1 are visible once the grid barrier has been passed (thread 0
                // says so through iter_bar); they are read next through the async proxy (TMA)
                mbar_wait(iter_bar, (l - 1) & 1);
                if (*go_s < 0) break;                                 // the step has converged: no more iterations
                asm volatile("fence.proxy.async;" ::: "memory");
            }
            for (int it = 0; it < my_items; ++it) {
                const int64_t item = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
                int64_t ct;
                int nt, blk;
                unsigned m0, m1;
                decode(item, ct, nt, blk, m0, m1);
                const int j0 = (int)ct * RK_M;
                const int i0 = blk * rpb + nt * RK_N;                // operator row in the tall matrix of all blocks
                const bool with_phi = PASS != PASS_FINAL && nt == 0;
                for (int kc = 0; kc < kch; ++kc, ++q) {
                    const int s = q % RK_STAGES;
                    if (q >= RK_STAGES) mbar_wait(&empty[s], ((q / RK_STAGES) - 1) & 1);
                    unsigned char* st = stages + (size_t)s * RK_STAGE_BYTES;
                    const int k0 = kc * RK_K;
                    // the MMA warps read this stage through the generic proxy (LDS); order those reads, made
                    // visible by the empty barrier, before the async-proxy write of the TMA unit
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(&full[s], RK_A_BYTES + RK_B_BYTES + (with_phi ? RK_P_BYTES : 0));
                    if (PASS == PASS_FIX) {
                        // y / z map rows: y carries the ghost row first (row = cell + 1), z and Q16 do not
                        if (k0 < N) tma_load_2d(st, my, N2 + k0, j0 + 1, &full[s]);
                        else if (k0 < K2) tma_load_2d(st, &map_z, N2 + k0 - N, j0, &full[s]);
                        else tma_load_2d(st, &map_q, 0, j0, &full[s]);
                    } else {
                        // k < N (mu<0) comes from the right neighbour, else from the left one (row a3)
                        tma_load_2d(st, my, k0, j0 + 1 + (k0 < N ? 1 : -1), &full[s]);
                    }
                    tma_load_2d(st + RK_A_BYTES, &map_op, k0, i0, &full[s]);
                    if (with_phi) tma_load_2d(st + RK_A_BYTES + RK_B_BYTES, &map_op8, k0, blk * rpb + prow, &full[s]);
                }
            }
          }
        }
        return;
    }

    // =========================== MMA warps ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    const int g4 = lane >> 2, t4 = lane & 3;
    const int wm = warp >> 2, wn = warp & 3;
    // byte offset of this lane's fragment element inside a 128-byte swizzled row, per k-step:
    // logical 16-byte unit ks + 4*(t4>>1), XOR row&7 (= g4), element t4&1
    int foff[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) foff[ks] = (((ks + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);
    const int a_row = (wm * 32 + g4) * 128;              // + g*1024
    const int b_row = (wn * 32 + g4) * 128;              // + t*1024
    // scalar-flux block: this warp's k-step is ks = wn (computed, not foff[wn]: a runtime index would push the
    // whole foff array into local memory and put a local load in front of every fragment load)
    const int p_off = g4 * 128 + (((wn + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);

    const bool refl_l = V.bcL == OCI_BC_REFLECTING, refl_r = V.bcR == OCI_BC_REFLECTING;

    int q = 0, itc = 0;
  for (int l = 0; l < nloop; ++l) {
    double* __restrict__ Yd = V.y[(PASS == PASS_ITER ? (ybase + l) & 1 : ysrc) ^ 1];
    double dmax = 0.0, rmax = 0.0;
    for (int it = 0; it < my_items; ++it, ++itc) {
        const int64_t item = (int64_t)blockIdx.x + (int64_t)it * gridDim.x;
        int64_t ct;
        int nt, blk;
        unsigned m0, m1;
        decode(item, ct, nt, blk, m0, m1);
        const int64_t j0 = ct * RK_M;
        const int i0 = nt * RK_N;
        const bool with_phi = PASS != PASS_FINAL && nt == 0;
        const unsigned mw = wm ? m1 : m0;                            // this warp's 32 cells of the tile

        // ---- additive operand of the epilogue, requested now
        double2 fx[4][4];
        if (PASS != PASS_FIX) {
            const double* __restrict__ fixp = PASS == PASS_FINAL ? V.ifix : V.yfix;
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                int64_t j = j0 + wm * 32 + 8 * g + g4;
                if (j >= J) j = J - 1;
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const int i = i0 + wn * 32 + 8 * t + 2 * t4;
                    fx[g][t] = i < orows ? *reinterpret_cast<const double2*>(fixp + j * K2 + i) : make_double2(0.0, 0.0);
                }
            }
        }

        // scalar flux of this item's cells: thread tid will finish (cell tid/4, slot tid%4); its operands are
        // requested now so that the epilogue has no dependent global load behind its barrier
        double pfix = 0.0, pold = 0.0;
        if (with_phi && PASS == PASS_ITER) {
            int64_t j = j0 + (tid >> 2);
            if (j >= J) j = J - 1;
            pfix = V.phifix[j * 4 + (tid & 3)];
            pold = V.phi[j * 4 + (tid & 3)];
        }
        double* phi_s = phi_s2 + (itc & 1) * (4 * RK_M * 4);   // alternating buffers: one barrier per item

        double acc[4][4][2], accp[4][2];
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            accp[g][0] = accp[g][1] = 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;
        }

        for (int kc = 0; kc < kch; ++kc, ++q) {
            const int s = q % RK_STAGES;
            mbar_wait(&full[s], (q / RK_STAGES) & 1);
            const unsigned char* st = stages + (size_t)s * RK_STAGE_BYTES;
            const unsigned char* As = st + a_row;
            const unsigned char* Bs = st + RK_A_BYTES + b_row;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                double a[4], b[4];
#pragma unroll
                for (int g = 0; g < 4; ++g) a[g] = *reinterpret_cast<const double*>(As + g * 1024 + foff[ks]);
#pragma unroll
                for (int t = 0; t < 4; ++t) b[t] = *reinterpret_cast<const double*>(Bs + t * 1024 + foff[ks]);
#pragma unroll
                for (int g = 0; g < 4; ++g)
#pragma unroll
                    for (int t = 0; t < 4; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
                if (with_phi && ks == wn) {
                    const double bp = *reinterpret_cast<const double*>(st + RK_A_BYTES + RK_B_BYTES + p_off);
#pragma unroll
                    for (int g = 0; g < 4; ++g) dmma(accp[g][0], accp[g][1], a[g], bp);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[s]);
        }

        // ---- epilogue
#pragma unroll
        for (int g = 0; g < 4; ++g) {
            const int r = wm * 32 + 8 * g + g4;
            const int64_t j = j0 + r;
            if (j < J && ((mw >> (8 * g + g4)) & 1u)) {
#pragma unroll
                for (int t = 0; t < 4; ++t) {
                    const int i = i0 + wn * 32 + 8 * t + 2 * t4;
                    if (i >= orows) continue;                        // partial last item: rows of the phi block / the next block
                    if (PASS == PASS_ITER) {
                        const double v0 = fx[g][t].x + acc[g][t][0], v1 = fx[g][t].y + acc[g][t][1];
                        *reinterpret_cast<double2*>(Yd + j * K2 + i) = make_double2(v0, v1);
                        // reading S4: the mirror image of the edge cell's outgoing flux becomes the ghost row
                        if (j == 0 && refl_l && i < N) {
                            Yd[-(int64_t)K2 + mirror_q(i, N)] = v0;
                            Yd[-(int64_t)K2 + mirror_q(i + 1, N)] = v1;
                        }
                        if (j == J - 1 && refl_r && i >= N) {
                            Yd[J * K2 + mirror_q(i, N)] = v0;
                            Yd[J * K2 + mirror_q(i + 1, N)] = v1;
                        }
                    } else if (PASS == PASS_FINAL) {
                        *reinterpret_cast<double2*>(V.z + j * K2 + i) = make_double2(fx[g][t].x + acc[g][t][0], fx[g][t].y + acc[g][t][1]);
                    } else {
                        double* dst = i < K2 ? V.yfix + j * K2 + i : V.ifix + j * K2 + (i - K2);
                        *reinterpret_cast<double2*>(dst) = make_double2(acc[g][t][0], acc[g][t][1]);
                    }
                }
            }
            if (with_phi && t4 < 2) {     // columns 0..3 of the scalar-flux block: this warp's k-partial
                phi_s[(wn * RK_M + r) * 4 + 2 * t4 + 0] = accp[g][0];
                phi_s[(wn * RK_M + r) * 4 + 2 * t4 + 1] = accp[g][1];
            }
        }
        if (with_phi) {                                              // uniform over the CTA
            named_bar_sync(1, 256);
            // thread tid owns (cell tid/4, slot tid%4) of the item
            const int64_t j = j0 + (tid >> 2);
            const bool mine = (((tid >> 7) ? m1 : m0) >> ((tid >> 2) & 31)) & 1u;
            const double ssum = phi_s[0 * RK_M * 4 + tid] + phi_s[1 * RK_M * 4 + tid] + phi_s[2 * RK_M * 4 + tid] + phi_s[3 * RK_M * 4 + tid];
            if (j < J && mine) {
                if (PASS == PASS_FIX) {
                    V.phifix[j * 4 + (tid & 3)] = ssum;
                } else {
                    const double a = pfix + ssum;
                    V.phi[j * 4 + (tid & 3)] = a;
                    dmax = nanmax(dmax, fabs(a - pold));
                    rmax = nanmax(rmax, fabs(a));
                }
            }
        }
    }
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) {
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * (slot + l) + 1], rmax);
        }
        if (nloop > 1) {
            // ---- grid-wide barrier over the MMA warps of all CTAs (cooperative launch: all resident), then the stopping
            // rule (a7) on the now final norms; the producer thread follows through iter_bar / go_s
            __threadfence();
            named_bar_sync(1, 256);
            if (tid == 0) {
                unsigned int* bar = reinterpret_cast<unsigned int*>(V.flags) + 8;
                atomicAdd(bar, 1u);
                const unsigned int target = (unsigned int)(l + 1) * gridDim.x;
                unsigned int seen;
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
                } while (seen < target);
            }
            named_bar_sync(1, 256);
            const bool stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;
            if (stop && blockIdx.x == 0 && tid == 0) publish_step(V, l + 1, slot + l);
            if (tid == 0) {
                *go_s = stop ? -1 : 1;
                mbar_arrive(iter_bar);
            }
            if (stop) break;
        }
    }
  }
}

// ---- ping-pong variant of the same kernel, used when every CTA has at least one item per math group.
// Two math groups of four warps share the SM, each warp 64 cells x 32 operator rows (32 accumulators), each group
// with its own ring of RP_STAGES stages and its own producer thread; group 1 starts half an item behind group 0, so
// one group's epilogue (global loads and stores, the scalar-flux barrier: 4 - 9 us of an item in the kernel above,
// where all eight warps sit through it together) overlaps the other group's DMMA stream.  Measured at config 4:
// FIX 0.176 -> 0.156 ms, ITER 0.107 -> 0.103 ms.  With fewer items than that an item would only get four warps,
// which is slower (measured +20 % on a 70-item problem): the launcher then takes the kernel above.
constexpr int RP_STAGES = 4;                  // per math group
constexpr size_t RP_SMEM = 1024 /*alignment slack*/ + (size_t)2 * RP_STAGES * RK_STAGE_BYTES + 2 * 4 * RK_M * 4 * 8 /*phi_s, one per group*/ +
                           (4 * RP_STAGES + 1) * 8 + 64;

template <int PASS>
__global__ void __launch_bounds__(384, 1)
oci_red_ktiled_pp_kernel(DevView V, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_y_alt,
                      const __grid_constant__ CUtensorMap map_z, const __grid_constant__ CUtensorMap map_q,
                      const __grid_constant__ CUtensorMap map_op, const __grid_constant__ CUtensorMap map_op8, int ybase, int slot,
                      int prev_slot, double tol, int cnt, int force)
{
    // map_y = tensor map of y[ybase], map_y_alt = of y[ybase ^ 1]
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
    const CUtensorMap* my = (ysrc == ybase) ? &map_y : &map_y_alt;
    if (PASS == PASS_FIX) clear_step_state(V);

    extern __shared__ unsigned char smem_raw[];
    // aligned up inside the shared window (pointer arithmetic on the array keeps the LDS/STS address space)
    unsigned char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    double* phi_all = reinterpret_cast<double*>(base + (size_t)2 * RP_STAGES * RK_STAGE_BYTES);   // [2 groups][4 wn][64][4]
    uint64_t* bars = reinterpret_cast<uint64_t*>(phi_all + 2 * 4 * RK_M * 4);
    uint64_t* stagger = bars + 4 * RP_STAGES;    // group 0 -> group 1: "I am half way through my first item"

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = V.N, K2 = V.n >> 1, N2 = N >> 1;
    const int64_t J = V.J;
    const int K = PASS == PASS_FIX ? K2 + RK_K : K2;
    const int kch = K / RK_K;                                         // chunks per item
    const int orows = PASS == PASS_FIX ? 2 * K2 : K2;                 // output rows (without the scalar-flux block)
    const int ntn = (orows + RK_N - 1) / RK_N;                        // items per cell tile (the last one may be partial)
    const int prow = PASS == PASS_FIX ? 2 * K2 : K2;                  // operator row of the scalar-flux block
    const int rpb = PASS == PASS_FIX ? 2 * K2 + 8 : PASS == PASS_ITER ? K2 + 8 : K2;   // operator rows per block
    const int64_t nct = (J + RK_M - 1) / RK_M;
    const int64_t ngroups = V.gitems ? V.ngroups : nct;              // (cell tile, block) groups
    const int64_t nitems = ngroups * ntn;
    // item -> (cell tile, output tile, block, mask of the tile's cells that have this block)
    auto decode = [&](int64_t item, int64_t& ct, int& nt, int& blk, unsigned& m0, unsigned& m1) {
        const int64_t g = item / ntn;
        nt = (int)(item - g * ntn);
        if (V.gitems) {
            const int4 e = __ldg(reinterpret_cast<const int4*>(V.gitems) + g);
            ct = e.x; blk = e.y; m0 = (unsigned)e.z; m1 = (unsigned)e.w;
        } else {
            ct = g; blk = 0; m0 = m1 = 0xffffffffu;
        }
    };
    // Two math groups of four warps share the SM: group mg takes the items blockIdx.x + (2 it + mg) W.  Each has its
    // own stage ring and producer thread, and group 1 starts half an item late, so while one group sits in its
    // epilogue (loads, stores, the scalar-flux barrier) the other one keeps the DMMA pipe busy.
    const int W = gridDim.x;
    auto items_of = [&](int mg) { const int64_t first = (int64_t)blockIdx.x + (int64_t)mg * W;
                                  return first < nitems ? (int)((nitems - first + 2 * W - 1) / (2 * W)) : 0; };

    if (tid == 0) {
        for (int s = 0; s < 2 * RP_STAGES; ++s) {
            mbar_init(&bars[s], 1);                          // full[mg][s]
            mbar_init(&bars[2 * RP_STAGES + s], 4);          // empty[mg][s]: the four warps of the group
        }
        mbar_init(stagger, 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= 8) {
        // ============ auxiliary warpgroup: lane 0 of warps 8 and 9 = the TMA producers of ring 0 and ring 1 ============
        asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
        if (warp < 10 && lane == 0) {
            const int mg = warp - 8;
            unsigned char* stages = base + (size_t)mg * RP_STAGES * RK_STAGE_BYTES;
            uint64_t* full = bars + mg * RP_STAGES;
            uint64_t* empty = bars + 2 * RP_STAGES + mg * RP_STAGES;
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(my)) : "memory");
            asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_op)) : "memory");
            if (PASS != PASS_FINAL) asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_op8)) : "memory");
            if (PASS == PASS_FIX) {
                asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_z)) : "memory");
                asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&map_q)) : "memory");
            }
            const int my_items = items_of(mg);
            int q = 0;
            for (int it = 0; it < my_items; ++it) {
                const int64_t item = (int64_t)blockIdx.x + (int64_t)(2 * it + mg) * W;
                int64_t ct;
                int nt, blk;
                unsigned m0, m1;
                decode(item, ct, nt, blk, m0, m1);
                const int j0 = (int)ct * RK_M;
                const int i0 = blk * rpb + nt * RK_N;                // operator row in the tall matrix of all blocks
                const bool with_phi = PASS != PASS_FINAL && nt == 0;
                for (int kc = 0; kc < kch; ++kc, ++q) {
                    const int s = q % RP_STAGES;
                    if (q >= RP_STAGES) mbar_wait(&empty[s], ((q / RP_STAGES) - 1) & 1);
                    unsigned char* st = stages + (size_t)s * RK_STAGE_BYTES;
                    const int k0 = kc * RK_K;
                    // the MMA warps read this stage through the generic proxy (LDS); order those reads, made
                    // visible by the empty barrier, before the async-proxy write of the TMA unit
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_expect_tx(&full[s], RK_A_BYTES + RK_B_BYTES + (with_phi ? RK_P_BYTES : 0));
                    if (PASS == PASS_FIX) {
                        // y / z map rows: y carries the ghost row first (row = cell + 1), z and Q16 do not
                        if (k0 < N) tma_load_2d(st, my, N2 + k0, j0 + 1, &full[s]);
                        else if (k0 < K2) tma_load_2d(st, &map_z, N2 + k0 - N, j0, &full[s]);
                        else tma_load_2d(st, &map_q, 0, j0, &full[s]);
                    } else {
                        // k < N (mu<0) comes from the right neighbour, else from the left one (row a3)
                        tma_load_2d(st, my, k0, j0 + 1 + (k0 < N ? 1 : -1), &full[s]);
                    }
                    tma_load_2d(st + RK_A_BYTES, &map_op, k0, i0, &full[s]);
                    if (with_phi) tma_load_2d(st + RK_A_BYTES + RK_B_BYTES, &map_op8, k0, blk * rpb + prow, &full[s]);
                }
            }
        }
        return;
    }

    // =========================== MMA warps: group mg = warp / 4, four warps x (64 cells x 32 rows) ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");   // 8 x 32 x 208 + 4 x 32 x 56 registers: slack in every SM partition
    const int g4 = lane >> 2, t4 = lane & 3;
    const int mg = warp >> 2, wn = warp & 3;
    const int gtid = tid & 127;                              // thread index inside the group
    unsigned char* stages = base + (size_t)mg * RP_STAGES * RK_STAGE_BYTES;
    uint64_t* full = bars + mg * RP_STAGES;
    uint64_t* empty = bars + 2 * RP_STAGES + mg * RP_STAGES;
    double* phi_s = phi_all + mg * (4 * RK_M * 4);           // [4 wn][64][4] k-partials of this group
    // byte offset of this lane's fragment element inside a 128-byte swizzled row, per k-step:
    // logical 16-byte unit ks + 4*(t4>>1), XOR row&7 (= g4), element t4&1
    int foff[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) foff[ks] = (((ks + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);
    const int a_row = g4 * 128;                              // + g*1024, g = 0..7: all 64 cells
    const int b_row = (wn * 32 + g4) * 128;                  // + t*1024
    // scalar-flux block: this warp's k-step is ks = wn (computed: a runtime index into foff would push it to local memory)
    const int p_off = g4 * 128 + (((wn + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);

    double* __restrict__ Yd = V.y[ysrc ^ 1];
    const double* __restrict__ fixp = PASS == PASS_FINAL ? V.ifix : V.yfix;
    double dmax = 0.0, rmax = 0.0;
    const bool refl_l = V.bcL == OCI_BC_REFLECTING, refl_r = V.bcR == OCI_BC_REFLECTING;
    const int my_items = items_of(mg);

    if (mg == 1) mbar_wait(stagger, 0);                      // start half an item behind group 0

    int q = 0;
    for (int it = 0; it < my_items; ++it) {
        const int64_t item = (int64_t)blockIdx.x + (int64_t)(2 * it + mg) * W;
        int64_t ct;
        int nt, blk;
        unsigned m0, m1;
        decode(item, ct, nt, blk, m0, m1);
        const int64_t j0 = ct * RK_M;
        const int i0 = nt * RK_N;
        const bool with_phi = PASS != PASS_FINAL && nt == 0;

        // scalar flux of this item's cells: thread gtid finishes (cell p/4, slot p%4) for p = gtid, gtid + 128; the
        // operands are requested now so that nothing behind the barrier waits for global memory
        double pfix[2] = {0.0, 0.0}, pold[2] = {0.0, 0.0};
        if (with_phi && PASS == PASS_ITER) {
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int p = gtid + 128 * u;
                int64_t j = j0 + (p >> 2);
                if (j >= J) j = J - 1;
                pfix[u] = V.phifix[j * 4 + (p & 3)];
                pold[u] = V.phi[j * 4 + (p & 3)];
            }
        }

        double acc[8][4][2], accp[8][2];
#pragma unroll
        for (int g = 0; g < 8; ++g) {
            accp[g][0] = accp[g][1] = 0.0;
#pragma unroll
            for (int t = 0; t < 4; ++t) acc[g][t][0] = acc[g][t][1] = 0.0;
        }

        for (int kc = 0; kc < kch; ++kc, ++q) {
            const int s = q % RP_STAGES;
            mbar_wait(&full[s], (q / RP_STAGES) & 1);
            const unsigned char* st = stages + (size_t)s * RK_STAGE_BYTES;
            const unsigned char* As = st + a_row;
            const unsigned char* Bs = st + RK_A_BYTES + b_row;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
                double a[8], b[4];
#pragma unroll
                for (int g = 0; g < 8; ++g) a[g] = *reinterpret_cast<const double*>(As + g * 1024 + foff[ks]);
#pragma unroll
                for (int t = 0; t < 4; ++t) b[t] = *reinterpret_cast<const double*>(Bs + t * 1024 + foff[ks]);
#pragma unroll
                for (int g = 0; g < 8; ++g)
#pragma unroll
                    for (int t = 0; t < 4; ++t) dmma(acc[g][t][0], acc[g][t][1], a[g], b[t]);
                if (with_phi && ks == wn) {
                    const double bp = *reinterpret_cast<const double*>(st + RK_A_BYTES + RK_B_BYTES + p_off);
#pragma unroll
                    for (int g = 0; g < 8; ++g) dmma(accp[g][0], accp[g][1], a[g], bp);
                }
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(&empty[s]);
                if (mg == 0 && it == 0 && kc == (kch >> 1)) mbar_arrive(stagger);
            }
        }
        if (mg == 0 && it == 0 && kch < 2 && lane == 0) mbar_arrive(stagger);   // (kch >= 2 always; belt and braces)

        // ---- epilogue: + additive operand (one cell block of 8 at a time), 16-byte stores, reflecting ghost rows
#pragma unroll
        for (int g = 0; g < 8; ++g) {
            const int r = 8 * g + g4;
            const int64_t j = j0 + r;
            const bool live = j < J && (((g < 4 ? m0 : m1) >> (r & 31)) & 1u);
            double2 f[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int i = i0 + wn * 32 + 8 * t + 2 * t4;
                f[t] = (PASS != PASS_FIX && live && i < orows) ? *reinterpret_cast<const double2*>(fixp + j * K2 + i) : make_double2(0.0, 0.0);
            }
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                const int i = i0 + wn * 32 + 8 * t + 2 * t4;
                if (!live || i >= orows) continue;                   // partial last item: rows of the phi block / the next block
                if (PASS == PASS_ITER) {
                    const double v0 = f[t].x + acc[g][t][0], v1 = f[t].y + acc[g][t][1];
                    *reinterpret_cast<double2*>(Yd + j * K2 + i) = make_double2(v0, v1);
                    // reading S4: the mirror image of the edge cell's outgoing flux becomes the ghost row
                    if (j == 0 && refl_l && i < N) {
                        Yd[-(int64_t)K2 + mirror_q(i, N)] = v0;
                        Yd[-(int64_t)K2 + mirror_q(i + 1, N)] = v1;
                    }
                    if (j == J - 1 && refl_r && i >= N) {
                        Yd[J * K2 + mirror_q(i, N)] = v0;
                        Yd[J * K2 + mirror_q(i + 1, N)] = v1;
                    }
                } else if (PASS == PASS_FINAL) {
                    *reinterpret_cast<double2*>(V.z + j * K2 + i) = make_double2(f[t].x + acc[g][t][0], f[t].y + acc[g][t][1]);
                } else {
                    double* dst = i < K2 ? V.yfix + j * K2 + i : V.ifix + j * K2 + (i - K2);
                    *reinterpret_cast<double2*>(dst) = make_double2(acc[g][t][0], acc[g][t][1]);
                }
            }
            if (with_phi && t4 < 2) {     // columns 0..3 of the scalar-flux block: this warp's k-partial
                phi_s[(wn * RK_M + r) * 4 + 2 * t4 + 0] = accp[g][0];
                phi_s[(wn * RK_M + r) * 4 + 2 * t4 + 1] = accp[g][1];
            }
        }
        if (with_phi) {                                              // uniform over the group
            named_bar_sync(1 + mg, 128);
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int p = gtid + 128 * u;                        // (cell p/4, slot p%4)
                const int r = p >> 2;
                const int64_t j = j0 + r;
                const double ssum = phi_s[0 * RK_M * 4 + p] + phi_s[1 * RK_M * 4 + p] + phi_s[2 * RK_M * 4 + p] + phi_s[3 * RK_M * 4 + p];
                if (j < J && (((r < 32 ? m0 : m1) >> (r & 31)) & 1u)) {
                    if (PASS == PASS_FIX) {
                        V.phifix[j * 4 + (p & 3)] = ssum;
                    } else {
                        const double a = pfix[u] + ssum;
                        V.phi[j * 4 + (p & 3)] = a;
                        dmax = nanmax(dmax, fabs(a - pold[u]));
                        rmax = nanmax(rmax, fabs(a));
                    }
                }
            }
            named_bar_sync(1 + mg, 128);                             // phi_s of this group reusable
        }
    }
    if (mg == 0 && my_items == 0 && lane == 0) mbar_arrive(stagger);  // never leave group 1 waiting
    if (PASS == PASS_ITER) {
        dmax = warp_max(dmax);
        rmax = warp_max(rmax);
        if (lane == 0) {
            atomic_max_nonneg(&V.norms[2 * slot + 0], dmax);
            atomic_max_nonneg(&V.norms[2 * slot + 1], rmax);
        }
    }
}

bool oci_red_ktiled_supported(const DevView& V)
{
    // chunks of 16 k must not straddle the halves of the gather: N a multiple of 16
    return (V.nblk == 1 || V.gitems != nullptr) && V.N % 16 == 0 && V.n <= 2048 && V.J + 2 < (int64_t)1 << 31;
}

bool oci_red_ktiled_prepare(const DevView& V, RedKtiledMaps* M)
{
    const uint64_t K2 = (uint64_t)V.n / 2, J = (uint64_t)V.J, nb = (uint64_t)V.nblk;
    return oci_encode_2d(&M->y[0], V.y[0] - K2, J + 2, K2, RK_M, RK_K, true) && oci_encode_2d(&M->y[1], V.y[1] - K2, J + 2, K2, RK_M, RK_K, true) &&
           oci_encode_2d(&M->z, V.z, J, K2, RK_M, RK_K, true) && oci_encode_2d(&M->q16, V.q16, J, 16, RK_M, RK_K, true) &&
           oci_encode_2d(&M->xop, V.xop, nb * (2 * K2 + 8), K2 + 16, RK_N, RK_K, true) && oci_encode_2d(&M->xop8, V.xop, nb * (2 * K2 + 8), K2 + 16, 8, RK_K, true) &&
           oci_encode_2d(&M->rop, V.rop, nb * (K2 + 8), K2, RK_N, RK_K, true) && oci_encode_2d(&M->rop8, V.rop, nb * (K2 + 8), K2, 8, RK_K, true) &&
           oci_encode_2d(&M->fop, V.fop, nb * K2, K2, RK_N, RK_K, true);
}

// the eight-warp kernel runs all iterations of a chunk in one cooperative launch; the ping-pong kernel (two producer
// threads, two staggered math groups) keeps one launch per iteration
bool oci_red_ktiled_fuses_loop(const DevView& V)
{
    const int K2 = V.n / 2;
    const int64_t nitems = (V.gitems ? V.ngroups : (V.J + RK_M - 1) / RK_M) * ((K2 + RK_N - 1) / RK_N);
    const int64_t grid = nitems < V.sm_count ? nitems : V.sm_count;
    return nitems < 2 * grid;
}

int launch_red_ktiled(const DevView& V, const RedKtiledMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt,
                      int force, cudaStream_t s)
{
    const int sm_count = V.sm_count;
    const int K2 = V.n / 2;
    const int64_t nitems = (V.gitems ? V.ngroups : (V.J + RK_M - 1) / RK_M) * (((pass == PASS_FIX ? 2 * K2 : K2) + RK_N - 1) / RK_N);
    const unsigned grid = (unsigned)(nitems < sm_count ? nitems : sm_count);
    const CUtensorMap& ya = M.y[ybase & 1];
    const CUtensorMap& yb = M.y[(ybase & 1) ^ 1];
    // ping-pong kernel when both math groups of every CTA get at least one item, else the eight-warp kernel
    const bool pp = nitems >= 2 * (int64_t)grid;
    if (pp) {
        if (pass == PASS_FIX)
            oci_red_ktiled_pp_kernel<PASS_FIX><<<grid, 384, RP_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.xop, M.xop8, ybase, 0, -1, tol, 0, 0);
        else if (pass == PASS_ITER)
            oci_red_ktiled_pp_kernel<PASS_ITER><<<grid, 384, RP_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.rop, M.rop8, ybase, slot, prev_slot, tol, 0, 0);
        else
            oci_red_ktiled_pp_kernel<PASS_FINAL><<<grid, 384, RP_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.fop, M.fop, ybase, 0, -1, tol, cnt, force);
        return launched(1);
    }
    if (pass == PASS_FIX)
        oci_red_ktiled_kernel<PASS_FIX><<<grid, 384, RK_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.xop, M.xop8, ybase, 0, -1, tol, 0, 0);
    else if (pass == PASS_ITER && cnt > 1) {
        // `cnt` iterations in one launch with a grid-wide barrier between them: every CTA is resident (grid <= SMs)
        DevView Vv = V;
        CUtensorMap a0 = ya, a1 = yb, a2 = M.z, a3 = M.q16, a4 = M.rop, a5 = M.rop8;
        int zero = 0;
        void* args[] = {&Vv, &a0, &a1, &a2, &a3, &a4, &a5, &ybase, &slot, &prev_slot, &tol, &cnt, &zero};
        cudaLaunchCooperativeKernel((const void*)oci_red_ktiled_kernel<PASS_ITER>, dim3(grid), dim3(384), args, RK_SMEM, s);
    } else if (pass == PASS_ITER)
        oci_red_ktiled_kernel<PASS_ITER><<<grid, 384, RK_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.rop, M.rop8, ybase, slot, prev_slot, tol, 0, 0);
    else
        oci_red_ktiled_kernel<PASS_FINAL><<<grid, 384, RK_SMEM, s>>>(V, ya, yb, M.z, M.q16, M.fop, M.fop, ybase, 0, -1, tol, cnt, force);
    return launched(1);
}

cudaError_t oci_red_ktiled_opt_in()
{
    cudaError_t e = cudaSuccess;
    const auto at = cudaFuncAttributeMaxDynamicSharedMemorySize;
    if ((e = cudaFuncSetAttribute(oci_red_ktiled_kernel<PASS_FIX>, at, (int)RK_SMEM)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_ktiled_kernel<PASS_ITER>, at, (int)RK_SMEM)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_ktiled_kernel<PASS_FINAL>, at, (int)RK_SMEM)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_ktiled_pp_kernel<PASS_FIX>, at, (int)RP_SMEM)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_ktiled_pp_kernel<PASS_ITER>, at, (int)RP_SMEM)) != cudaSuccess ||
        (e = cudaFuncSetAttribute(oci_red_ktiled_pp_kernel<PASS_FINAL>, at, (int)RP_SMEM)) != cudaSuccess)
        return e;
    return e;
}

}  // namespace oci
