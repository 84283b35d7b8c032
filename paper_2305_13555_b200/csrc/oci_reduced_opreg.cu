// Interface-reduced OCI step (oci_reduced.cu has the derivation), ONE shared block, K2 = 2N in {128, 256}
// (config 4: N = 128): the three passes with the OPERATOR STATIONARY IN REGISTERS.
//
//     out[j][i] = add[j][i] + sum_k Op[i][k] in_j[k]          (the "gathered GEMM" of oci_reduced_ktiled.cu)
//
// The K-tiled kernels stream both operands through shared memory in 16-wide K chunks and re-fetch the
// operator (0.5 MB for ITER at N = 128) from L2 for every 64-cell item; ncu showed them bound by that
// hand-off (DMMA pipe 58 % busy), not by the pipe.  Here the operator never moves:
//
//   * a CTA owns 64 operator rows for the whole launch ("row group"; ITER at N = 128 has 4, FIX 8); its eight
//     MMA warps own 8 rows each and keep their 8 x K2 slice as DMMA B-fragments IN REGISTERS (K2/4 doubles per
//     thread: 64 at K2 = 256), loaded from L2 once per launch;
//   * the CTA walks tiles of 64 cells (tiles t = c / NRG, c / NRG + G, ...; G = CTAs per row group): only the
//     input rows stream, as tensor-map TMA boxes (64 cells x 16 k, 128-byte swizzle, two boxes = 32 k per
//     stage) into an 8-stage ring; a warp reads every A fragment of a stage (8 cell blocks x 8 k-steps) and
//     issues 64 DMMA.8x8x4 per stage with no operator traffic at all: per k-step 8 LDS.64 + 8 DMMA;
//   * the additive operand (yfix for ITER, ifix for FINAL) of a tile arrives by TMA as well (4 boxes, double
//     buffered), so the epilogue is LDS + DADD + 16-byte stores with no global-load latency in it;
//   * the four scalar-flux rows (H of ITER, W B^{-1} rows of FIX) sit in shared memory (8 x K2, padded); the
//     row group t mod NRG does them for tile t, warp w for its cell block w (one more DMMA per k-step): a
//     warp ends with complete sums for 8 cells x 4 slots, no cross-warp or cross-CTA reduction;
//   * ITER: all iterations of a chunk run in ONE cooperative launch (grid-wide barrier + device-side stop,
//     row a7), the operator slices staying in registers across iterations;
//   * FIX: the 4 source columns ride along as one more box (Q16) and two k-steps.
//
// One DMMA consumes the k-set {2s, 2s+1, 2s+8, 2s+9} of a 16-chunk (s = k-step in the chunk): under the
// 128-byte swizzle that makes the A-fragment loads bank-conflict free; the B fragments are loaded from
// global memory with the same permutation.
#include <cuda.h>

#include <type_traits>

#include "device_utils.cuh"

namespace oci {

namespace {

constexpr int RO_M = 64;                          // cells per tile
constexpr int RO_ROWS = 64;                       // operator rows per CTA (8 warps x 8)
constexpr int RO_RING = 8;                        // stages in the input ring
constexpr int RO_BOX_BYTES = RO_M * 16 * 8;       // one box: 64 cells x 16 k = 8 KB
constexpr int RO_STAGE_BYTES = 2 * RO_BOX_BYTES;  // 32 k per stage
constexpr int RO_FX_BYTES = 4 * RO_BOX_BYTES;     // additive operand of a tile: 64 cells x 64 rows = 32 KB

template <int K2, int PASS>
struct OCfg {
    static constexpr int N = K2 / 2;
    static constexpr int MAIN_STAGES = K2 / 32;                          // stages of the gathered input vector
    static constexpr int SPT = MAIN_STAGES + (PASS == PASS_FIX ? 1 : 0);  // stages per tile (FIX: + the Q16 box)
    static constexpr int KST = K2 / 4;                                   // k-steps of the gathered input vector
    static constexpr int OROWS = PASS == PASS_FIX ? 2 * K2 : K2;         // output rows without the scalar-flux block
    static constexpr int NRG = OROWS / RO_ROWS;                          // row groups
    static constexpr bool PHI = PASS != PASS_FINAL;
    static constexpr bool ADD = PASS != PASS_FIX;
    static constexpr int PLD = K2 + 18;                                  // pitch of the scalar-flux operator: 2 (mod 16)
    static constexpr int OPLD = PASS == PASS_FIX ? K2 + 16 : K2;         // row stride of the operator in global memory
    static constexpr int PROW = PASS == PASS_FIX ? 2 * K2 : K2;          // operator row of the scalar-flux block
    static constexpr size_t SMEM = 1024 /*alignment slack*/ + (size_t)RO_RING * RO_STAGE_BYTES + (ADD ? 2 * RO_FX_BYTES : 0) +
                                   (PHI ? 8 * PLD * 8 : 0) + (2 * RO_RING + 8) * 8 + 64;
};

}  // namespace

template <int K2, int PASS>
__global__ void __launch_bounds__(384, 1)
oci_red_opreg_kernel(DevView V, const __grid_constant__ CUtensorMap map_y, const __grid_constant__ CUtensorMap map_y_alt,
                     const __grid_constant__ CUtensorMap map_z, const __grid_constant__ CUtensorMap map_q,
                     const __grid_constant__ CUtensorMap map_add, int ybase, int slot, int prev_slot, double tol, int cnt, int force)
{
    using C = OCfg<K2, PASS>;
    constexpr int N = C::N, N2 = N / 2;
    // map_y = tensor map of y[ybase], map_y_alt = of y[ybase ^ 1]; map_add = of yfix (ITER) / ifix (FINAL)
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
    if (PASS == PASS_FIX) clear_step_state(V);
    const int nloop = PASS == PASS_ITER ? (cnt > 1 ? cnt : 1) : 1;

    extern __shared__ unsigned char smem_raw[];
    unsigned char* base = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    unsigned char* ring = base;                                                       // [RING][2 boxes]
    unsigned char* fxbuf = ring + (size_t)RO_RING * RO_STAGE_BYTES;                  // [2][4 boxes]
    double* pop = reinterpret_cast<double*>(fxbuf + (C::ADD ? 2 * RO_FX_BYTES : 0));  // [8][PLD] scalar-flux operator
    uint64_t* full = reinterpret_cast<uint64_t*>(reinterpret_cast<unsigned char*>(pop) + (C::PHI ? 8 * C::PLD * 8 : 0));
    uint64_t* empty = full + RO_RING;
    uint64_t* fx_full = empty + RO_RING;      // [2]
    uint64_t* fx_empty = fx_full + 2;         // [2]
    uint64_t* iter_bar = fx_empty + 2;        // MMA warps -> producer: "the grid barrier after iteration l has been passed"
    uint64_t* stagger = iter_bar + 1;         // warps 0-3 -> warps 4-7: "one stage into this iteration"
    volatile int* go_s = reinterpret_cast<volatile int*>(stagger + 1);   // ... and whether another iteration follows

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t J = V.J;
    const int64_t nct = (J + RO_M - 1) / RO_M;
    const int rg = blockIdx.x % C::NRG;                      // this CTA's row group
    const int G = gridDim.x / C::NRG;                        // CTAs per row group (the launcher makes the grid a multiple)
    const int t0 = blockIdx.x / C::NRG;
    const int my_tiles = t0 < nct ? (int)((nct - t0 + G - 1) / G) : 0;

    if (tid == 0) {
        for (int s = 0; s < RO_RING; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], 8);
        }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&fx_full[s], 1);
            mbar_init(&fx_empty[s], 8);
        }
        mbar_init(iter_bar, 1);
        mbar_init(stagger, 4);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // the scalar-flux operator rows -> shared memory (plain loads: once per launch)
    if (C::PHI) {
        const double* __restrict__ Op = PASS == PASS_FIX ? V.xop : V.rop;
        for (int e = tid; e < 8 * C::PLD; e += blockDim.x) {
            const int r = e / C::PLD, k = e - r * C::PLD;
            pop[e] = (r < 4 && k < (PASS == PASS_FIX ? K2 + 4 : K2)) ? Op[(size_t)(C::PROW + r) * C::OPLD + k] : 0.0;
        }
    }
    __syncthreads();

    if (warp >= 8) {
        // =========================== TMA producer (one thread of the auxiliary warpgroup) ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
        if (warp == 8 && lane == 0) {
            int q = 0, f = 0;                                 // stages / additive tiles issued so far
            for (int l = 0; l < nloop; ++l) {
                const int ysrc_l = PASS == PASS_ITER ? (ybase + l) & 1 : ysrc;
                const CUtensorMap* my = (ysrc_l == ybase) ? &map_y : &map_y_alt;
                if (PASS == PASS_ITER && l > 0) {
                    // the rows other CTAs stored in iteration l-1 are visible once the grid barrier has been passed
                    // (thread 0 says so through iter_bar); they are read next through the async proxy (TMA)
                    mbar_wait(iter_bar, (l - 1) & 1);
                    if (*go_s < 0) break;                     // the step has converged: no more iterations
                    asm volatile("fence.proxy.async;" ::: "memory");
                }
                for (int it = 0; it < my_tiles; ++it) {
                    const int j0 = (t0 + it * G) * RO_M;
                    if (C::ADD) {
                        const int fs = f & 1;
                        if (f >= 2) mbar_wait(&fx_empty[fs], ((f >> 1) - 1) & 1);
                        fence_proxy_async();
                        mbar_expect_tx(&fx_full[fs], RO_FX_BYTES);
                        for (int b = 0; b < 4; ++b)
                            tma_load_2d(fxbuf + (size_t)fs * RO_FX_BYTES + b * RO_BOX_BYTES, &map_add, rg * RO_ROWS + 16 * b, j0, &fx_full[fs]);
                        ++f;
                    }
                    for (int s = 0; s < C::SPT; ++s, ++q) {
                        const int st = q & (RO_RING - 1);
                        if (q >= RO_RING) mbar_wait(&empty[st], ((q / RO_RING) - 1) & 1);
                        unsigned char* dst = ring + (size_t)st * RO_STAGE_BYTES;
                        fence_proxy_async();
                        if (s < C::MAIN_STAGES) {
                            mbar_expect_tx(&full[st], RO_STAGE_BYTES);
                            for (int b = 0; b < 2; ++b) {
                                const int k0 = 32 * s + 16 * b;
                                if (PASS == PASS_FIX) {
                                    // psi_{k-1/2}: the k+1/2 runs of y[j] and z[j] (y carries the ghost row first)
                                    if (k0 < N) tma_load_2d(dst + b * RO_BOX_BYTES, my, N2 + k0, j0 + 1, &full[st]);
                                    else tma_load_2d(dst + b * RO_BOX_BYTES, &map_z, N2 + k0 - N, j0, &full[st]);
                                } else {
                                    // k < N (mu < 0) from the right neighbour, else from the left one (row a3)
                                    tma_load_2d(dst + b * RO_BOX_BYTES, my, k0, j0 + 1 + (k0 < N ? 1 : -1), &full[st]);
                                }
                            }
                        } else {
                            mbar_expect_tx(&full[st], RO_BOX_BYTES);
                            tma_load_2d(dst, &map_q, 0, j0, &full[st]);
                        }
                    }
                }
            }
        }
        return;
    }

    // =========================== MMA warps ===========================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    const int g4 = lane >> 2, t4 = lane & 3;
    const int row0 = rg * RO_ROWS + 8 * warp;                // this warp's 8 operator rows
    // k index this lane holds for k-step kk of the gathered vector: chunk kk/4, set {2s, 2s+1, 2s+8, 2s+9}
    const int kperm = 8 * (t4 >> 1) + (t4 & 1);
    // ---- the operator slice, once per launch: b[kk] = Op[row0 + g4][16 (kk/4) + 2 (kk%4) + kperm]
    double bfr[C::KST];
    {
        const double* __restrict__ Op = (PASS == PASS_FIX ? V.xop : PASS == PASS_ITER ? V.rop : V.fop) + (size_t)(row0 + g4) * C::OPLD + kperm;
#pragma unroll
        for (int kk = 0; kk < C::KST; ++kk) bfr[kk] = __ldg(Op + 16 * (kk >> 2) + 2 * (kk & 3));
    }
    double bq0 = 0.0, bq1 = 0.0;                              // FIX: the four source columns (two k-steps of the Q16 box)
    if (PASS == PASS_FIX && (t4 >> 1) == 0) {
        const double* __restrict__ Xq = V.xop + (size_t)(row0 + g4) * C::OPLD + K2;
        bq0 = __ldg(Xq + (t4 & 1));
        bq1 = __ldg(Xq + 2 + (t4 & 1));
    }
    // byte offset of this lane's A-fragment element inside a box row, per k-step of a chunk
    int foff[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) foff[ks] = (((ks + 4 * (t4 >> 1)) ^ g4) << 4) + ((t4 & 1) << 3);
    const int a_row = g4 * 128;                               // + g * 1024 (cell block g)
    const double* pfr = pop + g4 * C::PLD + kperm;            // scalar-flux B fragment: + 16 (kk/4) + 2 (kk%4)
    // additive operand in shared memory: box b = warp/2, 16-byte unit 4 (warp&1) + t4 of row (cell), swizzled
    const int fx_off = (warp >> 1) * RO_BOX_BYTES + g4 * 128 + (((4 * (warp & 1) + t4) ^ g4) << 4);

    const bool refl_l = V.bcL == OCI_BC_REFLECTING, refl_r = V.bcR == OCI_BC_REFLECTING;
    int q = 0, f = 0;
    for (int l = 0; l < nloop; ++l) {
        const int ysrc_l = PASS == PASS_ITER ? (ybase + l) & 1 : ysrc;
        double* __restrict__ Yd = V.y[ysrc_l ^ 1];
        double dmax = 0.0, rmax = 0.0;
        // The two warps of every SM partition (w and w + 4) run one stage apart, so that the epilogue of one (shared-
        // memory loads, adds, stores: about the time of the 64 DMMAs of a stage) overlaps the other one's DMMA stream
        // instead of idling the pipe in lock step; the grid barrier re-aligns them, so the offset is set up per iteration.
        if (warp >= 4 && my_tiles > 0) mbar_wait(stagger, l & 1);
        for (int it = 0; it < my_tiles; ++it) {
            const int tile = t0 + it * G;
            const int64_t j0 = (int64_t)tile * RO_M;
            const bool with_phi = C::PHI && (tile % C::NRG) == rg;

            double acc[8][2], accp[2] = {0.0, 0.0};
#pragma unroll
            for (int g = 0; g < 8; ++g) acc[g][0] = acc[g][1] = 0.0;

            uint32_t ready = mbar_test(&full[q & (RO_RING - 1)], (q / RO_RING) & 1);
            // The k loop of a tile exists twice: without the scalar-flux rows (three tiles of four run this one: nothing
            // but the fragment loads and the DMMA stream) and with them (one more fragment pair and DMMA per k-step).
            // A branch or a predicate per k-step instead costs every tile about 15 % (measured): it breaks the stream up.
            auto tile_mma = [&](auto phi_tag) {
                constexpr bool WP = decltype(phi_tag)::value;
#pragma unroll
                for (int s = 0; s < C::MAIN_STAGES; ++s) {
                    const int st = (q + s) & (RO_RING - 1);
                    if (!ready) mbar_wait(&full[st], ((q + s) / RO_RING) & 1);
                    // the next stage's barrier is tested now and looked at after this stage's DMMAs (FIX: the Q16 stage last)
                    if (s + 1 < C::SPT) ready = mbar_test(&full[(q + s + 1) & (RO_RING - 1)], ((q + s + 1) / RO_RING) & 1);
                    const unsigned char* As = ring + (size_t)st * RO_STAGE_BYTES + a_row;
                    const unsigned char* Ap = As + warp * 1024;              // this warp's own cell block (scalar flux)
#pragma unroll
                    for (int k8 = 0; k8 < 8; ++k8) {
                        const int kk = 8 * s + k8;                           // k-step of the gathered vector
                        const int ko = (k8 >> 2) * RO_BOX_BYTES + foff[k8 & 3];
                        double a[8];
#pragma unroll
                        for (int g = 0; g < 8; ++g) a[g] = *reinterpret_cast<const double*>(As + ko + g * 1024);
#pragma unroll
                        for (int g = 0; g < 8; ++g) dmma(acc[g][0], acc[g][1], a[g], bfr[kk]);
                        if (WP) {
                            // cell block g = warp against the scalar-flux rows (a[warp] would be a runtime register index)
                            const double ap = *reinterpret_cast<const double*>(Ap + ko);
                            const double bp = pfr[16 * (kk >> 2) + 2 * (kk & 3)];
                            dmma(accp[0], accp[1], ap, bp);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) {
                        mbar_arrive(&empty[st]);
                        // group 0 (warps 0-3) tells group 1 (warps 4-7) that it is one stage into the iteration
                        if (s == 0 && it == 0 && warp < 4) mbar_arrive(stagger);
                    }
                }
            };
            if (with_phi) tile_mma(std::true_type{});
            else tile_mma(std::false_type{});
            if (PASS == PASS_FIX) {
                // the source columns: box Q16 (columns 0..3 used), k-steps 0 and 1 of its chunk
                const int st = (q + C::MAIN_STAGES) & (RO_RING - 1);
                if (!ready) mbar_wait(&full[st], ((q + C::MAIN_STAGES) / RO_RING) & 1);
                const unsigned char* As = ring + (size_t)st * RO_STAGE_BYTES + a_row;
#pragma unroll
                for (int ks = 0; ks < 2; ++ks) {
                    double a[8];
#pragma unroll
                    for (int g = 0; g < 8; ++g) a[g] = *reinterpret_cast<const double*>(As + g * 1024 + foff[ks]);
                    const double bq = ks ? bq1 : bq0;
#pragma unroll
                    for (int g = 0; g < 8; ++g) dmma(acc[g][0], acc[g][1], a[g], bq);
                    if (with_phi) {
                        const double ap = *reinterpret_cast<const double*>(As + warp * 1024 + foff[ks]);
                        const double bp = (t4 >> 1) == 0 ? pop[g4 * C::PLD + K2 + 2 * ks + (t4 & 1)] : 0.0;
                        dmma(accp[0], accp[1], ap, bp);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&empty[st]);
            }
            q += C::SPT;

            // ---- epilogue: + additive operand (shared memory), 16-byte stores, reflecting ghost rows
            const int i = rg * RO_ROWS + 8 * warp + 2 * t4;                  // output row (pair i, i+1)
            if (C::ADD) {
                const int fs = f & 1;
                mbar_wait(&fx_full[fs], (f >> 1) & 1);
                const unsigned char* Fx = fxbuf + (size_t)fs * RO_FX_BYTES + fx_off;
#pragma unroll
                for (int g = 0; g < 8; ++g) {
                    const double2 fx = *reinterpret_cast<const double2*>(Fx + g * 1024);
                    acc[g][0] += fx.x;
                    acc[g][1] += fx.y;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&fx_empty[fs]);
                ++f;
            }
#pragma unroll
            for (int g = 0; g < 8; ++g) {
                const int64_t j = j0 + 8 * g + g4;
                if (j >= J) continue;
                const double2 v = make_double2(acc[g][0], acc[g][1]);
                if (PASS == PASS_ITER) {
                    *reinterpret_cast<double2*>(Yd + j * K2 + i) = v;
                    // reading S4: the mirror image of the edge cell's outgoing flux becomes the ghost row
                    if (j == 0 && refl_l && i < N) {
                        Yd[-(int64_t)K2 + mirror_q(i, N)] = v.x;
                        Yd[-(int64_t)K2 + mirror_q(i + 1, N)] = v.y;
                    }
                    if (j == J - 1 && refl_r && i >= N) {
                        Yd[J * K2 + mirror_q(i, N)] = v.x;
                        Yd[J * K2 + mirror_q(i + 1, N)] = v.y;
                    }
                } else if (PASS == PASS_FINAL) {
                    *reinterpret_cast<double2*>(V.z + j * K2 + i) = v;
                } else {
                    double* dst = i < K2 ? V.yfix + j * K2 + i : V.ifix + j * K2 + (i - K2);
                    *reinterpret_cast<double2*>(dst) = v;
                }
            }
            if (with_phi && t4 < 2) {
                // complete sums of cell 8 warp + g4, slots 2 t4, 2 t4 + 1
                const int64_t j = j0 + 8 * warp + g4;
                if (j < J) {
                    if (PASS == PASS_FIX) {
                        *reinterpret_cast<double2*>(V.phifix + j * 4 + 2 * t4) = make_double2(accp[0], accp[1]);
                    } else {
                        const double2 pf = *reinterpret_cast<const double2*>(V.phifix + j * 4 + 2 * t4);
                        const double2 po = __ldcg(reinterpret_cast<const double2*>(V.phi + j * 4 + 2 * t4));
                        const double p0 = pf.x + accp[0], p1 = pf.y + accp[1];
                        *reinterpret_cast<double2*>(V.phi + j * 4 + 2 * t4) = make_double2(p0, p1);
                        dmax = nanmax(dmax, nanmax(fabs(p0 - po.x), fabs(p1 - po.y)));
                        rmax = nanmax(rmax, nanmax(fabs(p0), fabs(p1)));
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
                // ---- grid-wide barrier over the MMA warps of all CTAs (cooperative launch: all resident), then the
                // stopping rule (a7) on the now final norms; the producer thread follows through flags[9]
                __threadfence();
                named_bar_sync(1, 256);
                bool stop = false;
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
                stop = step_done(V.norms, slot + l, tol) || l + 1 == nloop;
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

bool oci_red_opreg_supported(const DevView& V)
{
    return V.nblk == 1 && (V.n == 512 || V.n == 256 || V.n == 128) && V.J + 2 < (int64_t)1 << 31 && V.sm_count >= 8;
}

bool oci_red_opreg_prepare(const DevView& V, RedOpregMaps* M)
{
    const uint64_t K2 = (uint64_t)V.n / 2, J = (uint64_t)V.J;
    return oci_encode_2d(&M->y[0], V.y[0] - K2, J + 2, K2, RO_M, 16, true) && oci_encode_2d(&M->y[1], V.y[1] - K2, J + 2, K2, RO_M, 16, true) &&
           oci_encode_2d(&M->z, V.z, J, K2, RO_M, 16, true) && oci_encode_2d(&M->q16, V.q16, J, 16, RO_M, 16, true) &&
           oci_encode_2d(&M->yfix, V.yfix, J, K2, RO_M, 16, true) && oci_encode_2d(&M->ifix, V.ifix, J, K2, RO_M, 16, true);
}

namespace {
template <int K2, int PASS>
int launch_ro(const DevView& V, const RedOpregMaps& M, int ybase, int slot, int prev_slot, double tol, int cnt, int force, cudaStream_t s)
{
    using C = OCfg<K2, PASS>;
    const int64_t nct = (V.J + RO_M - 1) / RO_M;
    int64_t G = V.sm_count / C::NRG;                       // CTAs per row group
    if (G > nct) G = nct;
    const unsigned grid = (unsigned)(G * C::NRG);
    const CUtensorMap& ya = M.y[ybase & 1];
    const CUtensorMap& yb = M.y[(ybase & 1) ^ 1];
    const CUtensorMap& add = PASS == PASS_FINAL ? M.ifix : M.yfix;
    if (PASS == PASS_ITER && cnt > 1) {
        DevView Vv = V;
        CUtensorMap a0 = ya, a1 = yb, a2 = M.z, a3 = M.q16, a4 = add;
        void* args[] = {&Vv, &a0, &a1, &a2, &a3, &a4, &ybase, &slot, &prev_slot, &tol, &cnt, &force};
        cudaLaunchCooperativeKernel((const void*)oci_red_opreg_kernel<K2, PASS>, dim3(grid), dim3(384), args, C::SMEM, s);
        return launched(1);
    }
    oci_red_opreg_kernel<K2, PASS><<<grid, 384, C::SMEM, s>>>(V, ya, yb, M.z, M.q16, add, ybase, slot, prev_slot, tol, cnt, force);
    return launched(1);
}

template <int K2>
int launch_ro_pass(const DevView& V, const RedOpregMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                   cudaStream_t s)
{
    if (pass == PASS_FIX) return launch_ro<K2, PASS_FIX>(V, M, ybase, 0, -1, tol, 0, 0, s);
    if (pass == PASS_ITER) return launch_ro<K2, PASS_ITER>(V, M, ybase, slot, prev_slot, tol, cnt, 0, s);
    return launch_ro<K2, PASS_FINAL>(V, M, ybase, 0, -1, tol, cnt, force, s);
}

template <int K2, int PASS>
cudaError_t opt_in_ro()
{
    return cudaFuncSetAttribute(oci_red_opreg_kernel<K2, PASS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)OCfg<K2, PASS>::SMEM);
}
}  // namespace

int launch_red_opreg(const DevView& V, const RedOpregMaps& M, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force,
                     cudaStream_t s)
{
    if (V.n == 512) return launch_ro_pass<256>(V, M, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    if (V.n == 256) return launch_ro_pass<128>(V, M, pass, ybase, slot, prev_slot, tol, cnt, force, s);
    return launch_ro_pass<64>(V, M, pass, ybase, slot, prev_slot, tol, cnt, force, s);
}

cudaError_t oci_red_opreg_opt_in()
{
    cudaError_t e = cudaSuccess;
    if ((e = opt_in_ro<256, PASS_FIX>()) != cudaSuccess || (e = opt_in_ro<256, PASS_ITER>()) != cudaSuccess ||
        (e = opt_in_ro<256, PASS_FINAL>()) != cudaSuccess || (e = opt_in_ro<128, PASS_FIX>()) != cudaSuccess ||
        (e = opt_in_ro<128, PASS_ITER>()) != cudaSuccess || (e = opt_in_ro<128, PASS_FINAL>()) != cudaSuccess ||
        (e = opt_in_ro<64, PASS_FIX>()) != cudaSuccess || (e = opt_in_ro<64, PASS_ITER>()) != cudaSuccess ||
        (e = opt_in_ro<64, PASS_FINAL>()) != cudaSuccess)
        return e;
    return e;
}

}  // namespace oci
