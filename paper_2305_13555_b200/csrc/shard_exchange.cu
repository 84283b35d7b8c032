// Row f4: one slab sharded over several GPUs by contiguous cell ranges ("can be dynamically
// decomposed to split over multiple accelerators within an iteration").  Within an OCI iteration cells only
// talk to their neighbours' previous iterate, so per iteration a shard owes each neighbour the N outgoing values of
// its edge cell (one half row of the packed iterate y) and every rank needs the MAX over ranks of the two norms of
// the stopping rule (exact, order independent: iteration counts equal the single-GPU run's).
//
// Transport: plain stores into PEER MEMORY.  Every rank owns a small mailbox that all ranks can address (NVLink peer
// mapping / symmetric memory set up by the caller):
//     halo [2 parity][2 face][N]      what arrives at my left (0) / right (1) face
//     norms[2 parity][world][2]       (d, r) of every rank
//     flags[world]  u64               the tag of the last exchange each rank has completed pushing
// push: stores the two half rows into the neighbours' mailboxes and (d, r) into everyone's, system-scope fence, then
// the tag into everyone's flags[my rank].  pull: waits until every rank's flag has reached the tag, copies the half
// rows into the ghost rows of y (the apply kernels read a HALO face exactly like a physical boundary) and replaces the
// local norms by the global maximum, which the next launch's device-side stop reads.  Both are stream-ordered
// single-CTA kernels behind each ITER launch: no host involvement per iteration, no collective library in the data
// path.  Consecutive exchanges alternate the parity half of the mailbox, so a rank that runs ahead by one exchange
// cannot overwrite data a slower rank has not pulled yet (it cannot run ahead by two: its next pull needs the slow
// rank's next push).
#include "device_utils.cuh"

namespace oci {

namespace {
__device__ __forceinline__ double* mbox_of(const DevView& V, int r) { return reinterpret_cast<double*>(V.peers[r]); }
}  // namespace

// ybuf: the y buffer whose edge rows are sent (the iteration's destination); slot: norm slot of the iteration, or -1
// for an exchange without norms (after set_flux)
__global__ void __launch_bounds__(128) shard_push_kernel(DevView V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    const int N = V.N, K2 = V.n >> 1, W = V.world, me = V.rank;
    const int par = (int)(tag & 1ull);
    const double* __restrict__ Y = V.y[ybuf];
    // what leaves through my left face (q < N of cell 0) arrives at the left neighbour's RIGHT face, and vice versa
    if (me > 0) {
        double* dst = mbox_of(V, me - 1) + (size_t)(par * 2 + 1) * N;
        for (int q = threadIdx.x; q < N; q += blockDim.x) dst[q] = __ldcg(Y + q);
    }
    if (me < W - 1) {
        double* dst = mbox_of(V, me + 1) + (size_t)(par * 2 + 0) * N;
        for (int q = threadIdx.x; q < N; q += blockDim.x) dst[q] = __ldcg(Y + (V.J - 1) * K2 + N + q);
    }
    if (slot >= 0) {
        for (int r = threadIdx.x; r < W; r += blockDim.x) {
            unsigned long long* nr = reinterpret_cast<unsigned long long*>(mbox_of(V, r) + 4 * (size_t)N) + (size_t)(par * W + me) * 2;
            nr[0] = __ldcg(V.norms + 2 * slot + 0);
            nr[1] = __ldcg(V.norms + 2 * slot + 1);
        }
    }
    __threadfence_system();
    __syncthreads();
    for (int r = threadIdx.x; r < W; r += blockDim.x) {
        unsigned long long* fl = reinterpret_cast<unsigned long long*>(mbox_of(V, r) + 4 * (size_t)N + 4 * (size_t)W) + me;
        asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(fl), "l"(tag) : "memory");
    }
}

__global__ void __launch_bounds__(128) shard_pull_kernel(DevView V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag)
{
    if (step_done(V.norms, prev_slot, tol)) return;
    const int N = V.N, K2 = V.n >> 1, W = V.world, me = V.rank;
    const int par = (int)(tag & 1ull);
    double* mine = mbox_of(V, me);
    for (int r = threadIdx.x; r < W; r += blockDim.x) {
        const unsigned long long* fl = reinterpret_cast<const unsigned long long*>(mine + 4 * (size_t)N + 4 * (size_t)W) + r;
        unsigned long long seen;
        do {
            asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(seen) : "l"(fl) : "memory");
        } while (seen < tag);
    }
    __syncthreads();
    double* __restrict__ Y = V.y[ybuf];
    if (me > 0) {          // ghost row -1: the entries cell 0 gathers from its left neighbour are q >= N
        const volatile double* src = mine + (size_t)(par * 2 + 0) * N;
        for (int q = threadIdx.x; q < N; q += blockDim.x) Y[-(int64_t)K2 + N + q] = src[q];
    }
    if (me < W - 1) {      // ghost row J: q < N
        const volatile double* src = mine + (size_t)(par * 2 + 1) * N;
        for (int q = threadIdx.x; q < N; q += blockDim.x) Y[V.J * K2 + q] = src[q];
    }
    if (slot >= 0 && threadIdx.x == 0) {
        const volatile unsigned long long* nr = reinterpret_cast<const volatile unsigned long long*>(mine + 4 * (size_t)N) + (size_t)par * W * 2;
        unsigned long long d = 0ull, r = 0ull;          // bit patterns of non-negative doubles (or NaN): integer max is exact
        for (int k = 0; k < W; ++k) {
            d = max(d, nr[2 * k + 0]);
            r = max(r, nr[2 * k + 1]);
        }
        V.norms[2 * slot + 0] = d;
        V.norms[2 * slot + 1] = r;
    }
}

int launch_shard_push(const DevView& V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag, cudaStream_t s)
{
    shard_push_kernel<<<1, 128, 0, s>>>(V, ybuf, slot, prev_slot, tol, tag);
    return launched(1);
}

int launch_shard_pull(const DevView& V, int ybuf, int slot, int prev_slot, double tol, unsigned long long tag, cudaStream_t s)
{
    shard_pull_kernel<<<1, 128, 0, s>>>(V, ybuf, slot, prev_slot, tol, tag);
    return launched(1);
}

}  // namespace oci
