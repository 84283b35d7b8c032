// Host driver behind the C ABI of include/oci.h: argument checking, quadrature, block
// classification, workspace layout, the time-step loop and error
// reporting.  Every arithmetic step of the path runs in the kernels of this directory.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>

#include "oci_internal.h"

namespace oci {
int launch_oci_generic(const DevView& V, int src, int prev_slot, double tol, cudaStream_t s);
int launch_oci_percell(const DevView& V, int src, int slot, int prev_slot, double tol, cudaStream_t s);
int launch_oci_shared_fast(const DevView& V, int src, int slot, int prev_slot, double tol, cudaStream_t s);
bool oci_shared_fast_supported(const DevView& V);
bool oci_ktiled_supported(const DevView& V);
bool oci_ktiled_prepare(const DevView& V, KtiledMaps* M);
int launch_oci_ktiled(const DevView& V, const KtiledMaps& M, int src, int slot, int prev_slot, double tol, cudaStream_t s);
}  // namespace oci

using namespace oci;

struct oci_ctx {
    // problem
    int64_t J = 0;
    int32_t N = 0, n = 0;
    double v = 0, dt = 0;
    oci_bc bcL{}, bcR{};
    std::vector<double> dx, sig, sigs, mu, w;
    // classification
    std::vector<int32_t> blk;
    std::vector<int64_t> rep;
    int64_t nblk = 0;
    int32_t path = OCI_PATH_SHARED;
    // device
    DevView V{};
    alignas(64) KtiledMaps maps{};
    alignas(64) RedKtiledMaps rmaps{};
    alignas(64) RedResidentMaps rrmaps{};
    alignas(64) RedOpregMaps romaps{};
    bool use_ktiled = false;
    int32_t forced_rkernel = OCI_RKERNEL_AUTO;   // oci_set_reduced_kernel
    int32_t small_mode = -1;                     // oci_set_small_step: -1 auto, 0 off, 1 required
    int32_t small_cluster = 0;                   // cluster size of the one-launch step, 0 = not used (resolved in oci_setup)
    int32_t si_small_cluster = 0;                // the same for the SI comparator's one-launch step (si_small.cu)
    // row f4: shard of a slab (shard_exchange.cu)
    bool sharded = false;
    unsigned long long xtag = 0;       // exchanges completed so far (the next one carries xtag + 1)
    int device = -1;                   // the device the workspace lives on; made current inside every entry point
    cudaStream_t stream = nullptr;
    void* ws = nullptr;
    int64_t ws_bytes = 0;
    bool ready = false, have_flux = false;
    int cur = 0;                       // psi[cur] holds the current iterate
    // interface-reduced iteration (oci_reduced.cu)
    int32_t iteration = OCI_ITERATION_AUTO;
    int ycur = 0;                      // (y[ycur], z) hold the current iterate in packed form ...
    bool yz_valid = false;             // ... when this is set (cleared by set_flux, si_step, a FULL-form oci_step)
    bool psi_valid = false;            // psi[cur] holds the current iterate in the full layout (cleared by a REDUCED step)
    int32_t red_kernel = OCI_RKERNEL_GEMV;
    bool coop = false;                 // device supports cooperative launches
    int32_t predicted[2] = {0, 0};     // last iteration count of oci / si, sizes the launch chunk
    unsigned long long* h_norms = nullptr;   // pinned
    unsigned long long* h_pub = nullptr;     // pinned + mapped: [4] = seq, iterations, bits(d), bits(r) written by a fused loop (a7)
    unsigned long long* d_pub = nullptr;     // its device address
    unsigned long long pub_seq = 0;
    cudaStream_t stream2 = nullptr;          // side stream of the norm read-back (REDUCED form)
    cudaEvent_t ev_norms = nullptr;
    cudaEvent_t ev_snap = nullptr, ev_snap_done = nullptr;   // oci_get_scalar_flux_async
    bool snap_pending = false;
    double* phi_stage = nullptr;
    // timing
    bool timing = false;
    std::vector<cudaEvent_t> ev;
    cudaEvent_t ev_aux[4] = {nullptr, nullptr, nullptr, nullptr};
    double kernel_ms = 0.0;
    double setup_ms = 0.0;             // device time of form + invert + pack in the last oci_setup
    int64_t kernel_launches = 0;
    double aux_ms[2] = {0.0, 0.0};     // reduced iteration: Psi_fix pass, finalisation
    int64_t aux_launches[2] = {0, 0};
    int64_t launches = 0;
    std::string err;
};

namespace {

int fail(const oci_ctx* c, int code, const std::string& msg)
{
    if (c) const_cast<oci_ctx*>(c)->err = msg;
    return code;
}

int cuda_fail(const oci_ctx* c, cudaError_t e, const char* where)
{
    return fail(c, OCI_E_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

#define CK(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call);      \
    } while (0)

// a launcher returns the number of kernels it launched, or -1 when CUDA refused a launch
#define LAUNCH(call)                                                  \
    do {                                                              \
        const int k_ = (call);                                        \
        if (k_ < 0) return cuda_fail(ctx, cudaGetLastError(), #call); \
        ctx->launches += k_;                                          \
    } while (0)

// a7 without a copy: wait until the fused iteration loop launched with sequence number `seq` has published its
// iteration count (device_utils.cuh: publish_step).  Spins on the mapped word; every so often it asks the stream whether
// it is still running, so that a failed launch or kernel ends the wait with the CUDA error instead of hanging.
int wait_published(oci_ctx* ctx, unsigned long long seq, int32_t* iterations, double* d, double* r)
{
    volatile unsigned long long* h = ctx->h_pub;
    for (unsigned long spins = 1;; ++spins) {
        if (h[0] == seq) break;
        if ((spins & 4095) == 0) {
            const cudaError_t q = cudaStreamQuery(ctx->stream);
            if (q != cudaErrorNotReady && h[0] != seq) {
                if (q != cudaSuccess) return cuda_fail(ctx, q, "fused iteration loop");
                return fail(ctx, OCI_E_CUDA, "the fused iteration loop ended without reporting its iteration count");
            }
        }
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    *iterations = (int32_t)h[1];
    const unsigned long long db = h[2], rb = h[3];
    std::memcpy(d, &db, 8);
    std::memcpy(r, &rb, 8);
    return OCI_OK;
}

// Makes the context's device current for the duration of an entry point (the caller's current device need not
// be the one the workspace lives on) and restores the previous one on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const oci_ctx* c)
    {
        if (c && c->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard()
    {
        if (switched) cudaSetDevice(prev);
    }
};

// N-point Gauss-Legendre nodes and weights on [-1,1], ascending (weights sum to 2, the 1/2 of
// eq. (1)).  Newton on P_N evaluated by the Bonnet recurrence, from the Tricomi initial guess;
// the negative half is the mirror image of the positive half.
void gauss_legendre(int N, std::vector<double>& mu, std::vector<double>& w)
{
    mu.assign(N, 0.0);
    w.assign(N, 0.0);
    const double pi = 3.141592653589793238462643383279502884;
    for (int i = 0; i < N / 2; ++i) {
        // i-th positive root counted from the largest
        double x = (1.0 - (N - 1.0) / (8.0 * N * N * N)) * std::cos(pi * (4.0 * i + 3.0) / (4.0 * N + 2.0));
        double deriv = 0.0;
        for (int it = 0; it < 64; ++it) {
            double pm1 = 1.0, p = x;
            for (int k = 1; k < N; ++k) {
                const double pn = ((2 * k + 1) * x * p - k * pm1) / (k + 1);
                pm1 = p;
                p = pn;
            }
            deriv = N * (pm1 - x * p) / (1.0 - x * x);
            const double step = p / deriv;
            x -= step;
            if (std::fabs(step) <= 1e-16 * std::fabs(x)) {
                pm1 = 1.0; p = x;
                for (int k = 1; k < N; ++k) {
                    const double pn = ((2 * k + 1) * x * p - k * pm1) / (k + 1);
                    pm1 = p;
                    p = pn;
                }
                deriv = N * (pm1 - x * p) / (1.0 - x * x);
                break;
            }
        }
        const double wt = 2.0 / ((1.0 - x * x) * deriv * deriv);
        mu[N - 1 - i] = x;
        mu[i] = -x;
        w[N - 1 - i] = wt;
        w[i] = wt;
    }
}

struct Layout {
    int64_t binv, psi0, psi1, cfix, phi, Q, qs, dx, sig, sigs, blk, rep, mu, w, coef, ainv4, si_scan, phi_part, norms, tickets, flags,
        xop, rop, fop, y0, y1, z, yfix, ifix, phifix, q16, gitems, perm, team_bar, peers, phi_stage, si_part, si_inflow, si_src1, si_agg, wba, wbd, wbm, total;
};

int64_t align_up(int64_t x) { return (x + 255) & ~int64_t(255); }

Layout make_layout(int64_t J, int32_t N, int64_t nblk)
{
    const int64_t n = 4 * (int64_t)N;
    Layout L{};
    int64_t o = 0;
    auto take = [&](int64_t bytes) { int64_t at = o; o = align_up(o + bytes); return at; };
    L.binv = take(nblk * n * n * 8);
    L.psi0 = take((J + 2) * n * 8);
    L.psi1 = take((J + 2) * n * 8);
    L.cfix = take(J * n * 8);
    L.phi = take(J * 4 * 8);
    L.Q = take(J * 4 * 8);
    L.qs = take(J * 4 * 8);
    L.dx = take(J * 8);
    L.sig = take(J * 8);
    L.sigs = take(J * 8);
    L.blk = take(J * 4);
    L.rep = take(nblk * 8);
    L.mu = take(N * 8);
    L.w = take(N * 8);
    L.coef = take(n * 8);
    L.ainv4 = take(nblk * N * 16 * 8);
    L.si_scan = take(((J + 7) / 8) * N * 8 * 8);          // sized for the smallest chunk si_chunk_cells() can pick
    L.phi_part = take(nblk == 1 ? ((n + 127) / 128) * J * 4 * 8 : 0);
    L.norms = take((kNormSlots + 1) * 2 * 8);
    L.tickets = take(nblk == 1 ? ((J + 63) / 64) * 4 : 0);
    L.flags = take(256);
    {
        const int64_t K2 = n / 2;
        L.xop = take(nblk * (2 * K2 + 8) * (K2 + 16) * 8);
        L.rop = take(nblk * (K2 + 8) * K2 * 8);
        L.fop = take(nblk * K2 * K2 * 8);
        L.y0 = take((J + 2) * K2 * 8);
        L.y1 = take((J + 2) * K2 * 8);
        L.z = take(J * K2 * 8);
        L.yfix = take(J * K2 * 8);
        L.ifix = take(J * K2 * 8);
        L.phifix = take(J * 4 * 8);
        const bool grouped = nblk > 1 && nblk <= kMaxGroupedBlocks && N % 16 == 0;
        L.q16 = take((nblk == 1 || grouped) && N % 16 == 0 ? J * 16 * 8 : 0);
        // (cell tile, block) groups of the K-tiled kernels: at most min(nblk, 64) per tile of 64 cells
        L.gitems = take(grouped ? ((J + 63) / 64) * (nblk < 64 ? nblk : 64) * 16 : 0);
    }
    L.perm = take(nblk * n * 4);
    L.team_bar = take(4096 * 4);
    L.peers = take(64 * 8);
    L.phi_stage = take(J * 4 * 8);
    L.si_part = take((N / 32 > 2 ? N / 32 : 2) * J * 4 * 8);
    L.si_inflow = take(2 * N * 2 * 8);
    L.si_src1 = take(J * 4 * 8);
    L.si_agg = take((int64_t)N * si_carry_segments((J + 7) / 8) * 8 * 8);   // (zeroed by oci_setup together with the flags)
    L.wba = take(nblk * 16 * N * 8);
    L.wbd = take(nblk * 16 * N * 8);
    L.wbm = take(nblk * 32 * 8);
    L.total = o;
    return L;
}

void classify(oci_ctx* c)
{
    struct Key {
        uint64_t a, b, d;
        bool operator==(const Key& o) const { return a == o.a && b == o.b && d == o.d; }
    };
    struct Hash {
        size_t operator()(const Key& k) const
        {
            uint64_t h = k.a * 0x9E3779B97F4A7C15ull;
            h ^= (k.b + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2));
            h ^= (k.d + 0x9E3779B97F4A7C15ull + (h << 6) + (h >> 2));
            return (size_t)h;
        }
    };
    auto bits = [](double x) { uint64_t u; std::memcpy(&u, &x, 8); return u; };
    std::unordered_map<Key, int32_t, Hash> seen;
    c->blk.resize(c->J);
    c->rep.clear();
    for (int64_t j = 0; j < c->J; ++j) {
        Key k{bits(c->dx[j]), bits(c->sig[j]), bits(c->sigs[j])};
        auto it = seen.find(k);
        if (it == seen.end()) {
            it = seen.emplace(k, (int32_t)c->rep.size()).first;
            c->rep.push_back(j);
        }
        c->blk[j] = it->second;
    }
    c->nblk = (int64_t)c->rep.size();
    c->path = (c->nblk == 1) ? OCI_PATH_SHARED : OCI_PATH_PER_CELL;
}

bool bc_ok(const oci_bc& b)
{
    return b.kind == OCI_BC_VACUUM || b.kind == OCI_BC_INCIDENT_ISOTROPIC || b.kind == OCI_BC_REFLECTING || b.kind == OCI_BC_HALO;
}

int launch_oci_iteration_any(oci_ctx* ctx, int src, int slot, int prev_slot, double tol)
{
    const DevView& V = ctx->V;
    if (ctx->path == OCI_PATH_PER_CELL) return launch_oci_percell(V, src, slot, prev_slot, tol, ctx->stream);
    if (oci_shared_fast_supported(V)) return launch_oci_shared_fast(V, src, slot, prev_slot, tol, ctx->stream);
    if (ctx->use_ktiled) return launch_oci_ktiled(V, ctx->maps, src, slot, prev_slot, tol, ctx->stream);
    const int k = launch_oci_generic(V, src, prev_slot, tol, ctx->stream);
    const int k2 = launch_phi_norm(V, src ^ 1, slot, prev_slot, tol, true, ctx->stream);
    return (k < 0 || k2 < 0) ? -1 : k + k2;
}

// AUTO: the reduced form wherever a kernel of that form is the faster one (oci.h)
int32_t resolved_iteration(const oci_ctx* ctx)
{
    if (ctx->iteration != OCI_ITERATION_AUTO) return ctx->iteration;
    if (ctx->path == OCI_PATH_PER_CELL) return OCI_ITERATION_REDUCED;
    if (ctx->ready && ctx->red_kernel != OCI_RKERNEL_GEMV) return OCI_ITERATION_REDUCED;
    return ctx->n <= 32 ? OCI_ITERATION_REDUCED : OCI_ITERATION_FULL;
}

int launch_reduced_pass(oci_ctx* ctx, int pass, int ybase, int slot, int prev_slot, double tol, int cnt, int force)
{
    if (ctx->red_kernel == OCI_RKERNEL_KTILED)
        return launch_red_ktiled(ctx->V, ctx->rmaps, pass, ybase, slot, prev_slot, tol, cnt, force, ctx->stream);
    if (ctx->red_kernel == OCI_RKERNEL_OPREG)
        return launch_red_opreg(ctx->V, ctx->romaps, pass, ybase, slot, prev_slot, tol, cnt, force, ctx->stream);
    if (ctx->red_kernel == OCI_RKERNEL_WOODBURY)
        return launch_red_woodbury(ctx->V, pass, ybase, slot, prev_slot, tol, cnt, force, ctx->stream);
    if (ctx->red_kernel == OCI_RKERNEL_RESIDENT)
        return launch_red_resident(ctx->V, ctx->rrmaps, pass, ybase, slot, prev_slot, tol, cnt, force, ctx->stream);
    return launch_red_gemv(ctx->V, pass, ybase, slot, prev_slot, tol, cnt, force, ctx->stream);
}

// the full-layout Psi on demand (a change of layout, no arithmetic)
int ensure_psi(oci_ctx* ctx)
{
    if (ctx->psi_valid) return 0;
    const int k = launch_unpack_yz(ctx->V, ctx->cur, ctx->ycur, ctx->stream);
    if (k >= 0) ctx->psi_valid = true;
    return k;
}

// Row f4: one time step of n shards that live in this process (n = 1: one process per GPU).  REDUCED form, one launch
// per iteration followed by the halo / norm exchange (shard_exchange.cu); launches of the shards are interleaved so
// that on one device and stream every pull is ordered behind every push.
int run_step_sharded(oci_ctx* const* cs, int32_t n, double tol, int32_t max_iters, int32_t* iters, double* resid)
{
    oci_ctx* ctx = cs[0];                                                    // errors are reported on the first shard
    for (int32_t c = 0; c < n; ++c) {
        if (!cs[c]) return fail(ctx, OCI_E_INVALID, "NULL shard");
        if (!cs[c]->ready || !cs[c]->sharded) return fail(ctx, OCI_E_ORDER, "shard not set up or not attached");
        if (!cs[c]->have_flux) return fail(ctx, OCI_E_ORDER, "step before oci_set_flux");
        if (n > 1 && (cs[c]->stream != ctx->stream || cs[c]->device != ctx->device))
            return fail(ctx, OCI_E_INVALID, "shards stepped together must share one device and one stream");
        if (cs[c]->iteration == OCI_ITERATION_FULL) return fail(ctx, OCI_E_INVALID, "the FULL form is not available on a sharded context");
    }
    if (max_iters < 1 || tol != tol) return fail(ctx, OCI_E_INVALID, "max_iters < 1 or tol is NaN");
    DeviceGuard guard(ctx);
#define EACH for (int32_t c_ = 0; c_ < n; ++c_)
#define C_ cs[c_]
    // the packed state and, after oci_set_flux, the neighbours' edge values in the ghost rows
    bool fresh = false;
    EACH if (!C_->yz_valid) fresh = true;
    if (fresh) {
        EACH {
            oci_ctx* ctx = C_;
            if (!ctx->yz_valid) { LAUNCH(launch_pack_yz(ctx->V, ctx->cur, 0, ctx->stream)); ctx->ycur = 0; ctx->yz_valid = true; }
        }
        // (all shards of a slab are restarted together, so every rank takes this branch in the same step)
        EACH { oci_ctx* ctx = C_; LAUNCH(launch_shard_push(ctx->V, ctx->ycur, -1, -1, tol, ctx->xtag + 1, ctx->stream)); }
        EACH { oci_ctx* ctx = C_; LAUNCH(launch_shard_pull(ctx->V, ctx->ycur, -1, -1, tol, ctx->xtag + 1, ctx->stream)); }
        EACH C_->xtag += 1;
    }
    EACH { oci_ctx* ctx = C_; ctx->psi_valid = false; LAUNCH(launch_reduced_pass(ctx, PASS_FIX, ctx->ycur, 0, -1, tol, 0, 0)); }
    int32_t done_iters = 0;
    bool conv = false;
    double d = 0.0, r = 0.0;
    const int32_t guess = ctx->predicted[0] > 0 ? ctx->predicted[0] + 1 : 8;
    while (done_iters < max_iters && !conv) {
        int32_t cnt = guess - done_iters;
        if (cnt < 4) cnt = 4;
        if (cnt > kNormSlots) cnt = kNormSlots;
        if (cnt > max_iters - done_iters) cnt = max_iters - done_iters;
        if (done_iters > 0) EACH { oci_ctx* ctx = C_; CK(cudaMemsetAsync(ctx->V.norms, 0, sizeof(unsigned long long) * 2 * cnt, ctx->stream)); }
        for (int32_t i = 0; i < cnt; ++i) {
            EACH { oci_ctx* ctx = C_; LAUNCH(launch_reduced_pass(ctx, PASS_ITER, (ctx->ycur + done_iters + i) & 1, i, i - 1, tol, 0, 0)); }
            EACH { oci_ctx* ctx = C_; LAUNCH(launch_shard_push(ctx->V, (ctx->ycur + done_iters + i + 1) & 1, i, i - 1, tol, ctx->xtag + 1 + i, ctx->stream)); }
            EACH { oci_ctx* ctx = C_; LAUNCH(launch_shard_pull(ctx->V, (ctx->ycur + done_iters + i + 1) & 1, i, i - 1, tol, ctx->xtag + 1 + i, ctx->stream)); }
        }
        EACH { oci_ctx* ctx = C_; LAUNCH(launch_reduced_pass(ctx, PASS_FINAL, (ctx->ycur + done_iters) & 1, 0, -1, tol, cnt, done_iters + cnt >= max_iters)); }
        // the norms are global after the pull, so any shard's copy tells the iteration count
        CK(cudaMemcpyAsync(ctx->h_norms, ctx->V.norms, sizeof(unsigned long long) * 2 * cnt, cudaMemcpyDeviceToHost, ctx->stream));
        EACH { oci_ctx* ctx = C_; CK(cudaStreamSynchronize(ctx->stream)); }
        CK(cudaGetLastError());
        int32_t executed = cnt;
        for (int32_t i = 0; i < cnt; ++i) {
            std::memcpy(&d, &ctx->h_norms[2 * i], 8);
            std::memcpy(&r, &ctx->h_norms[2 * i + 1], 8);
            if (stop_now(tol, d, r)) { conv = true; executed = i + 1; break; }
        }
        done_iters += executed;
        EACH C_->xtag += (unsigned long long)executed;                      // exchanges that really ran: parities keep alternating
    }
    EACH {
        C_->ycur = (C_->ycur + done_iters) & 1;
        C_->predicted[0] = done_iters;
    }
#undef EACH
#undef C_
    if (iters) *iters = done_iters;
    if (!finite_norms(d, r)) {
        if (resid) *resid = d;
        return fail(ctx, OCI_E_NONFINITE, "the scalar flux became NaN or Inf (non-finite input or overflow); restart with oci_set_flux");
    }
    if (resid) *resid = (r > 0.0) ? d / r : d;
    return conv ? OCI_OK : OCI_NOT_CONVERGED;
}

int run_step(oci_ctx* ctx, bool si, double tol, int32_t max_iters, int32_t* iters, double* resid)
{
    if (!ctx) return OCI_E_INVALID;
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "step before oci_setup");
    if (!ctx->have_flux) return fail(ctx, OCI_E_ORDER, "step before oci_set_flux");
    if (max_iters < 1 || tol != tol) return fail(ctx, OCI_E_INVALID, "max_iters < 1 or tol is NaN");
    const bool halo = ctx->bcL.kind == OCI_BC_HALO || ctx->bcR.kind == OCI_BC_HALO;
    if (halo && !ctx->sharded) return fail(ctx, OCI_E_ORDER, "a context with an OCI_BC_HALO face must be attached with oci_shard_attach");
    if (ctx->sharded) {
        if (si) return fail(ctx, OCI_E_INVALID, "si_step is not available on a sharded context");
        oci_ctx* one = ctx;
        return run_step_sharded(&one, 1, tol, max_iters, iters, resid);
    }
    DeviceGuard guard(ctx);
    DevView& V = ctx->V;
    cudaStream_t s = ctx->stream;
    const bool red = !si && resolved_iteration(ctx) == OCI_ITERATION_REDUCED;
    const bool timed = ctx->timing && !si;
    const bool si_fast = si && si_fast_supported(V);                     // phi-only iterations, Psi once at the end

    int32_t done_iters = 0;
    bool conv = false;
    double d = 0.0, r = 0.0;
    // small shared-block problems: FIX, all iterations and FINAL in ONE launch on one cluster (oci_reduced_small.cu);
    // the per-kernel timing of the roofline reports keeps the three passes apart
    const bool small = red && ctx->small_cluster > 0 && !timed && resolved_iteration(ctx) == OCI_ITERATION_REDUCED;
    if (red) {
        if (!ctx->yz_valid) {
            LAUNCH(launch_pack_yz(V, ctx->cur, 0, s));
            ctx->ycur = 0;
            ctx->yz_valid = true;
        }
        ctx->psi_valid = false;
    }
    if (small) {
        const int32_t cnt = max_iters < kNormSlots ? max_iters : kNormSlots;
        V.host_pub = ctx->d_pub;
        V.pub_seq = ++ctx->pub_seq;
        LAUNCH(launch_red_small(V, ctx->small_cluster, ctx->ycur, tol, cnt, cnt >= max_iters, s));
        V.host_pub = nullptr;
        int32_t executed = 0;
        if (int rc = wait_published(ctx, ctx->pub_seq, &executed, &d, &r)) return rc;   // the one read-back (a7), no copy
        conv = stop_now(tol, d, r);
        done_iters = executed;
        // (not converged and max_iters not reached: the three-pass kernels go on from the state the kernel left)
    } else if (red) {
        if (timed) CK(cudaEventRecord(ctx->ev_aux[0], s));
        LAUNCH(launch_reduced_pass(ctx, PASS_FIX, ctx->ycur, 0, -1, tol, 0, 0));   // a2 (+ a8 of the previous step)
        if (timed) CK(cudaEventRecord(ctx->ev_aux[1], s));
    } else {
        LAUNCH(ensure_psi(ctx));
        ctx->yz_valid = false;
        const bool si_small = si_fast && ctx->si_small_cluster > 0 && ctx->d_pub != nullptr;
        if (si_small) {}                                                    // (the one-launch step commits psi_{k-1/2} itself)
        else if (si_fast) LAUNCH(launch_si_fast_begin(V, ctx->cur, s));     // psi_{k-1/2}, compact (+ a8 of the previous step)
        else LAUNCH(launch_cfix(V, ctx->cur, s));                 // a2 (+ a8 of the previous step)
        if (si_small) {
            // small shared-block problems: every iteration and the final sweep in ONE launch on one cluster (si_small.cu)
            const int32_t cnt = max_iters < kNormSlots ? max_iters : kNormSlots;
            V.host_pub = ctx->d_pub;
            V.pub_seq = ++ctx->pub_seq;
            LAUNCH(launch_si_small(V, ctx->si_small_cluster, ctx->cur, tol, cnt, cnt >= max_iters, s));
            V.host_pub = nullptr;
            int32_t executed = 0;
            if (int rc = wait_published(ctx, ctx->pub_seq, &executed, &d, &r)) return rc;   // the one read-back (a7), no copy
            conv = stop_now(tol, d, r);
            done_iters = executed;
            // (not converged and max_iters not reached: the three-kernel iterations go on from the state the kernel left)
        }
    }
    int32_t guess = ctx->predicted[si ? 1 : 0] > 0 ? ctx->predicted[si ? 1 : 0] + 1 : 8;
    while (done_iters < max_iters && !conv) {
        int32_t cnt = guess - done_iters;
        if (cnt < 4) cnt = 4;
        if (cnt > kNormSlots) cnt = kNormSlots;
        const bool loop_kernel = red && ctx->coop && (ctx->red_kernel != OCI_RKERNEL_KTILED || oci_red_ktiled_fuses_loop(V));
        if (loop_kernel) cnt = kNormSlots;                                  // the fused loop stops itself
        if (cnt > max_iters - done_iters) cnt = max_iters - done_iters;
        // (the FIX pass has already cleared the norm slots and the barrier counter for the first chunk)
        if (!(red && done_iters == 0)) CK(cudaMemsetAsync(V.norms, 0, sizeof(unsigned long long) * 2 * cnt, s));
        // the resident and GEMV kernels of the reduced form run the whole chunk of iterations in ONE cooperative launch
        // (grid-wide barrier + device-side stop between iterations): no launch gap, operator staged once
        const bool fused_loop = loop_kernel && cnt > 1;
        // ... and reports its iteration count straight into mapped host memory (publish_step): no copy, no stream sync
        // (small problems only: the report costs the loop's last CTA a system-scope fence and a PCIe write, about 3 us
        // that a large problem's FINAL pass would wait for, while its host part overlaps that pass anyway)
        const bool polled = fused_loop && !timed && ctx->d_pub != nullptr && ctx->J * ctx->n <= 262144;
        if (fused_loop) {
            if (done_iters > 0) CK(cudaMemsetAsync(V.flags + 8, 0, 20, s));  // the grid barrier's arrival counter, the work tickets
            if (timed) CK(cudaEventRecord(ctx->ev[0], s));
            if (polled) { V.host_pub = ctx->d_pub; V.pub_seq = ++ctx->pub_seq; }
            LAUNCH(launch_reduced_pass(ctx, PASS_ITER, (ctx->ycur + done_iters) & 1, 0, -1, tol, cnt, 0));
            V.host_pub = nullptr;
            if (timed) CK(cudaEventRecord(ctx->ev[1], s));
        }
        for (int32_t i = 0; i < cnt && !fused_loop; ++i) {
            if (timed) CK(cudaEventRecord(ctx->ev[2 * i], s));
            if (si_fast) LAUNCH(launch_si_fast_iteration(V, ctx->cur, done_iters + i, i, i - 1, tol, s));
            else if (si) LAUNCH(launch_si_iteration(V, ctx->cur, i, i - 1, tol, s));
            else if (red) LAUNCH(launch_reduced_pass(ctx, PASS_ITER, (ctx->ycur + done_iters + i) & 1, i, i - 1, tol, 0, 0));
            else LAUNCH(launch_oci_iteration_any(ctx, (ctx->cur + done_iters + i) & 1, i, i - 1, tol));
            if (timed) CK(cudaEventRecord(ctx->ev[2 * i + 1], s));
        }
        // The norms are final once the iteration launches are done.  REDUCED form: their read-back goes through a
        // side stream, so the host gets the iteration count while the FINAL pass is still running and the host
        // part of the next step (Python, three launches) overlaps it; everything else stays ordered on `s`.
        const bool side_readback = red && !timed && !polled && ctx->stream2 != nullptr;
        if (side_readback) {
            CK(cudaEventRecord(ctx->ev_norms, s));
            CK(cudaStreamWaitEvent(ctx->stream2, ctx->ev_norms, 0));
            CK(cudaMemcpyAsync(ctx->h_norms, V.norms, sizeof(unsigned long long) * 2 * cnt, cudaMemcpyDeviceToHost, ctx->stream2));
        }
        if (red) {
            // finalisation, queued before the read-back: finds the last iteration on the device and
            // does nothing if this chunk neither converged nor ends at max_iters
            if (timed) CK(cudaEventRecord(ctx->ev_aux[2], s));
            LAUNCH(launch_reduced_pass(ctx, PASS_FINAL, (ctx->ycur + done_iters) & 1, 0, -1, tol, cnt, done_iters + cnt >= max_iters));
            if (timed) CK(cudaEventRecord(ctx->ev_aux[3], s));
        }
        if (si_fast) LAUNCH(launch_si_fast_final(V, ctx->cur, done_iters, tol, cnt, done_iters + cnt >= max_iters, s));
        int32_t executed = cnt;
        if (polled) {
            if (int rc = wait_published(ctx, ctx->pub_seq, &executed, &d, &r)) return rc;   // the one read-back (a7)
            conv = stop_now(tol, d, r);
        } else {
            if (side_readback) {
                CK(cudaStreamSynchronize(ctx->stream2));                    // the one read-back (a7)
            } else {
                CK(cudaMemcpyAsync(ctx->h_norms, V.norms, sizeof(unsigned long long) * 2 * cnt, cudaMemcpyDeviceToHost, s));
                CK(cudaStreamSynchronize(s));                               // the one read-back (a7)
            }
            CK(cudaGetLastError());
            for (int32_t i = 0; i < cnt; ++i) {
                std::memcpy(&d, &ctx->h_norms[2 * i], 8);
                std::memcpy(&r, &ctx->h_norms[2 * i + 1], 8);
                if (stop_now(tol, d, r)) { conv = true; executed = i + 1; break; }
            }
        }
        if (timed && fused_loop) {
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]));
            ctx->kernel_ms += ms;                                           // one launch = `executed` iterations
            ctx->kernel_launches += executed;
        }
        if (timed) {
            for (int32_t i = 0; i < executed && !fused_loop; ++i) {
                float ms = 0.f;
                CK(cudaEventElapsedTime(&ms, ctx->ev[2 * i], ctx->ev[2 * i + 1]));
                ctx->kernel_ms += ms;
                ctx->kernel_launches += 1;
            }
            if (red && (conv || done_iters + cnt >= max_iters)) {
                float ms = 0.f;
                CK(cudaEventElapsedTime(&ms, ctx->ev_aux[2], ctx->ev_aux[3]));
                ctx->aux_ms[1] += ms;
                ctx->aux_launches[1] += 1;
            }
        }
        done_iters += executed;
    }
    if (timed && red && !small) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ctx->ev_aux[0], ctx->ev_aux[1]));
        ctx->aux_ms[0] += ms;
        ctx->aux_launches[0] += 1;
    }
    if (red) ctx->ycur = (ctx->ycur + done_iters) & 1;                     // a8: (y[ycur], z) is the committed state
    else if (!si) ctx->cur = (ctx->cur + done_iters) & 1;                  // a8: pointer convention
    ctx->predicted[si ? 1 : 0] = done_iters;
    if (iters) *iters = done_iters;
    if (!finite_norms(d, r)) {
        if (resid) *resid = d;
        return fail(ctx, OCI_E_NONFINITE, "the scalar flux became NaN or Inf (non-finite input or overflow); restart with oci_set_flux");
    }
    if (resid) *resid = (r > 0.0) ? d / r : d;
    return conv ? OCI_OK : OCI_NOT_CONVERGED;
}

}  // namespace

extern "C" {

int oci_create(oci_ctx** out, int64_t cells, const double* dx, const double* sigma_t, const double* sigma_s,
               double v, double dt, int32_t n_angles, oci_bc left, oci_bc right)
{
    if (!out) return OCI_E_INVALID;
    *out = nullptr;
    if (cells < 1 || !dx || !sigma_t || !sigma_s) return OCI_E_INVALID;
    if (n_angles < 2 || (n_angles & 1) || n_angles > 512) return OCI_E_INVALID;   // oci.h: kernels stage O(4N) doubles per CTA
    if (!(v > 0.0) || !(dt > 0.0) || !std::isfinite(v) || !std::isfinite(dt)) return OCI_E_INVALID;
    if (!bc_ok(left) || !bc_ok(right) || !std::isfinite(left.value) || !std::isfinite(right.value))
        return OCI_E_INVALID;
    for (int64_t j = 0; j < cells; ++j)
        if (!(dx[j] > 0.0) || !(sigma_t[j] >= 0.0) || !(sigma_s[j] >= 0.0) || !std::isfinite(dx[j]) ||
            !std::isfinite(sigma_t[j]) || !std::isfinite(sigma_s[j]))
            return OCI_E_INVALID;
    oci_ctx* c = new (std::nothrow) oci_ctx();
    if (!c) return OCI_E_INVALID;
    c->J = cells;
    c->N = n_angles;
    c->n = 4 * n_angles;
    c->v = v;
    c->dt = dt;
    c->bcL = left;
    c->bcR = right;
    c->dx.assign(dx, dx + cells);
    c->sig.assign(sigma_t, sigma_t + cells);
    c->sigs.assign(sigma_s, sigma_s + cells);
    gauss_legendre(n_angles, c->mu, c->w);
    classify(c);
    *out = c;
    return OCI_OK;
}

int64_t oci_workspace_bytes(const oci_ctx* ctx)
{
    if (!ctx) return 0;
    return make_layout(ctx->J, ctx->N, ctx->nblk).total;
}

int oci_setup(oci_ctx* ctx, void* d_workspace, int64_t bytes, void* cuda_stream)
{
    if (!ctx || !d_workspace) return fail(ctx, OCI_E_INVALID, "NULL context or workspace");
    if (((uintptr_t)d_workspace & 255) != 0) return fail(ctx, OCI_E_INVALID, "workspace not 256-byte aligned");
    const Layout L = make_layout(ctx->J, ctx->N, ctx->nblk);
    if (bytes < L.total) return fail(ctx, OCI_E_WORKSPACE, "workspace too small");
    ctx->ready = false;
    ctx->have_flux = false;
    {
        // the device the workspace lives on is the context's device from here on
        cudaPointerAttributes pa{};
        CK(cudaPointerGetAttributes(&pa, d_workspace));
        if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)
            return fail(ctx, OCI_E_INVALID, "workspace is not device memory");
        ctx->device = pa.device;
    }
    DeviceGuard guard(ctx);
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->ws = d_workspace;
    ctx->ws_bytes = bytes;
    char* base = (char*)d_workspace;
    DevView& V = ctx->V;
    const int64_t n = ctx->n;
    V.J = ctx->J; V.N = ctx->N; V.n = ctx->n; V.nblk = ctx->nblk;
    V.binv = (double*)(base + L.binv);
    V.psi[0] = (double*)(base + L.psi0) + n;      // skip the left ghost row
    V.psi[1] = (double*)(base + L.psi1) + n;
    V.cfix = (double*)(base + L.cfix);
    V.phi = (double*)(base + L.phi);
    V.Q = (double*)(base + L.Q);
    V.qs = (double*)(base + L.qs);
    V.dx = (double*)(base + L.dx);
    V.sig = (double*)(base + L.sig);
    V.sigs = (double*)(base + L.sigs);
    V.blk = (int32_t*)(base + L.blk);
    V.rep = (int64_t*)(base + L.rep);
    V.mu = (double*)(base + L.mu);
    V.w = (double*)(base + L.w);
    V.coef = (double*)(base + L.coef);
    V.ainv4 = (double*)(base + L.ainv4);
    V.si_scan = (double*)(base + L.si_scan);
    V.phi_part = (double*)(base + L.phi_part);
    V.tickets = (int32_t*)(base + L.tickets);
    V.norms = (unsigned long long*)(base + L.norms);
    V.flags = (int32_t*)(base + L.flags);
    V.xop = (double*)(base + L.xop);
    V.rop = (double*)(base + L.rop);
    V.fop = (double*)(base + L.fop);
    V.y[0] = (double*)(base + L.y0) + n / 2;      // skip the left ghost row
    V.y[1] = (double*)(base + L.y1) + n / 2;
    V.z = (double*)(base + L.z);
    V.yfix = (double*)(base + L.yfix);
    V.ifix = (double*)(base + L.ifix);
    V.phifix = (double*)(base + L.phifix);
    V.q16 = (double*)(base + L.q16);
    V.gitems = nullptr;
    V.ngroups = 0;
    V.perm = (int32_t*)(base + L.perm);
    V.team_bar = (int32_t*)(base + L.team_bar);
    V.peers = (unsigned long long*)(base + L.peers);
    ctx->phi_stage = (double*)(base + L.phi_stage);
    V.si_prev = V.cfix;
    V.si_part = (double*)(base + L.si_part);
    V.si_inflow = (double*)(base + L.si_inflow);
    V.si_src1 = (double*)(base + L.si_src1);
    V.si_agg = (double*)(base + L.si_agg);
    V.wba = (double*)(base + L.wba);
    V.wbd = (double*)(base + L.wbd);
    V.wbm = (double*)(base + L.wbm);
    ctx->snap_pending = false;
    V.rank = 0;
    V.world = 1;
    ctx->sharded = false;
    ctx->xtag = 0;
    V.v = ctx->v; V.dt = ctx->dt;
    V.bcL = ctx->bcL.kind; V.bcR = ctx->bcR.kind;
    V.bcLv = ctx->bcL.value; V.bcRv = ctx->bcR.value;
    {
        int sms = 0, coop = 0;
        CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device));
        CK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ctx->device));
        V.sm_count = sms;
        ctx->coop = coop != 0;
        // more than 48 KB of dynamic shared memory is a per-device, per-kernel opt-in
        CK(oci_setup_opt_in());
        CK(oci_shared_fast_opt_in());
        CK(oci_ktiled_opt_in());
        CK(oci_red_gemv_opt_in());
        CK(oci_red_ktiled_opt_in());
        CK(oci_red_resident_opt_in());
        CK(oci_red_opreg_opt_in());
        CK(oci_red_woodbury_opt_in());
        CK(oci_red_small_opt_in());
        CK(si_fast_opt_in());
        CK(si_small_opt_in());
    }

    cudaStream_t s = ctx->stream;
    // coef[4m+s] = |mu_m| on the rows that take an incident flux (eqs. 27,28), else 0
    std::vector<double> coef(n, 0.0);
    for (int m = 0; m < ctx->N; ++m) {
        if (ctx->mu[m] > 0.0) { coef[4 * m + 0] = ctx->mu[m]; coef[4 * m + 2] = ctx->mu[m]; }
        else { coef[4 * m + 1] = -ctx->mu[m]; coef[4 * m + 3] = -ctx->mu[m]; }
    }
    // everything the kernels may read before a set_* call must be finite: zero the state
    CK(cudaMemsetAsync(base + L.psi0, 0, (size_t)(L.cfix - L.psi0), s));
    CK(cudaMemsetAsync(base + L.cfix, 0, (size_t)(L.dx - L.cfix), s));
    CK(cudaMemsetAsync(base + L.phi_part, 0, (size_t)(L.xop - L.phi_part), s));
    CK(cudaMemsetAsync(base + L.y0, 0, (size_t)(L.total - L.y0), s));
    CK(cudaMemcpyAsync(V.dx, ctx->dx.data(), ctx->J * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.sig, ctx->sig.data(), ctx->J * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.sigs, ctx->sigs.data(), ctx->J * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.blk, ctx->blk.data(), ctx->J * 4, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.rep, ctx->rep.data(), ctx->nblk * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.mu, ctx->mu.data(), ctx->N * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.w, ctx->w.data(), ctx->N * 8, cudaMemcpyHostToDevice, s));
    CK(cudaMemcpyAsync(V.coef, coef.data(), n * 8, cudaMemcpyHostToDevice, s));
    CK(cudaStreamSynchronize(s));   // host vectors above are read by the async copies

    if (ctx->nblk > 1 && ctx->nblk <= kMaxGroupedBlocks && ctx->N % 16 == 0) {
        // row f2: list, tile by tile, the blocks present and which of the tile's 64 cells have each
        std::vector<int32_t> items;
        const int64_t nct = (ctx->J + 63) / 64;
        for (int64_t ct = 0; ct < nct; ++ct) {
            const int64_t j0 = ct * 64, j1 = j0 + 64 < ctx->J ? j0 + 64 : ctx->J;
            for (int64_t ja = j0; ja < j1; ++ja) {
                const int32_t b = ctx->blk[ja];
                bool first = true;
                for (int64_t jb = j0; jb < ja; ++jb) first = first && ctx->blk[jb] != b;
                if (!first) continue;
                uint64_t mask = 0;
                for (int64_t jb = ja; jb < j1; ++jb)
                    if (ctx->blk[jb] == b) mask |= 1ull << (jb - j0);
                items.push_back((int32_t)ct);
                items.push_back(b);
                items.push_back((int32_t)(uint32_t)(mask & 0xffffffffull));
                items.push_back((int32_t)(uint32_t)(mask >> 32));
            }
        }
        V.gitems = (int32_t*)(base + L.gitems);
        V.ngroups = (int64_t)items.size() / 4;
        CK(cudaMemcpyAsync(V.gitems, items.data(), items.size() * 4, cudaMemcpyHostToDevice, s));
        CK(cudaStreamSynchronize(s));
    }

    if (ctx->ev.empty()) {
        ctx->ev.resize(2 * kNormSlots);
        for (auto& e : ctx->ev) CK(cudaEventCreate(&e));
        for (auto& e : ctx->ev_aux) CK(cudaEventCreate(&e));
    }
    CK(cudaEventRecord(ctx->ev[0], s));
    LAUNCH(launch_form_and_invert(V, s));                                // a0, a1
    LAUNCH(launch_pack_operators(V, s));                                 // f1: G, H, F
    LAUNCH(launch_woodbury_setup(V, s));                                 // f3: per-angle inverses element-major, M
    CK(cudaEventRecord(ctx->ev[1], s));
    int32_t flag = 0;
    CK(cudaMemcpyAsync(&flag, V.flags, 4, cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    CK(cudaGetLastError());
    {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, ctx->ev[0], ctx->ev[1]));
        ctx->setup_ms = ms;
    }
    if (flag != 0) {
        char buf[96];
        std::snprintf(buf, sizeof buf, "block %d is singular", flag - 1);
        return fail(ctx, OCI_E_SINGULAR, buf);
    }
    if (!ctx->h_norms) CK(cudaHostAlloc((void**)&ctx->h_norms, sizeof(unsigned long long) * 2 * kNormSlots, cudaHostAllocDefault));
    if (!ctx->h_pub) {
        CK(cudaHostAlloc((void**)&ctx->h_pub, 64, cudaHostAllocMapped));
        std::memset(ctx->h_pub, 0, 64);
        CK(cudaHostGetDevicePointer((void**)&ctx->d_pub, ctx->h_pub, 0));
    }
    V.host_pub = nullptr;
    V.pub_seq = 0;
    if (!ctx->stream2) {
        CK(cudaStreamCreateWithFlags(&ctx->stream2, cudaStreamNonBlocking));
        CK(cudaEventCreateWithFlags(&ctx->ev_norms, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->ev_snap, cudaEventDisableTiming));
        CK(cudaEventCreateWithFlags(&ctx->ev_snap_done, cudaEventDisableTiming));
    }
    ctx->use_ktiled = ctx->path == OCI_PATH_SHARED && !oci_shared_fast_supported(V) && oci_ktiled_supported(V) &&
                      oci_ktiled_prepare(V, &ctx->maps);
    {
        const int32_t want = ctx->forced_rkernel;
        auto may = [&](int32_t k) { return want == OCI_RKERNEL_AUTO || want == k; };
        if (want == OCI_RKERNEL_WOODBURY)                 // only on request: the dense families are the general method
            ctx->red_kernel = OCI_RKERNEL_WOODBURY;
        else if (may(OCI_RKERNEL_RESIDENT) && oci_red_resident_supported(V) && oci_red_resident_prepare(V, &ctx->rrmaps))
            ctx->red_kernel = OCI_RKERNEL_RESIDENT;
        else if (may(OCI_RKERNEL_OPREG) && oci_red_opreg_supported(V) && oci_red_opreg_prepare(V, &ctx->romaps))
            ctx->red_kernel = OCI_RKERNEL_OPREG;
        else if (may(OCI_RKERNEL_KTILED) && oci_red_ktiled_supported(V) && oci_red_ktiled_prepare(V, &ctx->rmaps))
            ctx->red_kernel = OCI_RKERNEL_KTILED;
        else if (may(OCI_RKERNEL_GEMV))
            ctx->red_kernel = OCI_RKERNEL_GEMV;
        else
            return fail(ctx, OCI_E_INVALID, "the kernel family forced with oci_set_reduced_kernel does not serve this problem");
    }
    {
        // the one-launch step (oci_reduced_small.cu): by itself for small problems on the default kernel family, never when
        // a family has been forced (tests and comparisons of the families), on request if the problem fits
        int cc = 0;
        CK(cudaDeviceGetAttribute(&cc, cudaDevAttrClusterLaunch, ctx->device));
        const int C = cc ? oci_red_small_cluster(V) : 0;
        ctx->small_cluster = 0;
        if (ctx->small_mode == 1) {
            if (C == 0) return fail(ctx, OCI_E_INVALID, "oci_set_small_step(1): the one-launch step does not serve this problem");
            ctx->small_cluster = C;
        } else if (ctx->small_mode == -1 && ctx->forced_rkernel == OCI_RKERNEL_AUTO && (C == 1 || C == 16)) {
            // measured: the one-CTA form wins (config 1: 0.064 -> 0.039 ms per step) and so does a cluster of 16 CTAs
            // where the device schedules one (config 2: 0.088 -> 0.072 ms; every size it serves: DESIGN.md 6.9); a
            // cluster of 8 is level with the three-pass kernels and runs on request only
            ctx->small_cluster = C;
        }
        // the comparator gets the same treatment at the same sizes (same switch: oci_set_small_step); any cluster size it
        // fits wins against three launches per iteration (6 us against 20 us per iteration at config 2)
        ctx->si_small_cluster = cc && ctx->small_mode != 0 ? si_small_cluster(V) : 0;
    }
    ctx->cur = 0;
    ctx->ycur = 0;
    ctx->yz_valid = false;
    ctx->psi_valid = true;
    ctx->predicted[0] = ctx->predicted[1] = 0;
    ctx->ready = true;
    return OCI_OK;
}

static int set_flux_common(oci_ctx* ctx, const double* d_edge)
{
    LAUNCH(launch_set_flux(ctx->V, d_edge, 0, ctx->stream));
    ctx->cur = 0;
    ctx->yz_valid = false;
    ctx->psi_valid = true;
    LAUNCH(launch_phi_norm(ctx->V, 0, 0, -1, -1.0, false, ctx->stream));   // phi^(0), ghost rows
    const bool halo = ctx->bcL.kind == OCI_BC_HALO || ctx->bcR.kind == OCI_BC_HALO;
    if (resolved_iteration(ctx) == OCI_ITERATION_REDUCED && !ctx->sharded && !halo) {
        // the packed layout the REDUCED steps work in belongs to setting the flux, not to the first step after it
        // (both layouts are valid from here on; a step of either form invalidates the other one).  A shard packs in its
        // first step instead, where the neighbours' edge values are exchanged as well.
        LAUNCH(launch_pack_yz(ctx->V, ctx->cur, 0, ctx->stream));
        ctx->ycur = 0;
        ctx->yz_valid = true;
    }
    CK(cudaStreamSynchronize(ctx->stream));
    CK(cudaGetLastError());
    ctx->have_flux = true;
    return OCI_OK;
}

int oci_set_flux(oci_ctx* ctx, const double* psi_edge)
{
    if (!ctx || !psi_edge) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_set_flux before oci_setup");
    DeviceGuard guard(ctx);
    // stage through c_fix (recomputed at the start of every step, and at least as large)
    CK(cudaMemcpyAsync(ctx->V.cfix, psi_edge, (size_t)ctx->J * ctx->N * 2 * 8, cudaMemcpyHostToDevice, ctx->stream));
    return set_flux_common(ctx, ctx->V.cfix);
}

int oci_set_flux_dev(oci_ctx* ctx, const double* d_psi_edge)
{
    if (!ctx || !d_psi_edge) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_set_flux_dev before oci_setup");
    DeviceGuard guard(ctx);
    return set_flux_common(ctx, d_psi_edge);
}

// Q padded to one 128-byte row per cell for the K-tiled FIX pass (a strided copy, the pad stays zero)
static int refresh_q16(oci_ctx* ctx)
{
    if (ctx->red_kernel != OCI_RKERNEL_KTILED && ctx->red_kernel != OCI_RKERNEL_OPREG) return OCI_OK;
    CK(cudaMemcpy2DAsync(ctx->V.q16, 128, ctx->V.Q, 32, 32, (size_t)ctx->J, cudaMemcpyDeviceToDevice, ctx->stream));
    return OCI_OK;
}

int oci_set_source(oci_ctx* ctx, const double* q)
{
    if (!ctx) return OCI_E_INVALID;
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_set_source before oci_setup");
    DeviceGuard guard(ctx);
    if (q) CK(cudaMemcpyAsync(ctx->V.Q, q, (size_t)ctx->J * 4 * 8, cudaMemcpyHostToDevice, ctx->stream));
    else CK(cudaMemsetAsync(ctx->V.Q, 0, (size_t)ctx->J * 4 * 8, ctx->stream));
    if (int rc = refresh_q16(ctx)) return rc;
    if (q) CK(cudaStreamSynchronize(ctx->stream));      // the caller may reuse its buffer at once; Q = 0 needs no host data
    return OCI_OK;
}

int oci_set_source_dev(oci_ctx* ctx, const double* d_q)
{
    if (!ctx) return OCI_E_INVALID;
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_set_source_dev before oci_setup");
    DeviceGuard guard(ctx);
    if (d_q) CK(cudaMemcpyAsync(ctx->V.Q, d_q, (size_t)ctx->J * 4 * 8, cudaMemcpyDeviceToDevice, ctx->stream));
    else CK(cudaMemsetAsync(ctx->V.Q, 0, (size_t)ctx->J * 4 * 8, ctx->stream));
    return refresh_q16(ctx);
}

int oci_step(oci_ctx* ctx, double tol, int32_t max_iters, int32_t* iters, double* resid)
{
    return run_step(ctx, false, tol, max_iters, iters, resid);
}

int si_step(oci_ctx* ctx, double tol, int32_t max_iters, int32_t* iters, double* resid)
{
    return run_step(ctx, true, tol, max_iters, iters, resid);
}

static int unpack_for_get(oci_ctx* ctx)
{
    if (!ctx || !ctx->ready) return OCI_OK;          // get_common reports these
    DeviceGuard guard(ctx);
    LAUNCH(ensure_psi(ctx));
    return OCI_OK;
}

static int get_common(const oci_ctx* ctx, double* dst, const double* src, size_t bytes, cudaMemcpyKind kind, bool sync)
{
    if (!ctx || !dst) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "get before oci_setup");
    DeviceGuard guard(ctx);
    CK(cudaMemcpyAsync(dst, src, bytes, kind, ctx->stream));
    if (sync) CK(cudaStreamSynchronize(ctx->stream));
    return OCI_OK;
}

int oci_get_scalar_flux(const oci_ctx* ctx, double* phi)
{
    return get_common(ctx, phi, ctx ? ctx->V.phi : nullptr, ctx ? (size_t)ctx->J * 32 : 0, cudaMemcpyDeviceToHost, true);
}
int oci_get_angular_flux(const oci_ctx* ctx, double* psi)
{
    if (int rc = unpack_for_get(const_cast<oci_ctx*>(ctx))) return rc;
    return get_common(ctx, psi, ctx ? ctx->V.psi[ctx->cur] : nullptr, ctx ? (size_t)ctx->J * ctx->n * 8 : 0,
                      cudaMemcpyDeviceToHost, true);
}
int oci_get_scalar_flux_dev(const oci_ctx* ctx, double* d_phi)
{
    return get_common(ctx, d_phi, ctx ? ctx->V.phi : nullptr, ctx ? (size_t)ctx->J * 32 : 0, cudaMemcpyDeviceToDevice, false);
}
int oci_get_angular_flux_dev(const oci_ctx* ctx, double* d_psi)
{
    if (int rc = unpack_for_get(const_cast<oci_ctx*>(ctx))) return rc;
    return get_common(ctx, d_psi, ctx ? ctx->V.psi[ctx->cur] : nullptr, ctx ? (size_t)ctx->J * ctx->n * 8 : 0,
                      cudaMemcpyDeviceToDevice, false);
}

int oci_get_scalar_flux_async(oci_ctx* ctx, double* phi_pinned)
{
    if (!ctx || !phi_pinned) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "get before oci_setup");
    DeviceGuard guard(ctx);
    const size_t bytes = (size_t)ctx->J * 32;
    // the staging array is free once the previous snapshot has left it
    if (ctx->snap_pending) CK(cudaStreamWaitEvent(ctx->stream, ctx->ev_snap_done, 0));
    CK(cudaMemcpyAsync(ctx->phi_stage, ctx->V.phi, bytes, cudaMemcpyDeviceToDevice, ctx->stream));
    CK(cudaEventRecord(ctx->ev_snap, ctx->stream));
    CK(cudaStreamWaitEvent(ctx->stream2, ctx->ev_snap, 0));
    CK(cudaMemcpyAsync(phi_pinned, ctx->phi_stage, bytes, cudaMemcpyDeviceToHost, ctx->stream2));
    CK(cudaEventRecord(ctx->ev_snap_done, ctx->stream2));
    ctx->snap_pending = true;
    return OCI_OK;
}

int oci_synchronize(oci_ctx* ctx)
{
    if (!ctx) return OCI_E_INVALID;
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_synchronize before oci_setup");
    DeviceGuard guard(ctx);
    CK(cudaStreamSynchronize(ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream2));
    ctx->snap_pending = false;
    return OCI_OK;
}

int oci_get_quadrature(const oci_ctx* ctx, double* mu, double* w)
{
    if (!ctx || !mu || !w) return fail(ctx, OCI_E_INVALID, "NULL argument");
    std::memcpy(mu, ctx->mu.data(), ctx->N * 8);
    std::memcpy(w, ctx->w.data(), ctx->N * 8);
    return OCI_OK;
}

int oci_get_info(const oci_ctx* ctx, oci_info* info)
{
    if (!ctx || !info) return fail(ctx, OCI_E_INVALID, "NULL argument");
    info->cells = ctx->J;
    info->n_angles = ctx->N;
    info->block_dim = ctx->n;
    info->n_blocks = ctx->nblk;
    info->path = ctx->path;
    info->apply_kernel = ctx->path == OCI_PATH_PER_CELL ? OCI_KERNEL_PER_CELL
                         : (ctx->ready && oci_shared_fast_supported(ctx->V)) ? OCI_KERNEL_RESIDENT
                         : ctx->use_ktiled ? OCI_KERNEL_KTILED : OCI_KERNEL_GENERIC;
    info->iteration = resolved_iteration(ctx);
    info->reduced_kernel = ctx->red_kernel;
    info->small_step_cluster = ctx->small_cluster;
    info->si_small_step_cluster = ctx->si_small_cluster;
    return OCI_OK;
}

int oci_get_block_inverse(const oci_ctx* ctx, int64_t blk, double* binv)
{
    if (!ctx || !binv) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_get_block_inverse before oci_setup");
    if (blk < 0 || blk >= ctx->nblk) return fail(ctx, OCI_E_INVALID, "block index out of range");
    const size_t nn = (size_t)ctx->n * ctx->n;
    DeviceGuard guard(ctx);
    CK(cudaMemcpyAsync(binv, ctx->V.binv + (size_t)blk * nn, nn * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return OCI_OK;
}

int oci_enable_kernel_timing(oci_ctx* ctx, int32_t on)
{
    if (!ctx) return OCI_E_INVALID;
    ctx->timing = on != 0;
    ctx->kernel_ms = 0.0;
    ctx->kernel_launches = 0;
    ctx->aux_ms[0] = ctx->aux_ms[1] = 0.0;
    ctx->aux_launches[0] = ctx->aux_launches[1] = 0;
    return OCI_OK;
}

int oci_get_aux_kernel_time(oci_ctx* ctx, double* fix_ms, int64_t* fix_launches, double* final_ms, int64_t* final_launches)
{
    if (!ctx) return OCI_E_INVALID;
    if (fix_ms) *fix_ms = ctx->aux_ms[0];
    if (fix_launches) *fix_launches = ctx->aux_launches[0];
    if (final_ms) *final_ms = ctx->aux_ms[1];
    if (final_launches) *final_launches = ctx->aux_launches[1];
    ctx->aux_ms[0] = ctx->aux_ms[1] = 0.0;
    ctx->aux_launches[0] = ctx->aux_launches[1] = 0;
    return OCI_OK;
}

int oci_set_iteration(oci_ctx* ctx, int32_t iteration)
{
    if (!ctx) return OCI_E_INVALID;
    if (iteration != OCI_ITERATION_FULL && iteration != OCI_ITERATION_REDUCED && iteration != OCI_ITERATION_AUTO)
        return fail(ctx, OCI_E_INVALID, "unknown iteration form");
    ctx->iteration = iteration;
    return OCI_OK;
}

int64_t oci_shard_mailbox_bytes(int32_t n_angles, int32_t world)
{
    if (n_angles < 2 || world < 1 || world > 64) return 0;
    return 8 * (4 * (int64_t)n_angles + 4 * (int64_t)world + (int64_t)world);
}

int oci_shard_attach(oci_ctx* ctx, int32_t rank, int32_t world, void* const* d_mailboxes)
{
    if (!ctx || !d_mailboxes) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_shard_attach before oci_setup");
    if (world < 1 || world > 64 || rank < 0 || rank >= world) return fail(ctx, OCI_E_INVALID, "rank / world out of range (world <= 64)");
    if ((ctx->bcL.kind == OCI_BC_HALO) != (rank > 0) || (ctx->bcR.kind == OCI_BC_HALO) != (rank < world - 1))
        return fail(ctx, OCI_E_INVALID, "exactly the cut faces of a shard must be OCI_BC_HALO");
    unsigned long long ptrs[64] = {0};
    for (int32_t r = 0; r < world; ++r) {
        if (!d_mailboxes[r] || ((uintptr_t)d_mailboxes[r] & 15) != 0) return fail(ctx, OCI_E_INVALID, "NULL or misaligned mailbox");
        ptrs[r] = (unsigned long long)(uintptr_t)d_mailboxes[r];
    }
    DeviceGuard guard(ctx);
    CK(cudaMemcpyAsync(ctx->V.peers, ptrs, sizeof(unsigned long long) * world, cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaMemsetAsync(d_mailboxes[rank], 0, (size_t)oci_shard_mailbox_bytes(ctx->N, world), ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));                                 // `ptrs` is on the stack
    ctx->V.rank = rank;
    ctx->V.world = world;
    ctx->sharded = true;
    ctx->xtag = 0;
    ctx->iteration = OCI_ITERATION_REDUCED;
    return OCI_OK;
}

int oci_shard_step(oci_ctx* const* ctxs, int32_t n, double tol, int32_t max_iters, int32_t* iters, double* resid)
{
    if (!ctxs || n < 1 || !ctxs[0]) return OCI_E_INVALID;
    return run_step_sharded(ctxs, n, tol, max_iters, iters, resid);
}

int oci_set_reduced_kernel(oci_ctx* ctx, int32_t kernel)
{
    if (!ctx) return OCI_E_INVALID;
    if (kernel < OCI_RKERNEL_AUTO || kernel > OCI_RKERNEL_WOODBURY) return fail(ctx, OCI_E_INVALID, "unknown kernel family");
    ctx->forced_rkernel = kernel;
    return OCI_OK;
}

int oci_set_small_step(oci_ctx* ctx, int32_t mode)
{
    if (!ctx) return OCI_E_INVALID;
    if (mode < -1 || mode > 1) return fail(ctx, OCI_E_INVALID, "oci_set_small_step: mode must be -1, 0 or 1");
    ctx->small_mode = mode;
    return OCI_OK;
}

int oci_get_kernel_time(oci_ctx* ctx, double* ms, int64_t* launches)
{
    if (!ctx) return OCI_E_INVALID;
    if (ms) *ms = ctx->kernel_ms;
    if (launches) *launches = ctx->kernel_launches;
    ctx->kernel_ms = 0.0;
    ctx->kernel_launches = 0;
    return OCI_OK;
}

int oci_get_setup_time(const oci_ctx* ctx, double* ms)
{
    if (!ctx || !ms) return fail(ctx, OCI_E_INVALID, "NULL argument");
    if (!ctx->ready) return fail(ctx, OCI_E_ORDER, "oci_get_setup_time before oci_setup");
    *ms = ctx->setup_ms;
    return OCI_OK;
}

int64_t oci_launch_count(const oci_ctx* ctx) { return ctx ? ctx->launches : 0; }

const char* oci_last_error(const oci_ctx* ctx) { return ctx ? ctx->err.c_str() : "NULL context"; }

void oci_destroy(oci_ctx* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx);
    if (ctx->h_norms) cudaFreeHost(ctx->h_norms);
    if (ctx->h_pub) cudaFreeHost(ctx->h_pub);
    if (ctx->stream2) cudaStreamDestroy(ctx->stream2);
    if (ctx->ev_norms) cudaEventDestroy(ctx->ev_norms);
    if (ctx->ev_snap) cudaEventDestroy(ctx->ev_snap);
    if (ctx->ev_snap_done) cudaEventDestroy(ctx->ev_snap_done);
    for (auto& e : ctx->ev) cudaEventDestroy(e);
    for (auto& e : ctx->ev_aux) if (e) cudaEventDestroy(e);
    delete ctx;
}

}  // extern "C"
