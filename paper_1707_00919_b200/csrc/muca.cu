// paper_1707_00919_b200/csrc/muca.cu -- host side of libmuca_b200 (C ABI declared in include/muca.h).
// Context, threshold-table build (double, host libm: DESIGN.md R12), weight update (Eq. (4)), launch logic.
// There is NO CPU fallback: every compute entry point needs a CUDA device and fails with MUCA_ECUDA otherwise.
#include "../../include/muca.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <mutex>
#include <utility>
#include <new>
#include <vector>

#include "muca_device.cuh"
#include "muca_resident.cuh"
#include "muca_random_site.cuh"
#include "muca_streamed.cuh"

using namespace muca;

struct muca_ctx {
    int L = 0, N = 0, W = 0, n_bins = 0;
    uint64_t seed = 0;
    uint32_t walker_offset = 0;
    uint32_t iteration = 0;
    cudaStream_t stream = nullptr;
    bool own_workspace = false;
    void* d_workspace = nullptr;
    // carved from the workspace
    uint32_t* d_spins = nullptr;
    int32_t* d_E = nullptr;
    uint32_t* d_table = nullptr;
    unsigned long long* d_H = nullptr;
    void* d_stage = nullptr;        // W*N bytes for muca_get_spins / muca_set_spins (in the workspace: a cudaMalloc per
                                    // context of 128 MB at configs 4 and 5 stalled for up to 0.3 s now and then)
    // host state
    std::vector<double> logw;       // omega, n_bins
    std::vector<uint64_t> H;        // last histogram
    uint32_t* h_table = nullptr;    // pinned, n_bins*8
    unsigned long long* h_H = nullptr;  // pinned, n_bins
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    double last_sweep_ms = 0.0;
    int last_launches = 0;
    int opt_kernel = MUCA_KERNEL_AUTO;
    int opt_tpb = 0;
    int opt_max_sweeps = 0;
    int opt_wpw = 0;
    int opt_role_map = 0;           // MUCA_OPT_ROLE_MAP (resident kernel, 4 pairs per block)
    int opt_window_rows = 0;        // MUCA_OPT_TABLE_WINDOW_ROWS: 0 = as many table rows as shared memory holds
    void* d_snap = nullptr;         // snapshot of spins + E for the windowed kernels' fallback (in the workspace, L >= 32)
    int* d_flag = nullptr;          // device int[4]: window-left flag, smallest / largest slot of the walkers
    int* h_flag = nullptr;          // pinned copy (tail of h_H's allocation)
    int stat_window_iterations = 0, stat_window_fallbacks = 0;
    int win_margin = 8;             // rows asked for between the outermost walker and a sentinel; grows after a fallback
    int* d_perm = nullptr;          // sorted-window launches: walker served by position i of the launch (in the workspace, L >= 32)
    int* d_blk_jlo = nullptr;       // ... and the first table row of every block's window
    unsigned long long* d_Hsnap = nullptr;   // ... and the histogram as it was before the launch
    int32_t* h_E = nullptr;         // pinned: energies, then the permutation and the window starts (3 W ints)
    int stat_sorted_launches = 0;
    int conv_w_prev = 0;            // width covered by the previous iteration of muca_converge (0: none yet)
    double conv_n_updates = 0.0;    // N_updates (flips per walker) of the previous iteration of muca_converge
    int opt_scheme = MUCA_SCHEME_TYPEWRITER;   // update scheme used by muca_converge / muca_production
    int opt_acceptance = MUCA_ACCEPT_THRESHOLD;   // MUCA_OPT_ACCEPTANCE (random-site scheme only)
    int conv_full = 0;              // the previous iteration already worked on the whole energy range
    int device = 0;                 // CUDA device the context lives on: every entry point selects it (DeviceGuard)
    int n_sm = 0;
    int max_smem_optin = 0;         // cudaDevAttrMaxSharedMemoryPerBlockOptin of that device
    char err[512] = {0};
};

namespace {

constexpr size_t ALIGN = 256;
inline size_t align_up(size_t x) { return (x + ALIGN - 1) / ALIGN * ALIGN; }

bool valid_L(int L) { return L == 8 || L == 16 || L == 32 || L == 64 || L == 128; }

struct Carve { size_t spins, E, table, H, flag, snap, perm, blkwin, hsnap, stage, total; };
Carve carve(int L, int W) {
    const size_t N = (size_t)L * L, bins = N + 1;
    Carve c;
    size_t off = 0;
    c.spins = off; off += align_up((size_t)W * (N / 8));
    c.E = off;     off += align_up((size_t)W * 4);
    c.table = off; off += align_up(bins * 8 * 4);
    c.H = off;     off += align_up(bins * 8);
    c.flag = off;  off += align_up(4 * sizeof(int));                       // windowed kernels: left-the-window flag, slot range
    c.snap = off;  off += L >= 32 ? align_up((size_t)W * (N / 8)) + align_up((size_t)W * 4) : 0;   // and their snapshot of spins + E
    c.perm = off;  off += L >= 32 ? align_up((size_t)W * 4) : 0;           // sorted-window launches (L >= 32): permutation,
    c.blkwin = off; off += L >= 32 ? align_up((size_t)((W + 31) / 32) * 4) : 0;   // window start per block,
    c.hsnap = off; off += L >= 32 ? align_up(bins * 8) : 0;                 // histogram before the launch
    c.stage = off; off += align_up((size_t)W * N);                        // int8 spins of muca_get_spins / muca_set_spins
    c.total = off;
    return c;
}

int fail(muca_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CU(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return fail(ctx, MUCA_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),     \
                        __FILE__, __LINE__);                                                         \
    } while (0)

// Every entry point that touches the device runs with the context's device current and restores the caller's.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const muca_ctx* c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (device, kernel): remembered per device, only ever raised.
int ensure_dynamic_smem(muca_ctx* ctx, const void* kernel, size_t bytes) {
    static std::mutex m;
    static std::map<std::pair<int, const void*>, size_t> configured;
    std::lock_guard<std::mutex> g(m);
    size_t& have = configured[std::make_pair(ctx->device, kernel)];
    if (bytes > have) {
        CU(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
        have = bytes;
    }
    return MUCA_OK;
}
#define SMEM(kernel, bytes)                                                             \
    do {                                                                                \
        const int rc_ = ensure_dynamic_smem(ctx, (const void*)(kernel), (bytes));       \
        if (rc_ != MUCA_OK) return rc_;                                                 \
    } while (0)

// Acceptance thresholds thresh[j][a], a = 0..4 (include/muca.h, muca_run_iteration step 1, R6/R7/R9).
void build_thresholds5(const std::vector<double>& omega, std::vector<uint32_t>& t5) {
    const int bins = (int)omega.size();
    t5.assign((size_t)bins * 5, 0u);
    const double two32 = 4294967296.0;
    for (int j = 0; j < bins; ++j)
        for (int a = 0; a < 5; ++a) {
            uint32_t t = 0u;
            const int jn = j + 2 - a;
            if (a == 2) t = 0xFFFFFFFFu;
            else if (jn >= 0 && jn < bins) {
                const double d = omega[jn] - omega[j];
                if (d >= 0.0) t = 0xFFFFFFFFu;
                else {
                    double T = std::floor(std::ldexp(std::exp(d), 32));
                    if (T < 1.0) T = 1.0;
                    if (T > two32) T = two32;
                    t = (uint32_t)((uint64_t)T - 1u);
                }
            }
            t5[(size_t)j * 5 + a] = t;
        }
}

// Device format T8[j][f], f = 4*hi + 2*lo + g, a = (lo + 2*hi) + g  (muca_device.cuh).
void expand_table8(const std::vector<uint32_t>& t5, int bins, uint32_t* t8) {
    for (int j = 0; j < bins; ++j)
        for (int f = 0; f < 8; ++f) {
            const int a = (f >> 1) + (f & 1);
            t8[(size_t)j * 8 + f] = t5[(size_t)j * 5 + a];
        }
}

template <int L>
int launch_sweep_v6(muca_ctx* ctx, const SweepParams& prm, int nw, int wpw) {
    SMEM(sweep_kernel_v6<L>, V6<L>::SMEM_BYTES);
    const int per_block = nw * wpw;
    const int grid = (prm.W + per_block - 1) / per_block;
    sweep_kernel_v6<L><<<grid, 64 * nw, V6<L>::SMEM_BYTES, ctx->stream>>>(prm, wpw, ctx->opt_role_map);
    CU(cudaGetLastError());
    return MUCA_OK;
}

template <int L>
int launch_sweep_l1(muca_ctx* ctx, const SweepParams& prm, int tpb) {
    SMEM(sweep_kernel_l1<L>, l1_smem_bytes<L>());
    sweep_kernel_l1<L><<<(prm.W + tpb - 1) / tpb, tpb, l1_smem_bytes<L>(), ctx->stream>>>(prm);
    CU(cudaGetLastError());
    return MUCA_OK;
}

// kernels: MODE_V6 = sweep_kernel_v6 (muca_resident.cuh, L <= 32), MODE_S6 = sweep_kernel_s6 (muca_streamed.cuh, L >= 32),
// MODE_L1 = sweep_kernel_l1 (muca_device.cuh, L >= 32)
enum { MODE_V6 = 0, MODE_L1 = 1, MODE_S6 = 2 };
struct Plan { int mode; int tpb; int nw; int wpw; };   // tpb = walkers per block; v6: nw warp pairs x wpw walkers per warp

// walkers per block of the L1 kernel: with few walkers one warp per block (they spread over the SMs), otherwise two
int l1_default_tpb(const muca_ctx* c) {
    const int n_sm = c->n_sm > 0 ? c->n_sm : 148;
    return c->W > 64 * n_sm ? 64 : 32;
}

Plan make_plan(const muca_ctx* c) {
    Plan p;
    const int L = c->L;
    int kern = c->opt_kernel;
    if (kern == MUCA_KERNEL_AUTO) kern = L <= 32 ? MUCA_KERNEL_RESIDENT : MUCA_KERNEL_STREAMED_PAIRS;
    if (L < 32) kern = MUCA_KERNEL_RESIDENT;                                        // the streamed kernels work on whole 32-site words
    if (L > 32 && kern == MUCA_KERNEL_RESIDENT) kern = MUCA_KERNEL_STREAMED_PAIRS;   // lattices of L >= 64 do not fit beside the table
    p.nw = p.wpw = 0;
    const int n_sm = c->n_sm > 0 ? c->n_sm : 148;
    if (kern == MUCA_KERNEL_RESIDENT) {
        // spread the walkers over all SMs: as few warps per SM as possible, then as few lanes per warp as possible
        // (one block per SM; a half-empty warp costs the same issue slots, but fewer lanes collide in the banks)
        p.mode = MODE_V6;
        const int warps = (c->W + 31) / 32;
        int nw = c->opt_tpb > 0 ? c->opt_tpb / 32 : (warps <= n_sm ? 1 : warps <= 2 * n_sm ? 2 : 4);
        if (nw < 1) nw = 1;
        if (nw > 4) nw = 4;
        int wpw = c->opt_wpw > 0 ? c->opt_wpw : (c->opt_tpb > 0 ? 32 : (c->W + n_sm * nw - 1) / (n_sm * nw));
        if (wpw < 1) wpw = 1;
        if (wpw > 32) wpw = 32;
        p.nw = nw; p.wpw = wpw; p.tpb = nw * wpw;
        return p;
    }
    int tpb = c->opt_tpb;
    if (kern == MUCA_KERNEL_STREAMED_PAIRS) {
        p.mode = MODE_S6;
        if (tpb <= 0) {   // one block per SM (147 KB of table at L = 64): spread the walkers over all SMs
            tpb = ((c->W + n_sm - 1) / n_sm + 31) / 32 * 32;
            if (tpb > 32 * s6_max_pairs(L)) tpb = 32 * s6_max_pairs(L);
        }
    } else {
        p.mode = MODE_L1;
        if (tpb <= 0) tpb = l1_default_tpb(c);
    }
    p.tpb = tpb;
    return p;
}

size_t plan_smem(int L, const Plan& p) {
    if (p.mode == MODE_S6) return 0;   // sized at run time from what the device allows
    if (p.mode == MODE_V6) return L == 8 ? V6<8>::SMEM_BYTES : L == 16 ? V6<16>::SMEM_BYTES : V6<32>::SMEM_BYTES;
    return L == 32 ? l1_smem_bytes<32>() : L == 64 ? l1_smem_bytes<64>() : l1_smem_bytes<128>();
}

struct Window { int j_lo = 0, n_rows = 0, sent_lo = 0, sent_hi = 0; };

template <int L>
int launch_s6_t(muca_ctx* ctx, const SweepParams& prm, int tpb, const Window& win, bool sorted) {
    const int npairs = tpb / 32;
    if (npairs < 1 || npairs > s6_max_pairs(L)) return fail(ctx, MUCA_EINVAL, "paired streamed kernel: 1 to %d warp pairs per block at L = %d", s6_max_pairs(L), L);
    const size_t smem = s6_smem_bytes(win.n_rows, npairs);
    SMEM((sweep_kernel_s6<L>), smem);
    sweep_kernel_s6<L><<<(prm.W + tpb - 1) / tpb, 2 * tpb, smem, ctx->stream>>>(prm, win.j_lo, win.n_rows, win.sent_lo, win.sent_hi,
                                                                               ctx->opt_role_map, ctx->d_flag, sorted ? ctx->d_perm : nullptr,
                                                                               sorted ? ctx->d_blk_jlo : nullptr);
    CU(cudaGetLastError());
    return MUCA_OK;
}

int launch_s6(muca_ctx* ctx, const SweepParams& prm, int tpb, const Window& win, bool sorted = false) {
    switch (ctx->L) {
        case 32: return launch_s6_t<32>(ctx, prm, tpb, win, sorted);
        case 64: return launch_s6_t<64>(ctx, prm, tpb, win, sorted);
        case 128: return launch_s6_t<128>(ctx, prm, tpb, win, sorted);
    }
    return fail(ctx, MUCA_EINVAL, "paired streamed kernel: L must be 32, 64 or 128");
}

int launch_sweep(muca_ctx* ctx, const SweepParams& prm, const Plan& p) {
    if (p.mode == MODE_V6) {
        switch (ctx->L) {
            case 8: return launch_sweep_v6<8>(ctx, prm, p.nw, p.wpw);
            case 16: return launch_sweep_v6<16>(ctx, prm, p.nw, p.wpw);
            case 32: return launch_sweep_v6<32>(ctx, prm, p.nw, p.wpw);
        }
    } else if (p.mode == MODE_L1) {
        switch (ctx->L) {
            case 32: return launch_sweep_l1<32>(ctx, prm, p.tpb);
            case 64: return launch_sweep_l1<64>(ctx, prm, p.tpb);
            case 128: return launch_sweep_l1<128>(ctx, prm, p.tpb);
        }
    }
    return fail(ctx, MUCA_EINVAL, "unsupported L=%d", ctx->L);
}

// Pinned host buffers are kept in a small process-wide pool instead of being freed with their context: a job that
// creates a context per step (bench.py) otherwise pays cudaMallocHost / cudaFreeHost -- page locking under a driver
// lock, 0.1 ms on a quiet host, hundreds of ms on a busy one -- inside its timed region.
struct PinnedPool {
    std::mutex m;
    std::vector<std::pair<size_t, void*>> free_list;
    void* get(size_t bytes) {
        {
            std::lock_guard<std::mutex> g(m);
            for (size_t i = 0; i < free_list.size(); ++i)
                if (free_list[i].first == bytes) {
                    void* p = free_list[i].second;
                    free_list.erase(free_list.begin() + i);
                    return p;
                }
        }
        void* p = nullptr;
        return cudaMallocHost(&p, bytes) == cudaSuccess ? p : nullptr;
    }
    void put(size_t bytes, void* p) {
        if (!p) return;
        std::lock_guard<std::mutex> g(m);
        if (free_list.size() < 16) free_list.emplace_back(bytes, p);
        else cudaFreeHost(p);
    }
};
PinnedPool& pinned_pool() { static PinnedPool* pool = new PinnedPool; return *pool; }   // never destroyed: contexts may outlive static destructors
size_t pinned_table_bytes(int n_bins) { return (size_t)n_bins * 8 * 4; }
size_t pinned_hist_bytes(int n_bins) { return (size_t)n_bins * 8 + 4 * sizeof(int); }

int create_common(muca_ctx** out, int L, int W, uint64_t seed, uint32_t walker_offset, void* d_ws, size_t ws_bytes,
                  void* stream, bool own) {
    if (!out) return MUCA_EINVAL;
    *out = nullptr;
    if (!valid_L(L) || W < 1 || (uint64_t)walker_offset + (uint64_t)W > 0xFFFFFFFFull) {
        if (own && d_ws) cudaFree(d_ws);
        return MUCA_EINVAL;
    }
    muca_ctx* ctx = new (std::nothrow) muca_ctx;
    if (!ctx) return MUCA_ENOMEM;
    ctx->L = L; ctx->N = L * L; ctx->W = W; ctx->n_bins = ctx->N + 1;
    ctx->seed = seed; ctx->walker_offset = walker_offset;
    ctx->stream = (cudaStream_t)stream;
    ctx->own_workspace = own;
    ctx->d_workspace = d_ws;
    const Carve c = carve(L, W);
    auto bail = [&](int code) { muca_destroy(ctx); return code; };
    if (!d_ws || ws_bytes < c.total || ((uintptr_t)d_ws % ALIGN) != 0) return bail(MUCA_ENOMEM);
    char* base = (char*)d_ws;
    ctx->d_spins = (uint32_t*)(base + c.spins);
    ctx->d_E = (int32_t*)(base + c.E);
    ctx->d_table = (uint32_t*)(base + c.table);
    ctx->d_H = (unsigned long long*)(base + c.H);
    ctx->d_flag = (int*)(base + c.flag);
    ctx->d_stage = (void*)(base + c.stage);
    ctx->d_snap = L >= 32 ? (void*)(base + c.snap) : nullptr;
    ctx->d_perm = L >= 32 ? (int*)(base + c.perm) : nullptr;
    ctx->d_blk_jlo = L >= 32 ? (int*)(base + c.blkwin) : nullptr;
    ctx->d_Hsnap = L >= 32 ? (unsigned long long*)(base + c.hsnap) : nullptr;
    ctx->logw.assign(ctx->n_bins, 0.0);   // R2: omega == 0
    ctx->H.assign(ctx->n_bins, 0);
    ctx->h_table = (uint32_t*)pinned_pool().get(pinned_table_bytes(ctx->n_bins));
    ctx->h_H = (unsigned long long*)pinned_pool().get(pinned_hist_bytes(ctx->n_bins));
    if (!ctx->h_table || !ctx->h_H ||
        cudaEventCreate(&ctx->ev0) != cudaSuccess || cudaEventCreate(&ctx->ev1) != cudaSuccess)
        return bail(MUCA_ECUDA);
    ctx->h_flag = reinterpret_cast<int*>(ctx->h_H + ctx->n_bins);
    // the context lives on the device that is current at creation (the workspace and the stream are that device's)
    if (cudaGetDevice(&ctx->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device) != cudaSuccess)
        return bail(MUCA_ECUDA);
    const int tpb = 128;
    init_kernel<<<(W + tpb - 1) / tpb, tpb, 0, ctx->stream>>>(ctx->d_spins, ctx->d_E, L, W, walker_offset,
                                                             (uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32));
    if (cudaGetLastError() != cudaSuccess) return bail(MUCA_ECUDA);
    if (cudaMemsetAsync(ctx->d_H, 0, (size_t)ctx->n_bins * 8, ctx->stream) != cudaSuccess) return bail(MUCA_ECUDA);
    *out = ctx;
    return MUCA_OK;
}

}  // namespace

namespace {
template <int L, int ACC>
int launch_random_site(muca_ctx* ctx, const RandomSiteParams& prm, int tpb) {
    const size_t smem = random_site_smem_bytes<L, ACC>(tpb);
    SMEM((random_site_kernel<L, ACC>), smem);
    random_site_kernel<L, ACC><<<(prm.W + tpb - 1) / tpb, tpb, smem, ctx->stream>>>(prm);
    CU(cudaGetLastError());
    return MUCA_OK;
}
}  // namespace

extern "C" {

#ifdef MUCA_CHECKED
const char* muca_version(void) { return "muca_b200 0.3 (sm_100a) +checked"; }
#else
const char* muca_version(void) { return "muca_b200 0.3 (sm_100a)"; }
#endif

int muca_abi_version(void) { return MUCA_ABI_VERSION; }

int muca_suggest_walkers(int L, int* n_walkers_out, int* pairs_per_sm_out) {
    if (!valid_L(L) || !n_walkers_out || !pairs_per_sm_out) return MUCA_EINVAL;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n_sm < 1)
        return MUCA_ECUDA;
    const int pairs = L <= 32 ? V6<32>::MAX_WARPS : s6_max_pairs(L);   // the most warp pairs make_plan() gives one block (= one SM)
    *pairs_per_sm_out = pairs;
    *n_walkers_out = n_sm * pairs * 32;
    return MUCA_OK;
}

size_t muca_workspace_bytes(int L, int n_walkers) {
    if (!valid_L(L) || n_walkers < 1) return 0;
    return carve(L, n_walkers).total;
}

int muca_create(muca_ctx** out, int L, int n_walkers, uint64_t seed) {
    if (!out) return MUCA_EINVAL;
    *out = nullptr;
    if (!valid_L(L) || n_walkers < 1) return MUCA_EINVAL;
    const size_t bytes = carve(L, n_walkers).total;
    void* ws = nullptr;
    if (cudaMalloc(&ws, bytes) != cudaSuccess) return MUCA_ECUDA;
    return create_common(out, L, n_walkers, seed, 0u, ws, bytes, nullptr, true);
}

int muca_create_in(muca_ctx** out, int L, int n_walkers, uint64_t seed, uint32_t walker_offset, void* d_workspace,
                   size_t workspace_bytes, void* cuda_stream) {
    return create_common(out, L, n_walkers, seed, walker_offset, d_workspace, workspace_bytes, cuda_stream, false);
}

void muca_destroy(muca_ctx* ctx) {
    if (!ctx) return;
    const DeviceGuard guard(ctx);
    if (ctx->stream || ctx->d_workspace) cudaStreamSynchronize(ctx->stream);
    pinned_pool().put(pinned_table_bytes(ctx->n_bins), ctx->h_table);
    pinned_pool().put(pinned_hist_bytes(ctx->n_bins), ctx->h_H);
    pinned_pool().put((size_t)ctx->W * 12, ctx->h_E);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);

    if (ctx->own_workspace && ctx->d_workspace) cudaFree(ctx->d_workspace);
    delete ctx;
}

int muca_set_option(muca_ctx* ctx, int option, int value) {
    if (!ctx) return MUCA_EINVAL;
    if (option == MUCA_OPT_KERNEL) {
        if (value < MUCA_KERNEL_AUTO || value > MUCA_KERNEL_STREAMED_PAIRS) return fail(ctx, MUCA_EINVAL, "bad kernel %d", value);
        ctx->opt_kernel = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_THREADS_PER_BLOCK) {
        if (value < 0 || value > 1024 || (value % 32) != 0) return fail(ctx, MUCA_EINVAL, "threads per block must be a multiple of 32 in [0, 1024]");
        ctx->opt_tpb = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_WALKERS_PER_WARP) {
        if (value < 0 || value > 32) return fail(ctx, MUCA_EINVAL, "walkers per warp must be in [0, 32]");
        ctx->opt_wpw = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_TABLE_WINDOW_ROWS) {
        if (value < 0) return fail(ctx, MUCA_EINVAL, "table window rows must be >= 0");
        ctx->opt_window_rows = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_UPDATE_SCHEME) {
        if (value != MUCA_SCHEME_TYPEWRITER && value != MUCA_SCHEME_RANDOM_SITE) return fail(ctx, MUCA_EINVAL, "bad update scheme %d", value);
        ctx->opt_scheme = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_ACCEPTANCE) {
        if (value != MUCA_ACCEPT_THRESHOLD && value != MUCA_ACCEPT_EXPF32) return fail(ctx, MUCA_EINVAL, "bad acceptance form %d", value);
        ctx->opt_acceptance = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_ROLE_MAP) {
        if (value < 0 || value > 1) return fail(ctx, MUCA_EINVAL, "role map must be 0 or 1");
        ctx->opt_role_map = value;
        return MUCA_OK;
    }
    if (option == MUCA_OPT_MAX_SWEEPS_PER_LAUNCH) {
        if (value < 0) return fail(ctx, MUCA_EINVAL, "max sweeps per launch must be >= 0");
        ctx->opt_max_sweeps = value;
        return MUCA_OK;
    }
    return fail(ctx, MUCA_EINVAL, "unknown option %d", option);
}

int muca_set_log_weights(muca_ctx* ctx, const double* logw, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (!logw || n_bins != ctx->n_bins) return fail(ctx, MUCA_EINVAL, "set_log_weights: n_bins must be %d", ctx->n_bins);
    std::memcpy(ctx->logw.data(), logw, sizeof(double) * n_bins);
    return MUCA_OK;
}

int muca_get_log_weights(muca_ctx* ctx, double* out, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (!out || n_bins != ctx->n_bins) return fail(ctx, MUCA_EINVAL, "get_log_weights: n_bins must be %d", ctx->n_bins);
    std::memcpy(out, ctx->logw.data(), sizeof(double) * n_bins);
    return MUCA_OK;
}

int muca_run_iteration(muca_ctx* ctx, int therm_sweeps, int sweeps, uint64_t* H_out, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (n_bins != ctx->n_bins || therm_sweeps < 0 || sweeps < 0)
        return fail(ctx, MUCA_EINVAL, "run_iteration: n_bins must be %d, sweeps >= 0", ctx->n_bins);
    if (ctx->iteration == 0xFFFFFFFFu) return fail(ctx, MUCA_ERANGE, "iteration counter exhausted");
    const DeviceGuard guard(ctx);
    Plan plan = make_plan(ctx);
    const int max_smem = ctx->max_smem_optin;
    if (plan_smem(ctx->L, plan) > (size_t)max_smem)
        return fail(ctx, MUCA_EINVAL, "kernel variant needs %zu B of shared memory per block, device allows %d",
                    plan_smem(ctx->L, plan), max_smem);
    // a1: thresholds from omega (host, double)
    std::vector<uint32_t> t5;
    build_thresholds5(ctx->logw, t5);
    expand_table8(t5, ctx->n_bins, ctx->h_table);
    CU(cudaMemcpyAsync(ctx->d_table, ctx->h_table, (size_t)ctx->n_bins * 8 * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_H, 0, (size_t)ctx->n_bins * 8, ctx->stream));

    const uint64_t total = (uint64_t)therm_sweeps + (uint64_t)sweeps;
    if (total > 0xFFFFFFFFull) return fail(ctx, MUCA_EINVAL, "too many sweeps");

    // windowed table (muca_streamed.cuh): pick the window around the walkers' slots, keep a snapshot for the fallback
    Plan fallback;
    fallback.mode = MODE_L1; fallback.tpb = l1_default_tpb(ctx); fallback.nw = fallback.wpw = 0;
    Window win;
    bool guarded = false;   // the window has sentinel rows: the result counts only if no walker entered one
    bool sorted = false;    // one window per block over walkers sorted by energy, a few sweeps per launch (run_sorted below)
    const bool windowed_plan = plan.mode == MODE_S6;
    if (windowed_plan) {
        const size_t spin_bytes = (size_t)ctx->W * (ctx->N / 8);
        ctx->h_flag[0] = 0; ctx->h_flag[1] = 0x7FFFFFFF; ctx->h_flag[2] = -1;
        CU(cudaMemcpyAsync(ctx->d_flag, ctx->h_flag, 3 * sizeof(int), cudaMemcpyHostToDevice, ctx->stream));
        slot_range_kernel<<<ctx->n_sm, 256, 0, ctx->stream>>>(ctx->d_E, ctx->W, ctx->N, ctx->d_flag + 1);
        CU(cudaGetLastError());
        CU(cudaMemcpyAsync(ctx->h_flag, ctx->d_flag, 3 * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        const int lo = ctx->h_flag[1], hi = ctx->h_flag[2];
        const size_t ring = s6_ring_bytes(plan.tpb / 32) + S6_RING_OFF;
        int cap = (int)(((size_t)max_smem - ring) / S6_RS) - 2 * S6_PAD_ROWS;
        if (ctx->opt_window_rows > 0 && ctx->opt_window_rows < cap) cap = ctx->opt_window_rows;
        // rows between the outermost walker and a sentinel at the start of the iteration.  An iteration that a walker left
        // through a sentinel ran twice, so the margin asked for is quadrupled after such an iteration (the plain kernel is
        // then taken at once where the walkers' span comes close to the window) and halved again after a clean one.
        const int margin = ctx->win_margin;
        if (cap >= ctx->n_bins) {
            win.j_lo = 0; win.n_rows = ctx->n_bins;                          // the whole table fits: nothing to guard
        } else if (hi - lo + 1 + 2 * (2 + margin) > cap) {
            sorted = true;                                                    // the walkers are spread too widely for ONE window
            win.n_rows = cap;
        } else {
            int j_lo = lo - (cap - (hi - lo + 1)) / 2;
            if (j_lo < 0) j_lo = 0;
            if (j_lo + cap > ctx->n_bins) j_lo = ctx->n_bins - cap;
            win.j_lo = j_lo; win.n_rows = cap;
            win.sent_lo = j_lo > 0 ? 2 : 0;
            win.sent_hi = j_lo + cap < ctx->n_bins ? 2 : 0;
            guarded = true;
            CU(cudaMemcpyAsync(ctx->d_snap, ctx->d_spins, spin_bytes, cudaMemcpyDeviceToDevice, ctx->stream));
            CU(cudaMemcpyAsync((char*)ctx->d_snap + align_up(spin_bytes), ctx->d_E, (size_t)ctx->W * 4, cudaMemcpyDeviceToDevice, ctx->stream));
        }
        if (plan.mode != MODE_L1 && !sorted) ctx->stat_window_iterations += 1;
    }

    // a2-a4: sweeps.  A block's uint32 bins must not overflow: tpb * measured sweeps * N < 2^32 per launch.
    SweepParams prm;
    prm.spins = ctx->d_spins; prm.E = ctx->d_E; prm.table = ctx->d_table; prm.H = ctx->d_H;
    prm.W = ctx->W; prm.walker_offset = ctx->walker_offset;
    prm.key0 = (uint32_t)(ctx->seed & 0xFFFFFFFFull); prm.key1 = (uint32_t)(ctx->seed >> 32);
    prm.iteration = ctx->iteration; prm.therm = (uint32_t)therm_sweeps;
    prm.check = ctx->d_flag + 3; prm.fault = 0u;
#ifdef MUCA_CHECKED
    if (const char* f = getenv("MUCA_CHECKED_FAULT")) prm.fault = (uint32_t)atoi(f);   // tests: make the self-check fire
#endif
    CU(cudaMemsetAsync(ctx->d_flag + 3, 0, sizeof(int), ctx->stream));
    int launches = windowed_plan ? 1 : 0;   // the slot-range kernel
    auto run_sweeps = [&](const Plan& pl) -> int {
        uint64_t max_meas = 0xFFFFFFFFull / ((uint64_t)pl.tpb * (uint64_t)ctx->N);
        if (max_meas < 1) max_meas = 1;
        const uint64_t max_any = ctx->opt_max_sweeps > 0 ? (uint64_t)ctx->opt_max_sweeps : total + 1;
        uint64_t s = 0;
        while (s < total) {
            uint64_t e = total;
            const uint64_t meas_begin = s > (uint64_t)therm_sweeps ? s : (uint64_t)therm_sweeps;
            if (e > meas_begin + max_meas) e = meas_begin + max_meas;
            if (e > s + max_any) e = s + max_any;
            prm.sweep_begin = (uint32_t)s; prm.sweep_end = (uint32_t)e;
            const int rc = pl.mode == MODE_S6 ? launch_s6(ctx, prm, pl.tpb, win) : launch_sweep(ctx, prm, pl);
            if (rc != MUCA_OK) return rc;
            ++launches;
            s = e;
        }
        return MUCA_OK;
    };
    // Walkers spread over more table rows than shared memory holds (L = 128 once the weights have spread them: the regime of
    // every production run): the iteration is cut into launches of a few sweeps.  Before each one the walkers are sorted by
    // energy on the host (8192 energies: a D2H copy and a counting sort, ~30 us against milliseconds of sweeps), every block is
    // handed neighbours in energy and a window of its own around them, and spins, energies and histogram are copied aside;
    // a launch that a walker left through a sentinel is undone and repeated with the plain kernel.  The number of sweeps per
    // launch follows from the rows left between a block's walkers and its sentinels: a sweep moves a walker by about
    // sqrt(3 N / 4) slots (N attempts, every second one accepted, mean squared step 1.5), and 6 sigma must fit.  That rule
    // alone decides whether a launch gets windows: win_margin, the back-off of the single-window path below, plays no part
    // here (it is only ever lowered by clean single-window iterations, which a spread population no longer has -- a margin
    // grown to thousands of rows would otherwise keep every later iteration on the plain kernel for good).
    auto run_sorted = [&]() -> int {
        const int W = ctx->W, tpb = plan.tpb, n_blocks = (W + tpb - 1) / tpb, cap = win.n_rows;
        const size_t spin_bytes = (size_t)W * (ctx->N / 8);
        if (!ctx->h_E) ctx->h_E = (int32_t*)pinned_pool().get((size_t)W * 12);
        if (!ctx->h_E) return fail(ctx, MUCA_ECUDA, "pinned allocation failed");
        int32_t* const h_perm = ctx->h_E + W;
        int32_t* const h_jlo = ctx->h_E + 2 * W;
        std::vector<int> order(W), count(ctx->n_bins + 1);
        const uint64_t max_meas = std::max<uint64_t>(1, 0xFFFFFFFFull / ((uint64_t)tpb * (uint64_t)ctx->N));
        const double sigma1 = std::sqrt(0.75 * (double)ctx->N);
        bool any_window = false;
        uint64_t s = 0;
        while (s < total) {
            CU(cudaMemcpyAsync(ctx->h_E, ctx->d_E, (size_t)W * 4, cudaMemcpyDeviceToHost, ctx->stream));
            CU(cudaStreamSynchronize(ctx->stream));
            // walkers by energy slot, ties by index: a counting sort (slots are 0 .. N; ~30 us for 8192 walkers)
            std::fill(count.begin(), count.end(), 0);
            for (int i = 0; i < W; ++i) count[((ctx->h_E[i] + 2 * ctx->N) >> 2) + 1] += 1;
            for (int j = 0; j < ctx->n_bins; ++j) count[j + 1] += count[j];
            for (int i = 0; i < W; ++i) order[count[(ctx->h_E[i] + 2 * ctx->N) >> 2]++] = i;
            int room = cap;   // rows between a block's walkers and its sentinels, smallest over the blocks
            for (int b = 0; b < n_blocks; ++b) {
                const int i0 = b * tpb, i1 = std::min(W, i0 + tpb) - 1;
                const int lo_b = (ctx->h_E[order[i0]] + 2 * ctx->N) >> 2, hi_b = (ctx->h_E[order[i1]] + 2 * ctx->N) >> 2;
                int j_lo = lo_b - (cap - (hi_b - lo_b + 1)) / 2;
                if (j_lo < 0) j_lo = 0;
                if (j_lo + cap > ctx->n_bins) j_lo = ctx->n_bins - cap;
                h_jlo[b] = j_lo;
                const int below = j_lo > 0 ? lo_b - j_lo - 2 : cap, above = j_lo + cap < ctx->n_bins ? j_lo + cap - 1 - hi_b - 2 : cap;
                room = std::min(room, std::min(below, above));
            }
            for (int i = 0; i < W; ++i) h_perm[i] = order[i];
            uint64_t e = total;
            const uint64_t meas_begin = s > (uint64_t)therm_sweeps ? s : (uint64_t)therm_sweeps;
            if (e > meas_begin + max_meas) e = meas_begin + max_meas;
            if (ctx->opt_max_sweeps > 0 && e > s + (uint64_t)ctx->opt_max_sweeps) e = s + (uint64_t)ctx->opt_max_sweeps;
            const double k = room > 0 ? (double)room / (6.0 * sigma1) : 0.0;
            uint64_t chunk = (uint64_t)(k * k);
            if (chunk > 64) chunk = 64;
            prm.sweep_begin = (uint32_t)s;
            if (chunk >= 1) {
                if (e > s + chunk) e = s + chunk;
                prm.sweep_end = (uint32_t)e;
                CU(cudaMemcpyAsync(ctx->d_perm, h_perm, (size_t)W * 4, cudaMemcpyHostToDevice, ctx->stream));
                CU(cudaMemcpyAsync(ctx->d_blk_jlo, h_jlo, (size_t)n_blocks * 4, cudaMemcpyHostToDevice, ctx->stream));
                CU(cudaMemcpyAsync(ctx->d_snap, ctx->d_spins, spin_bytes, cudaMemcpyDeviceToDevice, ctx->stream));
                CU(cudaMemcpyAsync((char*)ctx->d_snap + align_up(spin_bytes), ctx->d_E, (size_t)W * 4, cudaMemcpyDeviceToDevice, ctx->stream));
                CU(cudaMemcpyAsync(ctx->d_Hsnap, ctx->d_H, (size_t)ctx->n_bins * 8, cudaMemcpyDeviceToDevice, ctx->stream));
                CU(cudaMemsetAsync(ctx->d_flag, 0, sizeof(int), ctx->stream));
                const int rc = launch_s6(ctx, prm, tpb, win, true);
                if (rc != MUCA_OK) return rc;
                ++launches; ctx->stat_sorted_launches += 1; any_window = true;
                CU(cudaMemcpyAsync(ctx->h_flag, ctx->d_flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
                CU(cudaStreamSynchronize(ctx->stream));
                if (!ctx->h_flag[0]) { s = e; continue; }
                // a walker left its block's window: undo the launch
                CU(cudaMemcpyAsync(ctx->d_spins, ctx->d_snap, spin_bytes, cudaMemcpyDeviceToDevice, ctx->stream));
                CU(cudaMemcpyAsync(ctx->d_E, (char*)ctx->d_snap + align_up(spin_bytes), (size_t)W * 4, cudaMemcpyDeviceToDevice, ctx->stream));
                CU(cudaMemcpyAsync(ctx->d_H, ctx->d_Hsnap, (size_t)ctx->n_bins * 8, cudaMemcpyDeviceToDevice, ctx->stream));
                ctx->stat_window_fallbacks += 1;
            } else {
                if (e > s + 4) e = s + 4;   // no room for a window now: a few sweeps with the plain kernel, then look again
            }
            prm.sweep_end = (uint32_t)e;
            const int rc = launch_sweep(ctx, prm, fallback);
            if (rc != MUCA_OK) return rc;
            ++launches;
            s = e;
        }
        if (any_window) ctx->stat_window_iterations += 1;
        return MUCA_OK;
    };
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    {
        const int rc = sorted ? run_sorted() : run_sweeps(plan);
        if (rc != MUCA_OK) return rc;
    }
    if (plan.mode == MODE_S6 && guarded) {
        CU(cudaMemcpyAsync(ctx->h_flag, ctx->d_flag, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        if (ctx->h_flag[0]) {   // a walker left the window: repeat the iteration from the snapshot with the L1 kernel
            const size_t spin_bytes = (size_t)ctx->W * (ctx->N / 8);
            CU(cudaMemcpyAsync(ctx->d_spins, ctx->d_snap, spin_bytes, cudaMemcpyDeviceToDevice, ctx->stream));
            CU(cudaMemcpyAsync(ctx->d_E, (char*)ctx->d_snap + align_up(spin_bytes), (size_t)ctx->W * 4, cudaMemcpyDeviceToDevice, ctx->stream));
            CU(cudaMemsetAsync(ctx->d_H, 0, (size_t)ctx->n_bins * 8, ctx->stream));
            ctx->stat_window_fallbacks += 1;
            ctx->win_margin = ctx->win_margin * 4 > 4096 ? 4096 : ctx->win_margin * 4;
            const int rc = run_sweeps(fallback);
            if (rc != MUCA_OK) return rc;
        } else if (ctx->win_margin > 8) {
            ctx->win_margin /= 2;
        }
    }
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_H, ctx->d_H, (size_t)ctx->n_bins * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_flag + 3, ctx->d_flag + 3, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (ctx->h_flag[3] & CHK_SMEM_BASE)   // muca_device.cuh smem_base_ok(): the paired kernels refused to run
        return fail(ctx, MUCA_ECUDA, "sweep kernel refused to run: on this device / driver the dynamic shared memory does not start at "
                    "the offset the kernel's table addressing was built for; the iteration was not completed (MUCA_OPT_KERNEL = "
                    "MUCA_KERNEL_STREAMED does not depend on it, L >= 32)");
#ifdef MUCA_CHECKED
    if (ctx->h_flag[3])
        return fail(ctx, MUCA_ECUDA, "checked build: self-check failed, mask 0x%x (1 = state is not a table row, 2 = deviates read before "
                    "written, 4 = deviates overwritten while read)", ctx->h_flag[3]);
#endif
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    ctx->last_sweep_ms = ms;
    ctx->last_launches = launches;
    for (int j = 0; j < ctx->n_bins; ++j) ctx->H[j] = (uint64_t)ctx->h_H[j];
    if (H_out) std::memcpy(H_out, ctx->H.data(), sizeof(uint64_t) * ctx->n_bins);
    ctx->iteration += 1;
    return MUCA_OK;
}

// The paper's own update scheme (R22): same random site in all walkers.
int muca_run_iteration_random_site(muca_ctx* ctx, uint64_t therm_updates, uint64_t updates, uint64_t* H_out, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (n_bins != ctx->n_bins) return fail(ctx, MUCA_EINVAL, "run_iteration_random_site: n_bins must be %d", ctx->n_bins);
    if (ctx->iteration == 0xFFFFFFFFu) return fail(ctx, MUCA_ERANGE, "iteration counter exhausted");
    if (therm_updates > (1ull << 60) || updates > (1ull << 60)) return fail(ctx, MUCA_EINVAL, "too many updates");
    const DeviceGuard guard(ctx);
    const bool expf32 = ctx->opt_acceptance == MUCA_ACCEPT_EXPF32;
    if (expf32) {   // R23: the weights in single precision; the kernel evaluates U < exp32(omega_f[j'] - omega_f[j])
        float* wf = reinterpret_cast<float*>(ctx->h_table);
        for (int j = 0; j < ctx->n_bins; ++j) wf[j] = (float)ctx->logw[j];
    } else {
        std::vector<uint32_t> t5;
        build_thresholds5(ctx->logw, t5);                                       // a1, as in muca_run_iteration
        expand_table8(t5, ctx->n_bins, ctx->h_table);
    }
    CU(cudaMemcpyAsync(ctx->d_table, ctx->h_table, (size_t)ctx->n_bins * 8 * 4, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaMemsetAsync(ctx->d_H, 0, (size_t)ctx->n_bins * 8, ctx->stream));
    // one block per SM where the walkers allow it; the lattice words of a block's walkers must fit beside table and bins
    auto rs_smem = [&](int t) -> size_t {
        switch (ctx->L) {
            case 8: return expf32 ? random_site_smem_bytes<8, 1>(t) : random_site_smem_bytes<8, 0>(t);
            case 16: return expf32 ? random_site_smem_bytes<16, 1>(t) : random_site_smem_bytes<16, 0>(t);
            case 32: return expf32 ? random_site_smem_bytes<32, 1>(t) : random_site_smem_bytes<32, 0>(t);
            case 64: return expf32 ? random_site_smem_bytes<64, 1>(t) : random_site_smem_bytes<64, 0>(t);
            default: return expf32 ? random_site_smem_bytes<128, 1>(t) : random_site_smem_bytes<128, 0>(t);
        }
    };
    int tpb = ((ctx->W + ctx->n_sm - 1) / ctx->n_sm + 31) / 32 * 32;
    if (tpb > 512) tpb = 512;
    while (tpb > 32 && rs_smem(tpb) > (size_t)ctx->max_smem_optin) tpb -= 32;
    RandomSiteParams prm;
    prm.spins = ctx->d_spins; prm.E = ctx->d_E; prm.table = ctx->d_table; prm.H = ctx->d_H;
    prm.W = ctx->W; prm.walker_offset = ctx->walker_offset;
    prm.key0 = (uint32_t)(ctx->seed & 0xFFFFFFFFull); prm.key1 = (uint32_t)(ctx->seed >> 32);
    prm.iteration = ctx->iteration; prm.therm = therm_updates;
    const uint64_t total = therm_updates + updates;
    const uint64_t max_meas = 0xFFFFFFFFull / (uint64_t)tpb;                      // a block's uint32 bins must not overflow
    int launches = 0;
    CU(cudaEventRecord(ctx->ev0, ctx->stream));
    uint64_t u = 0;
    while (u < total) {
        const uint64_t meas_begin = u > therm_updates ? u : therm_updates;
        uint64_t e = total;
        if (e > meas_begin + max_meas) e = meas_begin + max_meas;
        prm.u_begin = u; prm.u_end = e;
        int rc = MUCA_EINVAL;
        switch (ctx->L) {
            case 8: rc = expf32 ? launch_random_site<8, 1>(ctx, prm, tpb) : launch_random_site<8, 0>(ctx, prm, tpb); break;
            case 16: rc = expf32 ? launch_random_site<16, 1>(ctx, prm, tpb) : launch_random_site<16, 0>(ctx, prm, tpb); break;
            case 32: rc = expf32 ? launch_random_site<32, 1>(ctx, prm, tpb) : launch_random_site<32, 0>(ctx, prm, tpb); break;
            case 64: rc = expf32 ? launch_random_site<64, 1>(ctx, prm, tpb) : launch_random_site<64, 0>(ctx, prm, tpb); break;
            case 128: rc = expf32 ? launch_random_site<128, 1>(ctx, prm, tpb) : launch_random_site<128, 0>(ctx, prm, tpb); break;
        }
        if (rc != MUCA_OK) return rc;
        ++launches;
        u = e;
    }
    CU(cudaEventRecord(ctx->ev1, ctx->stream));
    CU(cudaMemcpyAsync(ctx->h_H, ctx->d_H, (size_t)ctx->n_bins * 8, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    ctx->last_sweep_ms = ms;
    ctx->last_launches = launches;
    for (int j = 0; j < ctx->n_bins; ++j) ctx->H[j] = (uint64_t)ctx->h_H[j];
    if (H_out) std::memcpy(H_out, ctx->H.data(), sizeof(uint64_t) * ctx->n_bins);
    ctx->iteration += 1;
    return MUCA_OK;
}

int muca_get_histogram(muca_ctx* ctx, uint64_t* H_out, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (!H_out || n_bins != ctx->n_bins) return fail(ctx, MUCA_EINVAL, "get_histogram: n_bins must be %d", ctx->n_bins);
    std::memcpy(H_out, ctx->H.data(), sizeof(uint64_t) * n_bins);
    return MUCA_OK;
}

int muca_update_weights_with(muca_ctx* ctx, const uint64_t* H_total, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (!H_total || n_bins != ctx->n_bins) return fail(ctx, MUCA_EINVAL, "update_weights: n_bins must be %d", ctx->n_bins);
    // Eq. (4): omega <- omega - ln H on visited slots (R8: raw counts)
    for (int j = 0; j < n_bins; ++j)
        if (H_total[j] != 0) ctx->logw[j] -= std::log((double)H_total[j]);
    return MUCA_OK;
}

int muca_update_weights(muca_ctx* ctx) {
    if (!ctx) return MUCA_EINVAL;
    return muca_update_weights_with(ctx, ctx->H.data(), ctx->n_bins);
}

// ---- convergence driver (host logic; Eq. (6), (7), (A.1); R18) ----
int muca_flatness(const uint64_t* H, int n_bins, int w, muca_flatness_t* out) {
    if (!H || !out || n_bins < 3 || w < 0) return MUCA_EINVAL;
    const int N = n_bins - 1;
    uint64_t total = 0;
    int lo = -1, hi = -1;
    for (int j = 0; j < n_bins; ++j)
        if (H[j]) { total += H[j]; if (lo < 0) lo = j; hi = j; }
    out->j_lo = lo; out->j_hi = hi; out->width = lo < 0 ? 0 : hi - lo + 1; out->n_updates = total;
    out->d_k = 0.0; out->d_c = 0.0;
    if (total == 0) return MUCA_OK;
    if (w == 0) {   // R19: w = max(w', 10), w' = ACCESSIBLE slots of the range covered by THIS histogram
        w = out->width - ((lo <= 1 && hi >= 1) ? 1 : 0) - ((lo <= N - 1 && hi >= N - 1) ? 1 : 0);
        if (w < 10) w = 10;
    }
    double dk = 0.0;                                         // Eq. (6): empty bins do not contribute
    for (int j = 0; j < n_bins; ++j)
        if (H[j]) { const double P = (double)H[j] / (double)total; dk += P * std::log(P * (double)w); }
    out->d_k = dk;
    const double m = (double)total / (double)(N - 1);       // Eq. (A.1): N - 1 accessible slots
    double dc = 0.0;
    for (int j = 0; j < n_bins; ++j) {
        if (j == 1 || j == N - 1) continue;
        const double d = std::fabs((double)H[j] / m - 1.0);
        if (d > dc) dc = d;
    }
    out->d_c = dc;
    return MUCA_OK;
}

int muca_schedule(int L, int n_walkers, int w_prev, double* n_updates_io, int* full_range_io, int* w_out, int* therm_sweeps,
                  int* sweeps) {
    if (!valid_L(L) || n_walkers < 1 || w_prev < 0 || !n_updates_io || !full_range_io || !w_out || !therm_sweeps || !sweeps)
        return MUCA_EINVAL;
    const int N = L * L;
    const int w = w_prev > 10 ? w_prev : 10;                // w = max(w', 10)
    double n_up;
    const bool full = w >= N + 1;
    if (full && *full_range_io) n_up = std::floor(1.1 * *n_updates_io) + 1.0;                   // whole range covered before: x 1.1
    else n_up = std::floor(6.0 * std::pow((double)w, 2.25) / (double)n_walkers) + 1.0;          // Eq. (7), z = 2.25
    const double n_th = 30.0 * (double)w;                    // f_therm = 30
    const double max_sweeps = 1.0e9;
    double sw = std::ceil(n_up / (double)N), th = std::ceil(n_th / (double)N);
    if (sw < 1.0) sw = 1.0;
    if (th < 1.0) th = 1.0;
    if (sw > max_sweeps || th > max_sweeps) return MUCA_ERANGE;
    *n_updates_io = n_up; *full_range_io = full ? 1 : 0; *w_out = w; *therm_sweeps = (int)th; *sweeps = (int)sw;
    return MUCA_OK;
}

int muca_converge(muca_ctx* ctx, int max_iterations, double d_flat, muca_iteration_log_t* log, int log_capacity,
                  int* iterations_out, int* converged_out) {
    if (!ctx) return MUCA_EINVAL;
    if (max_iterations < 0 || (log && log_capacity < 0)) return fail(ctx, MUCA_EINVAL, "converge: bad arguments");
    int it = 0, conv = 0;
    while (it < max_iterations && !conv) {
        int w = 0, th = 0, sw = 0;
        int rc = muca_schedule(ctx->L, ctx->W, ctx->conv_w_prev, &ctx->conv_n_updates, &ctx->conv_full, &w, &th, &sw);
        if (rc != MUCA_OK) return fail(ctx, rc, "converge: schedule out of range");
        if (ctx->opt_scheme == MUCA_SCHEME_RANDOM_SITE)   // the paper's own units: attempted flips per walker
            rc = muca_run_iteration_random_site(ctx, (uint64_t)(30.0 * (double)w), (uint64_t)ctx->conv_n_updates, nullptr, ctx->n_bins);
        else
            rc = muca_run_iteration(ctx, th, sw, nullptr, ctx->n_bins);
        if (rc != MUCA_OK) return rc;
        muca_flatness_t fl;
        rc = muca_flatness(ctx->H.data(), ctx->n_bins, 0, &fl);
        if (rc != MUCA_OK) return fail(ctx, rc, "converge: flatness failed");
        rc = muca_update_weights(ctx);
        if (rc != MUCA_OK) return rc;
        if (log && it < log_capacity) {
            log[it].w = w; log[it].therm_sweeps = th; log[it].sweeps = sw; log[it].flat = fl; log[it].sweep_ms = ctx->last_sweep_ms;
        }
        ctx->conv_w_prev = fl.width;
        conv = fl.d_k < d_flat ? 1 : 0;
        ++it;
    }
    if (iterations_out) *iterations_out = it;
    if (converged_out) *converged_out = conv;
    return MUCA_OK;
}

// ---- production run + jackknife (host logic; R21) ----
namespace {
// ln Omega from one histogram (double counts): ln H - omega on visited slots, normalised to sum exp = 2^N; NaN elsewhere
void ln_omega_estimate(const std::vector<double>& H, const std::vector<double>& logw, int N, std::vector<double>& out) {
    const double nan = std::numeric_limits<double>::quiet_NaN();
    const int bins = (int)H.size();
    out.assign(bins, nan);
    double mx = -std::numeric_limits<double>::infinity();
    for (int j = 0; j < bins; ++j)
        if (H[j] > 0.0) { out[j] = std::log(H[j]) - logw[j]; if (out[j] > mx) mx = out[j]; }
    double sum = 0.0;
    for (int j = 0; j < bins; ++j)
        if (H[j] > 0.0) sum += std::exp(out[j] - mx);
    const double shift = (double)N * std::log(2.0) - (mx + std::log(sum));
    for (int j = 0; j < bins; ++j)
        if (H[j] > 0.0) out[j] += shift;
}
}  // namespace

int muca_production(muca_ctx* ctx, int n_calls, int therm_sweeps, int sweeps, double* ln_omega_out, double* err_out,
                    uint64_t* H_calls_out, int n_bins) {
    if (!ctx) return MUCA_EINVAL;
    if (n_calls < 2 || n_bins != ctx->n_bins || !ln_omega_out || !err_out)
        return fail(ctx, MUCA_EINVAL, "production: n_calls >= 2, n_bins must be %d, outputs must not be NULL", ctx->n_bins);
    const int bins = ctx->n_bins;
    std::vector<uint64_t> calls((size_t)n_calls * bins);
    for (int k = 0; k < n_calls; ++k) {
        const int rc = ctx->opt_scheme == MUCA_SCHEME_RANDOM_SITE
                           ? muca_run_iteration_random_site(ctx, (uint64_t)therm_sweeps * (uint64_t)ctx->N,
                                                            (uint64_t)sweeps * (uint64_t)ctx->N, calls.data() + (size_t)k * bins, bins)
                           : muca_run_iteration(ctx, therm_sweeps, sweeps, calls.data() + (size_t)k * bins, bins);
        if (rc != MUCA_OK) return rc;
    }
    if (H_calls_out) std::memcpy(H_calls_out, calls.data(), sizeof(uint64_t) * calls.size());
    std::vector<double> total(bins, 0.0), loo(bins), est, mean(bins, 0.0), var(bins, 0.0);
    for (int k = 0; k < n_calls; ++k)
        for (int j = 0; j < bins; ++j) total[j] += (double)calls[(size_t)k * bins + j];
    ln_omega_estimate(total, ctx->logw, ctx->N, est);
    for (int j = 0; j < bins; ++j) ln_omega_out[j] = est[j];
    std::vector<double> all((size_t)n_calls * bins);
    for (int k = 0; k < n_calls; ++k) {
        for (int j = 0; j < bins; ++j) loo[j] = total[j] - (double)calls[(size_t)k * bins + j];
        ln_omega_estimate(loo, ctx->logw, ctx->N, est);
        for (int j = 0; j < bins; ++j) { all[(size_t)k * bins + j] = est[j]; mean[j] += est[j]; }
    }
    for (int j = 0; j < bins; ++j) mean[j] /= (double)n_calls;
    for (int k = 0; k < n_calls; ++k)
        for (int j = 0; j < bins; ++j) { const double d = all[(size_t)k * bins + j] - mean[j]; var[j] += d * d; }
    for (int j = 0; j < bins; ++j) err_out[j] = std::sqrt((double)(n_calls - 1) / (double)n_calls * var[j]);   // NaN propagates
    return MUCA_OK;
}

int muca_get_energies(muca_ctx* ctx, int32_t* E_out, int n_walkers) {
    if (!ctx) return MUCA_EINVAL;
    if (!E_out || n_walkers != ctx->W) return fail(ctx, MUCA_EINVAL, "get_energies: n_walkers must be %d", ctx->W);
    const DeviceGuard guard(ctx);
    CU(cudaMemcpyAsync(E_out, ctx->d_E, sizeof(int32_t) * (size_t)ctx->W, cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    return MUCA_OK;
}

int muca_unpack_spins_device(muca_ctx* ctx, void* d_out, size_t n) {
    if (!ctx) return MUCA_EINVAL;
    if (!d_out || n != (size_t)ctx->W * ctx->N) return fail(ctx, MUCA_EINVAL, "unpack: n must be %zu", (size_t)ctx->W * ctx->N);
    const DeviceGuard guard(ctx);
    if (((uintptr_t)d_out % 16) != 0) return fail(ctx, MUCA_EINVAL, "unpack: device buffer must be 16-byte aligned");
    const size_t threads = (size_t)ctx->W * (ctx->N / 32);
    const int tpb = 256;
    unpack_kernel<<<(unsigned)((threads + tpb - 1) / tpb), tpb, 0, ctx->stream>>>(ctx->d_spins, (int8_t*)d_out, ctx->L, ctx->W);
    CU(cudaGetLastError());
    return MUCA_OK;
}

int muca_get_spins(muca_ctx* ctx, int8_t* out, size_t n) {
    if (!ctx) return MUCA_EINVAL;
    if (!out || n != (size_t)ctx->W * ctx->N) return fail(ctx, MUCA_EINVAL, "get_spins: n must be %zu", (size_t)ctx->W * ctx->N);
    const DeviceGuard guard(ctx);
    int rc = muca_unpack_spins_device(ctx, ctx->d_stage, n);
    if (rc == MUCA_OK) {
        cudaError_t e = cudaMemcpyAsync(out, ctx->d_stage, n, cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) rc = fail(ctx, MUCA_ECUDA, "get_spins copy failed: %s", cudaGetErrorString(e));
    }
    return rc;
}

int muca_set_spins(muca_ctx* ctx, const int8_t* spins, size_t n) {
    if (!ctx) return MUCA_EINVAL;
    if (!spins || n != (size_t)ctx->W * ctx->N) return fail(ctx, MUCA_EINVAL, "set_spins: n must be %zu", (size_t)ctx->W * ctx->N);
    const DeviceGuard guard(ctx);
    void* d_tmp = ctx->d_stage;
    int rc = MUCA_OK;
    cudaError_t e = cudaMemcpyAsync(d_tmp, spins, n, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) {
        const size_t threads = (size_t)ctx->W * (ctx->N / 32);
        const int tpb = 256;
        pack_kernel<<<(unsigned)((threads + tpb - 1) / tpb), tpb, 0, ctx->stream>>>((const int8_t*)d_tmp, ctx->d_spins, ctx->L, ctx->W);
        energy_kernel<<<(ctx->W + 127) / 128, 128, 0, ctx->stream>>>(ctx->d_spins, ctx->d_E, ctx->L, ctx->W);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    }
    if (e != cudaSuccess) rc = fail(ctx, MUCA_ECUDA, "set_spins failed: %s", cudaGetErrorString(e));
    return rc;
}

int muca_get_thresholds(muca_ctx* ctx, uint32_t* out, size_t n) {
    if (!ctx) return MUCA_EINVAL;
    if (!out || n != (size_t)ctx->n_bins * 5) return fail(ctx, MUCA_EINVAL, "get_thresholds: n must be %zu", (size_t)ctx->n_bins * 5);
    std::vector<uint32_t> t5;
    build_thresholds5(ctx->logw, t5);
    std::memcpy(out, t5.data(), sizeof(uint32_t) * n);
    return MUCA_OK;
}

int muca_get_iteration(muca_ctx* ctx, uint32_t* n_out) {
    if (!ctx || !n_out) return MUCA_EINVAL;
    *n_out = ctx->iteration;
    return MUCA_OK;
}

int muca_set_iteration(muca_ctx* ctx, uint32_t n) {
    if (!ctx) return MUCA_EINVAL;
    ctx->iteration = n;
    return MUCA_OK;
}

int muca_last_sweep_ms(muca_ctx* ctx, double* ms_out, int* launches_out) {
    if (!ctx) return MUCA_EINVAL;
    if (ms_out) *ms_out = ctx->last_sweep_ms;
    if (launches_out) *launches_out = ctx->last_launches;
    return MUCA_OK;
}

int muca_window_stats(muca_ctx* ctx, int* windowed_iterations_out, int* fallbacks_out) {
    if (!ctx) return MUCA_EINVAL;
    if (windowed_iterations_out) *windowed_iterations_out = ctx->stat_window_iterations;
    if (fallbacks_out) *fallbacks_out = ctx->stat_window_fallbacks;
    return MUCA_OK;
}

const char* muca_last_error(const muca_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int muca_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n) {
    if (!ctr || !key || !out || n < 1) return MUCA_EINVAL;
    uint32_t *d_c = nullptr, *d_k = nullptr, *d_o = nullptr;
    int rc = MUCA_OK;
    if (cudaMalloc((void**)&d_c, 16 * (size_t)n) != cudaSuccess || cudaMalloc((void**)&d_k, 8 * (size_t)n) != cudaSuccess ||
        cudaMalloc((void**)&d_o, 16 * (size_t)n) != cudaSuccess)
        rc = MUCA_ECUDA;
    if (rc == MUCA_OK && (cudaMemcpy(d_c, ctr, 16 * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess ||
                          cudaMemcpy(d_k, key, 8 * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess))
        rc = MUCA_ECUDA;
    if (rc == MUCA_OK) {
        philox_debug_kernel<<<(n + 127) / 128, 128>>>(d_c, d_k, d_o, n);
        if (cudaGetLastError() != cudaSuccess || cudaMemcpy(out, d_o, 16 * (size_t)n, cudaMemcpyDeviceToHost) != cudaSuccess)
            rc = MUCA_ECUDA;
    }
    cudaFree(d_c); cudaFree(d_k); cudaFree(d_o);
    return rc;
}

}  // extern "C"

// ---- muca_debug_philox_static: the Philox test hook for callers that must not allocate (include/muca.h) -----------------
// The staging rows live in a fixed device array that belongs to the library image: MUCA_PHILOX_STATIC_MAX rows of
// ctr (16 B), key (8 B) and out (16 B), i.e. 160 KiB on every GPU that loads this module, until the process exits.
// On the host side the NAME of the array is only a handle for the runtime, not an address a kernel could use: the device
// address is asked for once per device with cudaGetSymbolAddress (that device current) and it is this pointer that the
// kernel and the copies get.
static __device__ __align__(256) unsigned char philox_static_scratch[(size_t)MUCA_PHILOX_STATIC_MAX * 40];

namespace {
constexpr size_t PHILOX_STATIC_KEY_OFF = (size_t)MUCA_PHILOX_STATIC_MAX * 16;   // ctr rows first, then key rows,
constexpr size_t PHILOX_STATIC_OUT_OFF = (size_t)MUCA_PHILOX_STATIC_MAX * 24;   // then out rows (both offsets 256-aligned)
constexpr int PHILOX_STATIC_DEVICES = 64;                                       // device ordinals with a remembered address
std::mutex philox_static_mutex;                                                 // one call at a time: they share the array
unsigned char* philox_static_addr[PHILOX_STATIC_DEVICES] = {};                  // device address of the array, per device
}  // namespace

extern "C" int muca_debug_philox_static(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n) {
    if (!ctr || !key || !out || n < 1) return MUCA_EINVAL;
    if (n > MUCA_PHILOX_STATIC_MAX) return MUCA_ENOMEM;   // more rows than the fixed array holds: refused before any CUDA call
    std::lock_guard<std::mutex> lock(philox_static_mutex);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0) return MUCA_ECUDA;
    unsigned char* base = dev < PHILOX_STATIC_DEVICES ? philox_static_addr[dev] : nullptr;
    if (!base) {   // set-up, once per device, with that device current
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, philox_static_scratch) != cudaSuccess || !p) return MUCA_ECUDA;
        base = static_cast<unsigned char*>(p);
        if (dev < PHILOX_STATIC_DEVICES) philox_static_addr[dev] = base;
    }
    uint32_t* const d_c = reinterpret_cast<uint32_t*>(base);
    uint32_t* const d_k = reinterpret_cast<uint32_t*>(base + PHILOX_STATIC_KEY_OFF);
    uint32_t* const d_o = reinterpret_cast<uint32_t*>(base + PHILOX_STATIC_OUT_OFF);
    // Whatever the previous call left in the array is overwritten (rows 0 .. n-1 of ctr and key) or never read (the
    // rest): nothing has to be cleared.  The copies are blocking, so the call has left the GPU when the lock is dropped.
    if (cudaMemcpy(d_c, ctr, 16 * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(d_k, key, 8 * (size_t)n, cudaMemcpyHostToDevice) != cudaSuccess)
        return MUCA_ECUDA;
    philox_debug_kernel<<<(n + 127) / 128, 128>>>(d_c, d_k, d_o, n);
    if (cudaGetLastError() != cudaSuccess || cudaMemcpy(out, d_o, 16 * (size_t)n, cudaMemcpyDeviceToHost) != cudaSuccess)
        return MUCA_ECUDA;
    return MUCA_OK;
}
