/* include/muca.h -- C ABI of libmuca_b200: the data-parallel hot path of parallel
 * multicanonical (MUCA) simulation of the 2D Ising model (arXiv 1707.00919),
 * hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * What the library computes (citations: /root/reference/PAPER.md line numbers,
 * "R<n>" = reading listed in DESIGN.md section 3):
 *   - W independent walkers, each on its own L x L periodic Ising lattice
 *     ("p independent walkers", Eq. (5)),
 *   - single-spin-flip Metropolis updates accepted with
 *     min(1, exp[omega(E') - omega(E)]), omega = ln W,
 *     sites visited in typewriter order (R3), uniform deviates from the
 *     counter-based Philox4x32-10 generator keyed by (seed; site, sweep,
 *     iteration, walker) (R4),
 *   - one shared histogram H(E) of the energies met after every attempted flip
 *     of the measured sweeps (thermalisation sweeps are not
 *     recorded),
 *   - the weight recursion W(n+1)(E) = W(n)(E) / H(n)(E)  (Eq. (4), R8).
 *
 * Conventions
 *   N = L*L spins, n_bins = N + 1 energy slots, slot j = (E + 2N)/4, E = -2N + 4j
 *   (energies spaced by 4 on [-2N, 2N]; slots 1 and N-1 are unreachable).
 *   Spins are +1 / -1; packed on the device with bit 1 <-> spin -1.
 *
 * General rules
 *   - every call returns MUCA_OK (0) or a negative muca_status; no exceptions cross
 *     the boundary; muca_last_error() returns a NUL-terminated description of the
 *     last failure on that context (owned by the context, valid until the next call);
 *   - "host" pointers are ordinary host memory owned by the caller, sized exactly as
 *     stated; "device" pointers are CUDA device memory of the current device;
 *   - the context owns all device state except a workspace handed to muca_create_in();
 *   - calls on one context must not run concurrently; different contexts are independent;
 *   - there is no CPU fallback: without a CUDA device every compute entry point
 *     fails with MUCA_ECUDA.
 */
#ifndef MUCA_H_
#define MUCA_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Version of THIS interface: the numeric values of the enums below and the signatures of the entry points.  It is
 * raised whenever a value is renumbered or retired or a signature changes (history: 1 = round-1 kernels, values 3..6 of
 * MUCA_OPT_KERNEL in use; 2 = STREAMED_PAIRS renumbered from 6 to 3, values 4..6 retired; 3 = muca_abi_version,
 * muca_debug_philox_static).  A caller that passes raw integers compares muca_abi_version() of the library it loaded
 * with the MUCA_ABI_VERSION it was written against and refuses to run on a mismatch (the Python binding does). */
#define MUCA_ABI_VERSION 3
int muca_abi_version(void);

typedef struct muca_ctx muca_ctx;

typedef enum muca_status {
    MUCA_OK = 0,
    MUCA_EINVAL = -1, /* bad argument (L, n_walkers, n_bins, negative sweeps, NULL, wrong size) */
    MUCA_ECUDA = -2,  /* a CUDA runtime call or kernel failed; see muca_last_error()            */
    MUCA_ERANGE = -3, /* iteration counter exhausted (0xFFFFFFFF is reserved for init, R5)      */
    MUCA_ENOMEM = -4  /* workspace too small / allocation failed                                */
} muca_status;

/* Sweep-kernel variants (muca_set_option(ctx, MUCA_OPT_KERNEL, ...)); every variant gives the same Markov chains.
 * AUTO picks RESIDENT for L <= 32 and STREAMED_PAIRS for L >= 64.
 *   RESIDENT       (L <= 32) lattices, threshold table and histogram in shared memory, Philox in paired deviate warps;
 *   STREAMED_PAIRS (L >= 32) table and histogram in shared memory, lattice rows streamed from HBM / L2, Philox in paired
 *                  deviate warps.  At L = 128 the table no longer fits: shared memory then holds a WINDOW of it around
 *                  the walkers' energies (one window for all walkers while they fit into it, otherwise one per block
 *                  over walkers sorted by energy, a few sweeps per launch); a launch in which a walker leaves its window
 *                  is detected, undone from a snapshot and repeated with STREAMED -- same results
 *                  (muca_window_stats() counts both);
 *   STREAMED       (L >= 32) thresholds read through L1, histogram in shared memory, lattice rows streamed, Philox in the
 *                  walker thread: the plain kernel and the fallback of the window.
 * A variant that does not exist for the context's L is replaced by the one AUTO would pick. */
enum { MUCA_KERNEL_AUTO = 0, MUCA_KERNEL_RESIDENT = 1, MUCA_KERNEL_STREAMED = 2, MUCA_KERNEL_STREAMED_PAIRS = 3 };
enum {
    MUCA_OPT_KERNEL = 1,          /* one of MUCA_KERNEL_*                                        */
    MUCA_OPT_THREADS_PER_BLOCK = 2, /* walkers per block (a multiple of 32); 0 = library default (walkers spread over all
                                      SMs).  RESIDENT, L <= 32: value / 32 (at most 4) walker warps, each paired with a
                                      deviate warp, i.e. twice as many threads */
    MUCA_OPT_MAX_SWEEPS_PER_LAUNCH = 3, /* split an iteration into launches of at most this many sweeps;
                                          0 = only as needed to keep a block's uint32 bins from overflowing */
    MUCA_OPT_WALKERS_PER_WARP = 4, /* resident kernel, L <= 32: walkers served by one warp (1..32); 0 = spread
                                     the walkers evenly over all SMs */
    MUCA_OPT_UPDATE_SCHEME = 5,   /* update scheme of muca_converge / muca_production: MUCA_SCHEME_TYPEWRITER (default;
                                     schedule rounded up to whole sweeps, R18) or MUCA_SCHEME_RANDOM_SITE (the paper's
                                     own scheme and units: N_therm = 30 w and N_updates attempted flips per walker;
                                     muca_production then runs therm_sweeps * N and sweeps * N updates per call) */
    MUCA_OPT_TABLE_WINDOW_ROWS = 6, /* STREAMED_PAIRS kernel: rows of the threshold-table window held in shared memory;
                                     0 = as many as fit.  A value below L*L+1 forces a window (testing) */
    MUCA_OPT_ROLE_MAP = 7,        /* resident kernel with 4 warp pairs per block: 0 = walker warps share schedulers with
                                     walker warps, 1 = every scheduler runs one walker and one deviate warp (A/B knob) */
    MUCA_OPT_ACCEPTANCE = 8       /* muca_run_iteration_random_site only: MUCA_ACCEPT_THRESHOLD (default: integer thresholds from
                                     double omega, R6/R7) or MUCA_ACCEPT_EXPF32, the paper's single-precision form (
                                     DESIGN.md R23): omega rounded to fp32, a proposal j -> j' is accepted iff the difference
                                     D = omega_f[j'] - omega_f[j] >= 0 or U < exp32(D), U the Philox word mapped to (0, 1] as
                                     cuRAND's curand_uniform maps it, exp32 a fixed sequence of fp32 operations (identical on
                                     CPU and GPU, which is what the paper asks of its own code) */
};
enum { MUCA_SCHEME_TYPEWRITER = 0, MUCA_SCHEME_RANDOM_SITE = 1 };
enum { MUCA_ACCEPT_THRESHOLD = 0, MUCA_ACCEPT_EXPF32 = 1 };

/* The walker count at which the current CUDA device is fully and evenly loaded by the default kernel for lattice size L --
 * the analogue of the paper's N_opt, "the first and lowest minimum" of the time per spin flip over the number of walkers,
 * which its code sets automatically when the user gives no W (W = 8 blocks x 256 threads x number of SMX;
 * :201 "the first optimum as automatically chosen by our code").  Here one block runs per SM and a walker warp is paired
 * with a deviate warp, so the optimum is
 *     n_walkers = (number of SMs) x pairs_per_sm x 32,   pairs_per_sm = 4 (L <= 32), 8 (L = 64), 4 (L = 128)
 * (the most warp pairs the default kernel runs per SM: the time per site of a walker grows more slowly than the number
 * of pairs, profiles/README.md "flips/s over W"); any multiple of it loads the SMs evenly as well and runs in as many
 * rounds.  Fewer walkers leave schedulers idle, a count in between loads the SMs unevenly.
 * Host logic + one device-attribute query.  MUCA_EINVAL for an unsupported L or NULL outputs, MUCA_ECUDA without a device. */
int muca_suggest_walkers(int L, int* n_walkers_out, int* pairs_per_sm_out);

/* Device workspace needed by muca_create_in() for (L, n_walkers); 0 on bad arguments. */
size_t muca_workspace_bytes(int L, int n_walkers);

/* Create a context and initialise the walkers on the device (R1, R2, R5):
 *   spin of site i = y*L + x of GLOBAL walker g = walker_offset + w is
 *   1 - 2*bit(i & 31) of word ((i >> 5) & 3) of Philox4x32-10(ctr = (i >> 7, 0, 0xFFFFFFFF, g),
 *   key = (seed & 0xFFFFFFFF, seed >> 32)); energies are computed from scratch (Eq. (5));
 *   omega == 0; iteration counter n = 0.
 * L must be one of 8, 16, 32, 64, 128 (R13); n_walkers >= 1.
 * muca_create      : the library allocates its own device memory and uses the legacy default stream.
 * muca_create_in   : device memory and stream are the caller's (e.g. a torch tensor and torch's
 *                    current stream): d_workspace must hold muca_workspace_bytes() bytes, be
 *                    256-byte aligned and outlive the context; cuda_stream is a cudaStream_t
 *                    (NULL = default stream).  walker_offset shards walkers over several
 *                    contexts/GPUs with results independent of the split (R16).
 * On failure *out is NULL and the status is returned. */
int muca_create(muca_ctx** out, int L, int n_walkers, uint64_t seed);
int muca_create_in(muca_ctx** out, int L, int n_walkers, uint64_t seed, uint32_t walker_offset,
                   void* d_workspace, size_t workspace_bytes, void* cuda_stream);
void muca_destroy(muca_ctx* ctx);

/* Tuning knobs (see the enums above). Returns MUCA_EINVAL for unknown options/values. */
int muca_set_option(muca_ctx* ctx, int option, int value);

/* omega(E_j) = ln W(E_j), j = 0..n_bins-1, host double[n_bins], n_bins must equal L*L+1.
 * set: copies the table into the context; does not touch spins or the iteration counter.
 * (the log-weights are the only state shared by the walkers.) */
int muca_set_log_weights(muca_ctx* ctx, const double* logw, int n_bins);
int muca_get_log_weights(muca_ctx* ctx, double* logw_out, int n_bins);

/* One MUCA iteration with the current fixed weights (Fig. 1):
 *   1. acceptance thresholds from omega, in double, on the host (R6, R7, R12):
 *        for slot j, a antiparallel neighbours, j' = j + 2 - a:
 *        a == 2 -> t = 0xFFFFFFFF;  j' outside [0, N] -> t = 0;
 *        d = omega[j'] - omega[j];  T = 2^32 if d >= 0 else floor(exp(d) * 2^32) clamped to [1, 2^32];
 *        t = T - 1;  a move is accepted iff the Philox word r <= t;
 *   2. therm_sweeps + sweeps typewriter sweeps of every walker on the device; the deviate of site i
 *      in sweep s of iteration n of global walker g is word (i & 3) of
 *      Philox4x32-10(ctr = (i >> 2, s, n, g), key);
 *   3. H[j] += 1 after every attempt (accepted or not) of the last `sweeps` sweeps, j the slot after
 *      the decision; per-block shared-memory histograms are merged into one uint64 histogram;
 *   4. n <- n + 1.
 * H_out: host uint64[n_bins] (may be NULL: H stays in the context for muca_update_weights /
 * muca_get_histogram).  sum(H) = n_walkers * sweeps * N.  therm_sweeps, sweeps >= 0.
 * Synchronises the context's stream before returning. */
int muca_run_iteration(muca_ctx* ctx, int therm_sweeps, int sweeps, uint64_t* H_out, int n_bins);

/* One iteration with the PAPER'S OWN update scheme (R22) instead of
 * typewriter sweeps: every update proposes the same random site in all walkers, each walker accepts with a deviate
 * of its own stream:
 *   update u = 0 .. therm_updates + updates - 1 of iteration n:
 *     site i_u = word (u & 3) of Philox4x32-10(ctr = (u >> 2 mod 2^32, u >> 34, n, 0xFFFFFFFF), key)  mod N,
 *     global walker g accepts iff word (u & 3) of Philox4x32-10(ctr = (u >> 2 mod 2^32, u >> 34, n, g), key) <= t,
 *     t = thresh[j][a] as in muca_run_iteration;  H[j] += 1 after every update with u >= therm_updates.
 * Work is counted in updates (attempted flips per walker), the paper's own unit.
 * Everything else (thresholds, H, iteration counter, muca_update_weights, muca_last_sweep_ms) as muca_run_iteration.
 * Kernel: threshold table and bins in shared memory, the shared site stream turned into per-update descriptors once per
 * block, the next update's neighbourhood loaded ahead of the current decision; 3.6e11 flips/s at L = 32
 * with 30 720 walkers -- about half the rate of the typewriter sweeps, which remain the tuned path. */
int muca_run_iteration_random_site(muca_ctx* ctx, uint64_t therm_updates, uint64_t updates, uint64_t* H_out, int n_bins);

/* Histogram of the last muca_run_iteration (host uint64[n_bins]). */
int muca_get_histogram(muca_ctx* ctx, uint64_t* H_out, int n_bins);

/* Eq. (4), R8: omega[j] -= ln(H[j]) for every j with H[j] > 0 (raw counts,
 * natural log, host double); unvisited slots keep their omega.
 * muca_update_weights      uses the H of the last muca_run_iteration on this context;
 * muca_update_weights_with uses a caller-supplied total histogram (host uint64[n_bins]) --
 *                          H summed over all shards when walkers are split over GPUs. */
int muca_update_weights(muca_ctx* ctx);
int muca_update_weights_with(muca_ctx* ctx, const uint64_t* H_total, int n_bins);

/* Per-walker energies E (host int32[n_walkers]) as tracked incrementally by the sweeps. */
int muca_get_energies(muca_ctx* ctx, int32_t* E_out, int n_walkers);

/* Spin configurations, host int8[n = n_walkers*L*L], out[w*N + y*L + x] = +1 / -1.
 * set: replaces the configurations and recomputes the energies from scratch on the device. */
int muca_get_spins(muca_ctx* ctx, int8_t* spins_out, size_t n);
int muca_set_spins(muca_ctx* ctx, const int8_t* spins, size_t n);

/* Same as muca_get_spins but into DEVICE memory int8[n] (no host copy); asynchronous on the
 * context's stream. */
int muca_unpack_spins_device(muca_ctx* ctx, void* d_spins_out, size_t n);

/* ---- Convergence driver (Sec. 3, Eq. (6), (7), Appendix A Eq. (A.1)) ----------------
 * Host logic around muca_run_iteration / muca_update_weights; the paper's schedule with whole sweeps as the unit
 * of work (R18: a number of attempted flips per walker is rounded UP to whole sweeps, at least one).
 *
 * muca_flatness: statistics of one histogram H (host uint64[n_bins]) against the flat distribution Q = 1/w:
 *   j_lo, j_hi  first / last visited slot;  width = j_hi - j_lo + 1 slots ("w'", in units of dE = 4; 0 if H == 0)
 *   d_k = sum_{H>0} P ln(P w),  P = H / sum(H)                                  (Eq. (6))
 *   d_c = max over the N - 1 accessible slots of |H / m - 1|,  m = sum(H)/(N - 1)   (Eq. (A.1))
 * w >= 1: the width of the flat reference;  w = 0: the paper's w = max(w', 10) under DESIGN.md R19:
 * w' = number of ACCESSIBLE slots (not 1 and N-1) in [j_lo, j_hi] of THIS histogram.  With the width
 * of an earlier, narrower histogram, or with the two unreachable slots counted, Q would not be normalised over the
 * support of P: d_k could be negative, and a perfectly flat histogram would give ln((N+1)/(N-1)) > 1e-4. */
typedef struct muca_flatness_t {
    int j_lo, j_hi, width;
    double d_k, d_c;
    uint64_t n_updates;   /* sum(H) */
} muca_flatness_t;
int muca_flatness(const uint64_t* H, int n_bins, int w, muca_flatness_t* out);

/* muca_schedule: work of the next iteration from the width w' covered by the previous one (0 before the first):
 *   w = max(w', 10);  N_therm = 30 w attempted flips per walker;
 *   N_updates = floor(6 w^2.25 / n_walkers) + 1 flips per walker (Eq. (7)), also in the first iteration with
 *   w = N + 1; from the second such iteration on N_updates <- floor(1.1 N_updates) + 1.
 *   *n_updates_io and *full_range_io carry N_updates and "the previous iteration had w = N + 1" over (start: 0, 0).
 *   therm_sweeps = ceil(N_therm / N), sweeps = ceil(N_updates / N)   (R18). */
int muca_schedule(int L, int n_walkers, int w_prev, double* n_updates_io, int* full_range_io, int* w_out,
                  int* therm_sweeps, int* sweeps);

/* One record per iteration of muca_converge (therm_sweeps / sweeps: the typewriter schedule; with
 * MUCA_SCHEME_RANDOM_SITE the iteration ran 30 w and flat.n_updates / n_walkers updates per walker instead). */
typedef struct muca_iteration_log_t {
    int w, therm_sweeps, sweeps;
    muca_flatness_t flat;
    double sweep_ms;      /* device time of the sweep kernel(s) */
} muca_iteration_log_t;

/* muca_converge: repeat { schedule; run_iteration; flatness; update_weights } until d_k < d_flat (the paper: 1e-4)
 * or max_iterations.  The weights are updated after EVERY iteration, the last one included.  log: host array of
 * log_capacity records (may be NULL); *iterations_out = iterations done; *converged_out = 1 if d_k < d_flat.
 * w_prev / n_updates start from 0 (first call on a context) -- the context keeps them, so a second call continues. */
int muca_converge(muca_ctx* ctx, int max_iterations, double d_flat, muca_iteration_log_t* log, int log_capacity,
                  int* iterations_out, int* converged_out);

/* ---- Production run with fixed weights and jackknife errors (Fig. 7) -----------------
 * n_calls >= 2 calls of muca_run_iteration(therm_sweeps, sweeps) with the CURRENT weights (which are not updated),
 * then, all in logarithms (R21):
 *   ln Omega(E_j) = ln H(E_j) - omega(E_j), H the sum of the call histograms, shifted so that
 *                   sum_j exp[ln Omega(E_j)] = 2^(L*L)
 *   err(E_j)      = delete-one jackknife error over the n_calls histograms, every leave-one-out estimate normalised
 *                   on its own: sqrt((n-1)/n * sum_k (x_k - mean x)^2)                       (ref. [46])
 * ln_omega_out, err_out: host double[n_bins]; NaN where a slot was not visited (ln Omega) or not visited by every
 * leave-one-out histogram (err).  H_calls_out: host uint64[n_calls * n_bins] or NULL.  The iteration counter advances
 * by n_calls; muca_get_histogram afterwards returns the histogram of the last call. */
int muca_production(muca_ctx* ctx, int n_calls, int therm_sweeps, int sweeps, double* ln_omega_out, double* err_out,
                    uint64_t* H_calls_out, int n_bins);

/* Debug / diagnostics.
 * thresholds: host uint32[n = n_bins*5], out[j*5 + a] as defined under muca_run_iteration, from the
 *             current omega.
 * iteration : the counter n that the next muca_run_iteration will use in the Philox counter.
 * last_sweep_ms: device time (CUDA events on the context's stream) of the sweep kernel launch(es)
 *             of the last muca_run_iteration, in milliseconds; *launches = number of kernel launches. */
int muca_get_thresholds(muca_ctx* ctx, uint32_t* out, size_t n);
int muca_get_iteration(muca_ctx* ctx, uint32_t* n_out);
int muca_set_iteration(muca_ctx* ctx, uint32_t n);
int muca_last_sweep_ms(muca_ctx* ctx, double* ms_out, int* launches_out);
/* STREAMED_PAIRS kernel with a table window (L = 128, or MUCA_OPT_TABLE_WINDOW_ROWS): iterations in which at least one
 * launch ran with a window so far, and launches that a walker left through a sentinel row and that were therefore undone
 * and repeated with the plain STREAMED kernel (same results either way).  Walkers spread over more rows than one window
 * holds are sorted by energy and served with one window per block, a few sweeps per launch. */
int muca_window_stats(muca_ctx* ctx, int* windowed_iterations_out, int* fallbacks_out);
const char* muca_last_error(const muca_ctx* ctx);

/* Test hook: Philox4x32-10 evaluated ON THE DEVICE for n (ctr, key) pairs.
 * ctr: host uint32[4n], key: host uint32[2n], out: host uint32[4n]. */
int muca_debug_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n);

/* The same test hook for callers that are not allowed to allocate device memory.
 *
 * Who that is: muca_debug_philox() above stages its rows in three buffers it cudaMalloc's and cudaFree's on every call.
 * That is fine for a stand-alone test program, but not for a host process in which someone else owns the GPU's memory --
 * a PyTorch (or similar) caching allocator that has already taken most of the HBM, or a job that runs with a fixed
 * memory partition: there a raw cudaMalloc can fail although the framework still has plenty of room, and both cudaMalloc
 * and cudaFree stall every stream of the device while they run, a running muca_run_iteration included.  Such a caller
 * (a start-up self-test of the device generator inside a long simulation, say) uses this entry point instead.
 *
 * What it does: the same kernel on the same rows, with the staging area in a fixed array that is part of the library
 * image: MUCA_PHILOX_STATIC_MAX rows of (ctr, key, out) = 160 KiB of device memory, held by every GPU on which the
 * library has been used, from the moment the CUDA runtime loads the library's device code there until the process
 * exits.  The function calls neither cudaMalloc / cudaFree nor any other allocating routine.
 *
 * ctr: host uint32[4n], key: host uint32[2n], out: host uint32[4n], all caller-owned; runs on the CURRENT device, legacy
 * default stream, and returns after `out` has been filled.
 *   n < 1 or a NULL pointer    -> MUCA_EINVAL;
 *   n > MUCA_PHILOX_STATIC_MAX -> MUCA_ENOMEM: the fixed array cannot hold the rows; nothing is copied or launched and
 *                                 `out` is untouched (split the rows over several calls, or use muca_debug_philox);
 *   a CUDA failure             -> MUCA_ECUDA.
 * First call on a device: it looks up where that device keeps the array (one cudaGetSymbolAddress with that device
 * current; the answer is remembered per device).  Make that first call at set-up, before any stream capture begins.
 * Shared state: all calls on one device use the same array, and it still holds the previous call's rows afterwards.
 * Nothing in it has to be zero at the start -- every word the kernel reads was written by this call's own copy-in, and
 * only the first n output rows, all of them written by this call's kernel, are copied out -- so stale rows never leak
 * into a result.  But two calls whose GPU work overlaps would overwrite each other's rows: the function therefore
 * holds a lock from copy-in to copy-out, which keeps calls made through this one loaded copy of the library apart.
 * Any other route to running two of them at once on one GPU is a data race. */
#define MUCA_PHILOX_STATIC_MAX 4096
int muca_debug_philox_static(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int n);

/* Library version string. */
const char* muca_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MUCA_H_ */
