// oracle/muca_oracle.cpp
//
// TEST INFRASTRUCTURE — NOT PRODUCT CODE.
// A plain, slow, obviously-correct CPU implementation of the hot path of
// parallel multicanonical simulation (arXiv 1707.00919) for the 2D Ising model.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load this.  It shares no code with the CUDA path
// in paper_1707_00919_b200/csrc and neither includes the other.
//
// Every function cites the passage of /root/reference/PAPER.md it follows
// ("PAPER.md:<line>") or the DESIGN.md reading ("R<n>") that fills a gap the
// paper leaves open.  Representation is deliberately naive: one int8 per spin,
// index arithmetic with explicit modulo, one histogram per thread.
//
// Pins (tests/test_oracle_pins.py, tests/test_philox_pin.py):
//   philox4x32_10      -> cuRAND's own Philox4x32-10 (toolkit routine, host build) + cuRAND host generator
//   energy / slot      -> brute force over all 2^16 states of L=4; exact g(E)
//   thresholds         -> arbitrary-precision evaluation (mpmath) of the same definition, +-1 ulp of libm
//   sweep order / H    -> omega == 0 closed form (every proposal accepted)
//   acceptance         -> omega = -beta*E: canonical <E>, H(E) against exact g(E) exp(-beta E)
//   whole recursion    -> exact finite-lattice density of states (Beale/Kaufman), max |d ln g| < 0.05
//   weight update      -> Eq. (4) retold in numpy on hand-made H
//   invariants         -> tracked E == recomputed E, sum H = W*sweeps*N, forbidden slots empty
//   random-site scheme -> omega == 0 closed form (site stream recomputed from the pinned Philox, H replayed in
//                         numpy), canonical weights against exact g(E) at L = 4   (tests/test_random_site.py)
//   fp32 acceptance    -> exp32 against mpmath (2 ulp), uniform32 against cuRAND's host generator (its uniform floats
//                         from the same raw words), canonical weights against exact g(E) at L = 4, threshold and fp32
//                         chains identical where every weight difference is 0 or -infinity-like   (tests/test_random_site.py)
// No function here is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ---------------------------------------------------------------------------
// Philox4x32-10 counter-based generator.
// PAPER.md:107 (Sec. 2.3): "stateless, counter-based RNG Philox proposed in
// Ref. [41]"; variant and round count are not stated in the paper -> DESIGN.md
// reading R4: Philox4x32, 10 rounds, multipliers 0xD2511F53 / 0xCD9E8D57,
// Weyl key increments 0x9E3779B9 / 0xBB67AE85 (Salmon et al., SC'11).
// One round:  (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)).
// ---------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

struct Oracle {
    int L = 0;                 // linear lattice size
    int N = 0;                 // N = L*L spins
    int W = 0;                 // number of walkers on this instance    ("p walkers")
    uint64_t seed = 0;
    uint32_t walker_offset = 0;   // global id of local walker 0 (R16: Philox uses the GLOBAL walker id)
    uint32_t iteration = 0;       // n, the weight-iteration counter
    std::vector<int8_t> spin;     // spin[w*N + y*L + x] in {+1,-1}
    std::vector<int32_t> E;       // tracked energy of every walker
    std::vector<double> logw;     // omega(E_j) = ln W(E_j), j = (E+2N)/4
    std::vector<uint64_t> H;      // histogram of the last iteration
};

// ---------------------------------------------------------------------------
// Ising energy, Eq. (5): H = -J sum_<ij> s_i s_j, J = 1,
// L x L periodic square lattice; every bond counted once (right and down
// neighbour of every site).
// ---------------------------------------------------------------------------
int energy_from_scratch(int L, const int8_t* s) {
    int E = 0;
    for (int y = 0; y < L; ++y)
        for (int x = 0; x < L; ++x) {
            const int here = s[y * L + x];
            const int right = s[y * L + (x + 1) % L];
            const int down = s[((y + 1) % L) * L + x];
            E -= here * right + here * down;
        }
    return E;
}

// Energy slot: "States are spaced at intervals dE = 4" on
// [-2L^2, 2L^2]  ->  j = (E + 2N)/4 in [0, N]   (R15: N+1 slots, slots 1 and N-1 unreachable).
inline int slot_of(int E, int N) { return (E + 2 * N) / 4; }

// ---------------------------------------------------------------------------
// Acceptance thresholds.  PAPER.md:109: Metropolis acceptance
// min(1, exp[omega(E') - omega(E)]).  R6/R7: the uniform deviate is a raw
// 32-bit Philox word r and the move is accepted iff r <= t, with
//   d = omega[j'] - omega[j]                     (one IEEE-754 double subtraction)
//   T = 2^32                     if d >= 0
//   T = floor(exp(d) * 2^32)     otherwise, clamped to [1, 2^32]
//   t = T - 1                    (so P(accept) = T / 2^32)
// a = number of antiparallel neighbours, move j -> j' = j + 2 - a.
// a == 2 (dE = 0) is always accepted (R9); j' outside [0,N] cannot occur for a
// real configuration and gets t = 0.
// Layout: out[j*5 + a], a = 0..4.
// ---------------------------------------------------------------------------
void build_thresholds(int n_bins, const double* logw, uint32_t* out) {
    for (int j = 0; j < n_bins; ++j) {
        for (int a = 0; a <= 4; ++a) {
            uint32_t t;
            const int jp = j + 2 - a;
            if (a == 2) {
                t = 0xFFFFFFFFu;
            } else if (jp < 0 || jp >= n_bins) {
                t = 0u;
            } else {
                const double d = logw[jp] - logw[j];
                uint64_t T;
                if (d >= 0.0) {
                    T = (uint64_t)1 << 32;
                } else {
                    const double scaled = std::floor(std::ldexp(std::exp(d), 32));
                    T = (uint64_t)scaled;
                    if (T < 1) T = 1;
                    if (T > ((uint64_t)1 << 32)) T = (uint64_t)1 << 32;
                }
                t = (uint32_t)(T - 1);
            }
            out[j * 5 + a] = t;
        }
    }
}

// ---------------------------------------------------------------------------
// Initial configuration.  The paper does not state it -> R1: uniform +-1 from
// the seed: site i of walker g takes bit (i & 31) of word ((i >> 5) & 3) of
// Philox(ctr = (i >> 7, 0, 0xFFFFFFFF, g), key = (seed_lo, seed_hi));
// bit 1 <-> spin -1.  R5: ctr[2] = 0xFFFFFFFF separates init from sweeps.
// ---------------------------------------------------------------------------
void init_walker(Oracle& o, int w) {
    const uint32_t key[2] = {(uint32_t)(o.seed & 0xFFFFFFFFu), (uint32_t)(o.seed >> 32)};
    const uint32_t g = o.walker_offset + (uint32_t)w;
    int8_t* s = &o.spin[(size_t)w * o.N];
    for (int i = 0; i < o.N; ++i) {
        const uint32_t ctr[4] = {(uint32_t)(i >> 7), 0u, 0xFFFFFFFFu, g};
        uint32_t r[4];
        philox4x32_10(ctr, key, r);
        const uint32_t word = r[(i >> 5) & 3];
        const uint32_t bit = (word >> (i & 31)) & 1u;
        s[i] = (int8_t)(1 - 2 * (int)bit);
    }
    o.E[w] = energy_from_scratch(o.L, s);
}

// ---------------------------------------------------------------------------
// One iteration for one walker.  PAPER.md:87 (walkers independent under shared
// fixed weights), PAPER.md:109 (Metropolis single spin flip)
// (thermalisation updates are not recorded), PAPER.md:119/:138 (H records the
// energy after EVERY attempted flip).  R3: sites are visited in typewriter
// order i = 0..N-1 (i = y*L + x) in every sweep.  R4: the deviate for site i in
// sweep s of iteration n of global walker g is word (i & 3) of
// Philox(ctr = (i >> 2, s, n, g), key).
// ---------------------------------------------------------------------------
void run_walker(const Oracle& o, int w, int therm, int sweeps, const uint32_t* thresh,
                int8_t* s, int32_t& E_io, uint64_t* H) {
    const int L = o.L, N = o.N;
    const uint32_t key[2] = {(uint32_t)(o.seed & 0xFFFFFFFFu), (uint32_t)(o.seed >> 32)};
    const uint32_t g = o.walker_offset + (uint32_t)w;
    int E = E_io;
    uint32_t r[4] = {0, 0, 0, 0};
    for (int sweep = 0; sweep < therm + sweeps; ++sweep) {
        for (int i = 0; i < N; ++i) {
            const int x = i % L, y = i / L;
            const int here = s[i];
            const int nb[4] = {
                s[y * L + (x + 1) % L],        // right
                s[y * L + (x + L - 1) % L],    // left
                s[((y + 1) % L) * L + x],      // down
                s[((y + L - 1) % L) * L + x],  // up
            };
            int a = 0;  // antiparallel neighbours, current values
            for (int k = 0; k < 4; ++k) a += (nb[k] != here);
            const int dE = 8 - 4 * a;  // flipping s_i turns a broken bonds into 4-a broken bonds
            if ((i & 3) == 0) {
                const uint32_t ctr[4] = {(uint32_t)(i >> 2), (uint32_t)sweep, o.iteration, g};
                philox4x32_10(ctr, key, r);
            }
            const uint32_t u = r[i & 3];
            const int j = slot_of(E, N);
            if (u <= thresh[j * 5 + a]) {
                s[i] = (int8_t)(-here);
                E += dE;
            }
            if (sweep >= therm) H[slot_of(E, N)] += 1;
        }
    }
    E_io = E;
}

// ---------------------------------------------------------------------------
// The paper's own update scheme: "using the same
// random number sequence for selecting the spins for all walkers, such that
// an update attempt simultaneously occurs at the same site of each replica
// ... The acceptance of updates using the Metropolis criterion is then tested
// with a second stream of random numbers that is chosen independently for
// each walker".  Work is counted in updates (attempted flips per walker,
// PAPER.md:138, :150-157), not sweeps.  Reading R22: update u = 0, 1, ... of
// iteration n proposes site i_u = (word (u & 3) of Philox(ctr = (u >> 2 mod 2^32,
// u >> 34, n, 0xFFFFFFFF), key)) mod N for EVERY walker; global walker g
// accepts iff word (u & 3) of Philox(ctr = (u >> 2 mod 2^32, u >> 34, n, g), key)
// <= thresh[j][a]  (walker ids are < 0xFFFFFFFF, so the site stream is nobody's
// acceptance stream).  The first `therm` updates are not recorded.
// ---------------------------------------------------------------------------
void run_walker_random_site(const Oracle& o, int w, uint64_t therm, uint64_t updates, const uint32_t* thresh,
                            int8_t* s, int32_t& E_io, uint64_t* H) {
    const int L = o.L, N = o.N;
    const uint32_t key[2] = {(uint32_t)(o.seed & 0xFFFFFFFFu), (uint32_t)(o.seed >> 32)};
    const uint32_t g = o.walker_offset + (uint32_t)w;
    int E = E_io;
    uint32_t rs[4] = {0, 0, 0, 0}, ra[4] = {0, 0, 0, 0};
    for (uint64_t u = 0; u < therm + updates; ++u) {
        if ((u & 3) == 0) {
            const uint32_t cs[4] = {(uint32_t)((u >> 2) & 0xFFFFFFFFu), (uint32_t)(u >> 34), o.iteration, 0xFFFFFFFFu};
            const uint32_t ca[4] = {(uint32_t)((u >> 2) & 0xFFFFFFFFu), (uint32_t)(u >> 34), o.iteration, g};
            philox4x32_10(cs, key, rs);
            philox4x32_10(ca, key, ra);
        }
        const int i = (int)(rs[u & 3] % (uint32_t)N);
        const int x = i % L, y = i / L;
        const int here = s[i];
        const int nb[4] = {s[y * L + (x + 1) % L], s[y * L + (x + L - 1) % L], s[((y + 1) % L) * L + x],
                           s[((y + L - 1) % L) * L + x]};
        int a = 0;
        for (int k = 0; k < 4; ++k) a += (nb[k] != here);
        const int j = slot_of(E, N);
        if (ra[u & 3] <= thresh[j * 5 + a]) {
            s[i] = (int8_t)(-here);
            E += 8 - 4 * a;
        }
        if (u >= therm) H[slot_of(E, N)] += 1;
    }
    E_io = E;
}

// ---------------------------------------------------------------------------
// Single-precision acceptance of the paper's own scheme (SURVEY 8(f)3 "optionally"; "We store the
// weights in single precision and hence also use a single precision version of the exponential function ... To ensure
// identical results between the CPU and GPU versions of the code, the example code provided does not use the hardware
// version __expf()").  Reading R23: omega_f[j] = (float) omega[j]; a proposal j -> j' = j + 2 - a with a != 2 is
// accepted iff D = omega_f[j'] - omega_f[j] (one fp32 subtraction) >= 0 or U < exp32(D), where
//   U        = fma32(fl32(x), 2^-32, 2^-33) in (0, 1]: the Philox word x mapped as cuRAND's curand_uniform does;
//   exp32(D) = the fixed sequence of IEEE fp32 operations below (so that CPU and GPU agree bit for bit, the paper's own
//              requirement; libm's expf differs between host and device): 0 for D < -24 (exp(-24) < 2^-33 <= U: such
//              a move is never accepted), else n = rint(D * log2 e), r = D - n ln 2 in two fma steps, a degree-6
//              Taylor polynomial of exp(r) in Horner form with fma, times 2^n.
// a == 2 (dE = 0) is always accepted (R9); j' outside [0, N] cannot occur and is rejected.
// ---------------------------------------------------------------------------
float uniform32(uint32_t x) { return fmaf((float)x, 2.3283064365386963e-10f, 1.1641532182693481e-10f); }

float exp32(float d) {
    if (d < -24.0f) return 0.0f;
    const float t = d * 1.4426950408889634f;          // log2(e), one fp32 product
    const long n = lrintf(t);                          // round to nearest even (default rounding mode)
    const float fn = (float)n;
    float r = fmaf(fn, -0.693145751953125f, d);        // ln 2 split: high part has 13 significant bits, n * hi is exact
    r = fmaf(fn, -1.428606765330187e-06f, r);
    float p = 1.0f / 720.0f;
    p = fmaf(p, r, 1.0f / 120.0f);
    p = fmaf(p, r, 1.0f / 24.0f);
    p = fmaf(p, r, 1.0f / 6.0f);
    p = fmaf(p, r, 0.5f);
    p = fmaf(p, r, 1.0f);
    p = fmaf(p, r, 1.0f);
    uint32_t bits = (uint32_t)(n + 127) << 23;         // 2^n, n in [-35, 0]
    float s;
    std::memcpy(&s, &bits, 4);
    return p * s;
}

void run_walker_random_site_expf(const Oracle& o, int w, uint64_t therm, uint64_t updates, const float* wf,
                                 int8_t* s, int32_t& E_io, uint64_t* H) {
    const int L = o.L, N = o.N;
    const uint32_t key[2] = {(uint32_t)(o.seed & 0xFFFFFFFFu), (uint32_t)(o.seed >> 32)};
    const uint32_t g = o.walker_offset + (uint32_t)w;
    int E = E_io;
    uint32_t rs[4] = {0, 0, 0, 0}, ra[4] = {0, 0, 0, 0};
    for (uint64_t u = 0; u < therm + updates; ++u) {
        if ((u & 3) == 0) {                            // the two streams of R22
            const uint32_t cs[4] = {(uint32_t)((u >> 2) & 0xFFFFFFFFu), (uint32_t)(u >> 34), o.iteration, 0xFFFFFFFFu};
            const uint32_t ca[4] = {(uint32_t)((u >> 2) & 0xFFFFFFFFu), (uint32_t)(u >> 34), o.iteration, g};
            philox4x32_10(cs, key, rs);
            philox4x32_10(ca, key, ra);
        }
        const int i = (int)(rs[u & 3] % (uint32_t)N);
        const int x = i % L, y = i / L;
        const int here = s[i];
        const int nb[4] = {s[y * L + (x + 1) % L], s[y * L + (x + L - 1) % L], s[((y + 1) % L) * L + x],
                           s[((y + L - 1) % L) * L + x]};
        int a = 0;
        for (int k = 0; k < 4; ++k) a += (nb[k] != here);
        const int j = slot_of(E, N), jn = j + 2 - a;
        bool accept;
        if (a == 2) accept = true;
        else if (jn < 0 || jn > N) accept = false;
        else {
            const float D = wf[jn] - wf[j];
            accept = D >= 0.0f || uniform32(ra[u & 3]) < exp32(D);
        }
        if (accept) {
            s[i] = (int8_t)(-here);
            E += 8 - 4 * a;
        }
        if (u >= therm) H[slot_of(E, N)] += 1;
    }
    E_io = E;
}

}  // namespace

// ---------------------------------------------------------------------------
// C exports (ctypes).  Return 0 on success, negative on bad arguments.
// ---------------------------------------------------------------------------
extern "C" {

void oracle_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
    philox4x32_10(ctr, key, out);
}

int oracle_energy(int L, const int8_t* spins) { return energy_from_scratch(L, spins); }

int oracle_thresholds(int n_bins, const double* logw, uint32_t* out) {
    if (n_bins < 2) return -1;
    build_thresholds(n_bins, logw, out);
    return 0;
}

// Eq. (4): W^(n+1)(E) = W^(n)(E) / H^(n)(E)  <=>
// omega[j] -= ln H[j].  R8: H is the RAW count; bins with H = 0 keep omega.
int oracle_weight_update(int n_bins, double* logw, const uint64_t* H) {
    for (int j = 0; j < n_bins; ++j)
        if (H[j] > 0) logw[j] = logw[j] - std::log((double)H[j]);
    return 0;
}

void* oracle_create(int L, int n_walkers, uint64_t seed, uint32_t walker_offset) {
    if (L < 4 || (L % 2) != 0 || n_walkers <= 0) return nullptr;  // R13: even L >= 4
    Oracle* o = new Oracle;
    o->L = L; o->N = L * L; o->W = n_walkers; o->seed = seed; o->walker_offset = walker_offset;
    o->spin.assign((size_t)n_walkers * o->N, 0);
    o->E.assign(n_walkers, 0);
    o->logw.assign(o->N + 1, 0.0);  // R2: omega == 0 initially
    o->H.assign(o->N + 1, 0);
    for (int w = 0; w < n_walkers; ++w) init_walker(*o, w);
    return o;
}

void oracle_destroy(void* h) { delete (Oracle*)h; }

int oracle_set_log_weights(void* h, const double* logw, int n_bins) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1) return -1;
    std::memcpy(o->logw.data(), logw, sizeof(double) * n_bins);
    return 0;
}

int oracle_get_log_weights(void* h, double* out, int n_bins) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1) return -1;
    std::memcpy(out, o->logw.data(), sizeof(double) * n_bins);
    return 0;
}

// PAPER.md:87-95 / Fig. 1: all walkers run with the same fixed weights, the
// total histogram is the sum of the walkers' histograms.  n_threads > 1 splits
// the walkers over OpenMP threads, each with a private histogram, summed at
// the end (integer sums: the result does not depend on n_threads).
int oracle_run_iteration(void* h, int therm_sweeps, int sweeps, uint64_t* H_out, int n_bins,
                         int n_threads) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1 || therm_sweeps < 0 || sweeps < 0) return -1;
    if (o->iteration == 0xFFFFFFFFu) return -2;  // R5: reserved for initialisation
    std::vector<uint32_t> thresh((size_t)n_bins * 5);
    build_thresholds(n_bins, o->logw.data(), thresh.data());
    if (n_threads < 1) n_threads = 1;
    std::vector<std::vector<uint64_t>> Hpriv(n_threads, std::vector<uint64_t>(n_bins, 0));
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(n_threads)
#endif
    for (int w = 0; w < o->W; ++w) {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        run_walker(*o, w, therm_sweeps, sweeps, thresh.data(), &o->spin[(size_t)w * o->N], o->E[w],
                   Hpriv[t].data());
    }
    for (int j = 0; j < n_bins; ++j) {
        uint64_t sum = 0;
        for (int t = 0; t < n_threads; ++t) sum += Hpriv[t][j];
        o->H[j] = sum;
        H_out[j] = sum;
    }
    o->iteration += 1;
    return 0;
}

int oracle_run_iteration_random_site(void* h, uint64_t therm_updates, uint64_t updates, uint64_t* H_out, int n_bins,
                                     int n_threads) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1) return -1;
    if (o->iteration == 0xFFFFFFFFu) return -2;
    std::vector<uint32_t> thresh((size_t)n_bins * 5);
    build_thresholds(n_bins, o->logw.data(), thresh.data());
    if (n_threads < 1) n_threads = 1;
    std::vector<std::vector<uint64_t>> Hpriv(n_threads, std::vector<uint64_t>(n_bins, 0));
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(n_threads)
#endif
    for (int w = 0; w < o->W; ++w) {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        run_walker_random_site(*o, w, therm_updates, updates, thresh.data(), &o->spin[(size_t)w * o->N], o->E[w],
                               Hpriv[t].data());
    }
    for (int j = 0; j < n_bins; ++j) {
        uint64_t sum = 0;
        for (int t = 0; t < n_threads; ++t) sum += Hpriv[t][j];
        o->H[j] = sum;
        H_out[j] = sum;
    }
    o->iteration += 1;
    return 0;
}

float oracle_exp32(float d) { return exp32(d); }
float oracle_uniform32(uint32_t x) { return uniform32(x); }

int oracle_run_iteration_random_site_expf(void* h, uint64_t therm_updates, uint64_t updates, uint64_t* H_out, int n_bins,
                                          int n_threads) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1) return -1;
    if (o->iteration == 0xFFFFFFFFu) return -2;
    std::vector<float> wf(n_bins);
    for (int j = 0; j < n_bins; ++j) wf[j] = (float)o->logw[j];   // R23: weights stored in single precision
    if (n_threads < 1) n_threads = 1;
    std::vector<std::vector<uint64_t>> Hpriv(n_threads, std::vector<uint64_t>(n_bins, 0));
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(n_threads)
#endif
    for (int w = 0; w < o->W; ++w) {
        int t = 0;
#ifdef _OPENMP
        t = omp_get_thread_num();
#endif
        run_walker_random_site_expf(*o, w, therm_updates, updates, wf.data(), &o->spin[(size_t)w * o->N], o->E[w],
                                    Hpriv[t].data());
    }
    for (int j = 0; j < n_bins; ++j) {
        uint64_t sum = 0;
        for (int t = 0; t < n_threads; ++t) sum += Hpriv[t][j];
        o->H[j] = sum;
        H_out[j] = sum;
    }
    o->iteration += 1;
    return 0;
}

int oracle_update_weights(void* h) {
    Oracle* o = (Oracle*)h;
    return oracle_weight_update(o->N + 1, o->logw.data(), o->H.data());
}

// Same update from an externally summed histogram (multi-rank: H = sum over ranks).
int oracle_update_weights_with(void* h, const uint64_t* H, int n_bins) {
    Oracle* o = (Oracle*)h;
    if (n_bins != o->N + 1) return -1;
    return oracle_weight_update(n_bins, o->logw.data(), H);
}

int oracle_get_energies(void* h, int32_t* out, int n_walkers) {
    Oracle* o = (Oracle*)h;
    if (n_walkers != o->W) return -1;
    std::memcpy(out, o->E.data(), sizeof(int32_t) * n_walkers);
    return 0;
}

int oracle_get_spins(void* h, int8_t* out, uint64_t n) {
    Oracle* o = (Oracle*)h;
    if (n != (uint64_t)o->W * o->N) return -1;
    std::memcpy(out, o->spin.data(), n);
    return 0;
}

int oracle_set_spins(void* h, const int8_t* in, uint64_t n) {
    Oracle* o = (Oracle*)h;
    if (n != (uint64_t)o->W * o->N) return -1;
    std::memcpy(o->spin.data(), in, n);
    for (int w = 0; w < o->W; ++w) o->E[w] = energy_from_scratch(o->L, &o->spin[(size_t)w * o->N]);
    return 0;
}

uint32_t oracle_get_iteration(void* h) { return ((Oracle*)h)->iteration; }
int oracle_set_iteration(void* h, uint32_t n) { ((Oracle*)h)->iteration = n; return 0; }

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
