// paper_1707_00919_b200/csrc/muca_streamed.cuh
// Sweep kernel for L >= 32 with the lattices STREAMED from HBM / L2 (walker-interleaved rows, one 4/8/16-byte vector per
// thread and row) and the v6 site chain of muca_resident.cuh: state in the address, two-candidate
// select, next state from the delta table, Philox in paired deviate warps, the unit one lattice row below prepared in
// the shadow of the table loads.  A "unit" is one 32-site word of a row (L / 32 words per row).
// Citations: "PAPER.md:<line>" = /root/reference/PAPER.md, "R<n>" = DESIGN.md section 3.
//
// Shared memory: DT[8] | Philox scratch (1 KB) | deviate ring (8 KB per pair) | threshold table, rows of 36 bytes (t[8] | bin).  The table
// holds rows [j_lo, j_lo + n_rows) of the N + 1 slots: all of them at L <= 64 (4097 rows = 147 KB), a WINDOW around the
// walkers' energies at L = 128 (16385 rows do not fit).  A walker may leave the window during the iteration.  That
// cannot be excluded beforehand, so it is DETECTED and the host repeats the iteration with the L1 kernel from a
// snapshot (muca.cu): the two outermost rows on a side that is not the end of the real table are sentinels with all
// thresholds 0 -- a walker that enters one cannot move on (up to an r = 0 deviate, probability 2^-32 per attempt, which
// the two zeroed pad rows beyond absorb) -- and every walker looks at its row after every 32-site word and remembers
// having seen a sentinel (for a walker to come back unseen, the r = 0 deviate would have to fall into those 32 attempts).
#pragma once
#include "muca_resident.cuh"

namespace muca {

constexpr int S6_PAD_ROWS = 2;        // zeroed rows before and behind the window
// walker/deviate warp pairs per block (barrier ids 1 .. 8): 8 pairs = 512 threads leave 128 registers per thread, which
// the four field-word sets of a 128-site row do not fit into (spills): at L = 128 at most 4 pairs (255 registers)
__host__ __device__ constexpr int s6_max_pairs(int L) { return L >= 128 ? 4 : 8; }
constexpr uint32_t S6_RS = 36, S6_BIN_OFF = 32;
constexpr uint32_t S6_SBASE = 1024;   // dynamic shared memory starts behind the 1 KB the system reserves on sm_100 (checked)
constexpr uint32_t S6_DTA = S6_SBASE; // the delta table sits first: the site macro addresses it by an immediate

__host__ __device__ constexpr size_t s6_ring_bytes(int npairs) { return (size_t)npairs * 2 * 8 * 32 * 16; }
constexpr uint32_t S6_SCRATCH_OFF = 32, S6_SCRATCH_BYTES = 8 * 8 * 16;   // behind DT: 16 bytes per call and deviate warp (philox_unit)
constexpr uint32_t S6_TAG_OFF = S6_SCRATCH_OFF + S6_SCRATCH_BYTES, S6_TAG_BYTES = 2 * 8 * 4;   // MUCA_CHECKED build: hand-over tags
constexpr uint32_t S6_RING_OFF = S6_TAG_OFF + S6_TAG_BYTES;
__host__ __device__ constexpr size_t s6_smem_bytes(int n_rows, int npairs) {
    return S6_RING_OFF + s6_ring_bytes(npairs) + (size_t)(n_rows + 2 * S6_PAD_ROWS) * S6_RS;
}

// Walker warp: sweeps s0 .. s1-1 over the streamed rows of one walker.
//   rows / row_stride: row y of this walker at rows + y * row_stride (WPR words); `store` false: a lane without a walker
//   win_lo / win_span: byte address of the first real row and bytes spanned by the real rows (sentinels excluded)
template <int L, bool MEAS>
__device__ __forceinline__ void sweeps_s6(uint32_t* __restrict__ rows, const size_t row_stride, const bool store, uint32_t& S,
                                          uint32_t& chk, bool& left, const uint32_t win_lo, const uint32_t win_span, const uint32_t s0,
                                          const uint32_t s1, const uint4* ring, const int slots, int& buf,
                                          const int bar_id, RingCheck& rc, const uint32_t all_lo, const uint32_t all_span) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR;
    static_assert(G::BITS == 32, "streamed kernel: rows of whole 32-site words");
    if (s1 <= s0) return;
    // rows y, y + 1, y + 2 (old values; R0 is replaced word by word by its new value) and the prefetch of row y + 3
    uint32_t R0[WPR], R1[WPR], R2[WPR], R3[WPR], up[WPR];
    ld_row<WPR>(rows + (size_t)(L - 1) * row_stride, up);
    ld_row<WPR>(rows, R0);
    ld_row<WPR>(rows + row_stride, R1);
    ld_row<WPR>(rows + (size_t)(2 % L) * row_stride, R2);
    uint32_t FWc[WPR][4], FWn[WPR][4], rnd[32], patch = 0, patch_n = 0;
    NextRow<L> n;
    SitePipe pp{0u, 0u, 0u};                   // unused by the non-pipelined site macro
#pragma unroll
    for (int k = 0; k < WPR; ++k) {            // field words of row 0 (the row above it, row L - 1, is final)
        n.c = R0[k]; n.left = R0[(k + WPR - 1) % WPR]; n.right = R0[(k + 1) % WPR]; n.dn = R1[k];
        prep_steps<L, 0, PREP_STEPS>(n);
#pragma unroll
        for (int r = 0; r < 4; ++r) FWc[k][r] = finish_word<L>(n, up[k], r);
        if (k == WPR - 1) patch = n.patch;
    }
    pair_barrier(bar_id);                      // the deviates of the first word are in ring[buf]
    ring_expect(rc, buf, CHK_RING_EARLY);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const uint4 v = ring[(buf * 8 + q) * slots];
        rnd[4 * q] = v.x; rnd[4 * q + 1] = v.y; rnd[4 * q + 2] = v.z; rnd[4 * q + 3] = v.w;
    }
    ring_fetched(rc, buf);
    buf ^= 1;
    uint32_t off = (FWc[0][0] << 2) & 0x1Cu;   // site 0: its left neighbour (site L-1) has not been visited in this sweep
    uint32_t A = S + off;
    uint32_t g1 = (FWc[0][1] << 2) & 0x1Cu, gx1 = g1 ^ 4u;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            const bool more_rows = s + 1 < s1 || y + 1 < L;
            ld_row<WPR>(rows + (size_t)((y + 3) & (L - 1)) * row_stride, R3);   // prefetch; rows 0 .. 2 of the next sweep are this sweep's
#pragma unroll
            for (int k = 0; k < WPR; ++k) {
                const bool more = more_rows || k + 1 < WPR;
                // the deviates of the next word are in ring[buf]; ring[buf ^ 1] (this word's, all fetched) may be refilled
                if (more) {
                    pair_barrier(bar_id);
                    ring_expect(rc, buf, CHK_RING_EARLY);
                }
                n.c = R1[k]; n.left = R1[(k + WPR - 1) % WPR]; n.right = R1[(k + 1) % WPR]; n.dn = R2[k];
                uint32_t flips = 0;
                if (k == 0 && k == WPR - 1)
                    RowSites<L, MEAS, 0, true, true, S6_DTA, false>::run(S, A, flips, chk, off, g1, gx1, R0[k], FWc[k], FWc[WPR - 1][3], patch, rnd, n,
                                                                  FWn[k], FWn[0], ring, slots, buf, more, pp);
                else if (k == 0)
                    RowSites<L, MEAS, 0, true, false, S6_DTA, false>::run(S, A, flips, chk, off, g1, gx1, R0[k], FWc[k], FWc[WPR - 1][3], patch, rnd, n,
                                                                   FWn[k], FWc[(k + 1) % WPR], ring, slots, buf, more, pp);
                else if (k == WPR - 1)
                    RowSites<L, MEAS, 0, false, true, S6_DTA, false>::run(S, A, flips, chk, off, g1, gx1, R0[k], FWc[k], FWc[WPR - 1][3], patch, rnd, n,
                                                                   FWn[k], FWn[0], ring, slots, buf, more, pp);
                else
                    RowSites<L, MEAS, 0, false, false, S6_DTA, false>::run(S, A, flips, chk, off, g1, gx1, R0[k], FWc[k], FWc[WPR - 1][3], patch, rnd, n,
                                                                    FWn[k], FWc[(k + 1) % WPR], ring, slots, buf, more, pp);
                if (more) ring_fetched(rc, buf);
                state_check(rc, S - all_lo < all_span && (S - all_lo) % S6_RS == 0u);   // a row of the window, its sentinels or its pads
                buf ^= (int)more;
                R0[k] ^= flips;
                FWn[k][3] = finish_word<L>(n, R0[k], 3);
                if (k == WPR - 1) patch_n = n.patch;
                left = left || (S - win_lo >= win_span);   // in a sentinel or pad row (unsigned compare; the parking row counts as well)
            }
            if (store) st_row<WPR>(rows + (size_t)y * row_stride, R0);
#pragma unroll
            for (int k = 0; k < WPR; ++k) {
                R0[k] = R1[k]; R1[k] = R2[k]; R2[k] = R3[k];
#pragma unroll
                for (int r = 0; r < 4; ++r) FWc[k][r] = FWn[k][r];
            }
            patch = patch_n;
        }
    }
}

// Deviate warp: the 8 Philox calls of a 32-site word advance round-major (philox_unit), results go to the double-buffered
// ring rnd[buf][call][slot] as one 16-byte store per call (lanes without a walker store nothing: their slots hold
// 0xFFFFFFFF for good).  One barrier per word hands the buffer over.  R4: ctr = (i >> 2, sweep, iteration, walker).
template <int L>
__device__ __forceinline__ void deviates_s6(uint4* ring, uint4* scratch, const int slots, int& buf, const int bar_id, const uint32_t s0,
                                            const uint32_t s1, const SweepParams& prm, const uint32_t walker, const bool active, const int lane,
                                            RingCheck& rc) {
    constexpr int WPR = Geo<L>::WPR;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
        const PhiloxSweep pc = philox_sweep_consts(s, prm.iteration, prm.key0, prm.key1);
#pragma unroll 1
        for (int word = 0; word < L * WPR; ++word) {      // typewriter word: sites 32 word .. 32 word + 31, calls 8 word .. + 7
            uint32_t st[8][4];
            philox_unit<8>(st, scratch, (uint32_t)(word * 8), pc, walker, lane);
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (active) ring[(buf * 8 + q) * slots] = make_uint4(st[q][0], st[q][1], st[q][2], st[q][3]);
            ring_publish(rc, buf, lane);
            pair_barrier(bar_id);
            buf ^= 1;
        }
    }
}

// Block = npairs walker warps + npairs deviate warps; pair p serves the 32 walkers blockIdx.x * 32 * npairs + 32 p ...
// A warp runs on scheduler (warp id % 4).  role_map 0: walker warps have even warp ids, deviate warps odd ones --
// walker warps share schedulers with walker warps; role_map 1: walker and deviate warps alternate on every scheduler.
template <int L>
__global__ void __launch_bounds__(64 * s6_max_pairs(L), 1)
sweep_kernel_s6(const SweepParams prm, const int j_lo_all, const int n_rows, const int sent_lo_all, const int sent_hi_all, const int role_map,
                int* __restrict__ overflow, const int* __restrict__ perm, const int* __restrict__ blk_j_lo) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, N = G::N;
    extern __shared__ __align__(16) uint32_t smem[];
    char* const sm = reinterpret_cast<char*>(smem);
    const int tid = threadIdx.x, nthr = blockDim.x, npairs = nthr >> 6;
    const int warp_id = tid >> 5, lane = tid & 31;
    const bool is_walker = role_map == 0 ? (warp_id & 1) == 0 : (((warp_id >> 2) + warp_id) & 1) == 0;
    // role_map 1: warps 4m .. 4m + 3 (one per scheduler) alternate W D W D for even m and D W D W for odd m; pair = rank of
    // the warp among the warps of its role
    const int pair = role_map == 0 ? warp_id >> 1 : ((warp_id >> 2) << 1) | ((warp_id & 3) >> 1);
    const int slot = 32 * pair + lane, slots = 32 * npairs;
    // Walkers are independent and identified by their GLOBAL id (R16), so which block serves which walker is free: with
    // `perm` the host hands every block walkers of neighbouring energies (sorted) and a table window of its own
    // (blk_j_lo[block]) -- the way the window keeps up with walkers that are spread over the whole energy range.
    const int idx = blockIdx.x * slots + slot;
    const bool active = idx < prm.W;
    const int w = perm ? perm[active ? idx : prm.W - 1] : idx;
    const int j_lo = blk_j_lo ? blk_j_lo[blockIdx.x] : j_lo_all;
    const int sent_lo = blk_j_lo ? (j_lo > 0 ? 2 : 0) : sent_lo_all;
    const int sent_hi = blk_j_lo ? (j_lo + n_rows < N + 1 ? 2 : 0) : sent_hi_all;
    if (!smem_base_ok(prm, (uint32_t)__cvta_generic_to_shared(smem), S6_SBASE)) return;   // the site macro addresses the delta table by an immediate
    uint4* const ring = reinterpret_cast<uint4*>(sm + S6_RING_OFF) + slot;
    uint4* const scratch = reinterpret_cast<uint4*>(sm + S6_SCRATCH_OFF) + pair * 8;
    char* const win = sm + S6_RING_OFF + s6_ring_bytes(npairs);
    char* const tbl = win + S6_PAD_ROWS * S6_RS;                        // row 0 of the window
    // ---- table window: row jl = t[8] | bin; pad and sentinel rows: all thresholds 0
    for (int idx = tid; idx < (n_rows + 2 * S6_PAD_ROWS) * 9; idx += nthr) {
        const int jl = idx / 9 - S6_PAD_ROWS, e = idx - (jl + S6_PAD_ROWS) * 9;
        const bool real = jl >= sent_lo && jl < n_rows - sent_hi;      // neither pad nor sentinel
        uint32_t v = 0u;
        if (e < 8 && real) {
            const int j = j_lo + jl, jn = j + 2 - ((e >> 1) + (e & 1));
            // R17: a move out of [0, N] cannot occur for a real configuration; its entry is never consulted
            if (jn >= 0 && jn <= N) v = prm.table[(size_t)j * 8 + e];
        }
        *reinterpret_cast<uint32_t*>(win + (size_t)idx * 4) = v;
    }
    if (tid < 8) *reinterpret_cast<int32_t*>(sm + 4 * tid) = (int)S6_RS * (2 - ((tid >> 1) + (tid & 1)));   // DT[f] = RS * (2 - a(f))
    // a lane without a walker never accepts: its ring slots hold the deviate 0xFFFFFFFF for good and it sits on pad row -1
    if (!is_walker && !active)
        for (int q = 0; q < 16; ++q) ring[q * slots] = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);
    __syncthreads();

    const uint32_t o_base = S6_SBASE + S6_RING_OFF + (uint32_t)s6_ring_bytes(npairs) + S6_PAD_ROWS * S6_RS;   // address of window row 0
    const uint32_t win_lo = o_base + (uint32_t)sent_lo * S6_RS, win_span = (uint32_t)(n_rows - sent_lo - sent_hi) * S6_RS;
    const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                          : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
    // Lanes without a walker take part in the pair barriers of their warp, so they run the same code: they read the
    // rows of the last walker and store nothing.
    const int wl = active ? w : (perm ? w : prm.W - 1);
    uint32_t* rows = prm.spins + (size_t)wl * WPR;
    const size_t row_stride = (size_t)prm.W * WPR;
    const uint32_t walker = prm.walker_offset + (uint32_t)w;
    // slot j = (E + 2N)/4; the host put every walker inside the window
    uint32_t S = active && is_walker ? o_base + (uint32_t)(((prm.E[w] + 2 * N) >> 2) - j_lo) * S6_RS : o_base - S6_RS;
    int buf = 0;
    uint32_t chk = 0;
    bool left = false;
    const int bar_id = 1 + pair;
    RingCheck rc;
#ifdef MUCA_CHECKED
    rc.tags = reinterpret_cast<volatile uint32_t*>(sm + S6_TAG_OFF) + pair;
    rc.stride = 8;
    rc.flag = prm.check;
    rc.fault = blockIdx.x == 0 && pair == 0 ? prm.fault : 0u;
#endif
    const uint32_t all_lo = o_base - S6_PAD_ROWS * S6_RS, all_span = (uint32_t)(n_rows + 2 * S6_PAD_ROWS) * S6_RS;
    if (is_walker) {
        sweeps_s6<L, false>(rows, row_stride, active, S, chk, left, win_lo, win_span, prm.sweep_begin, s_th, ring, slots, buf, bar_id, rc, all_lo, all_span);
        // measured sweeps: every site counts the state it starts from, so the state before the first measured attempt
        // is taken out again here and the state after the last one is added below
        if (s_th < prm.sweep_end) atomicSub(reinterpret_cast<uint32_t*>(sm + (S - S6_SBASE) + S6_BIN_OFF), 1u);
        sweeps_s6<L, true>(rows, row_stride, active, S, chk, left, win_lo, win_span, s_th, prm.sweep_end, ring, slots, buf, bar_id, rc, all_lo, all_span);
        if (s_th < prm.sweep_end) atomicAdd(reinterpret_cast<uint32_t*>(sm + (S - S6_SBASE) + S6_BIN_OFF), 1u);
        if (chk == 0x9E3779B9u && !active) ring[0] = make_uint4(chk, chk, chk, chk);   // keeps the checksum of the site macro alive (never true for a parked lane: its addresses are constant)
        if (active) {
            prm.E[w] = ((int)((S - o_base) / S6_RS) + j_lo) * 4 - 2 * N;
            if (left) atomicOr(overflow, 1);
        }
    } else {
        deviates_s6<L>(ring, scratch, slots, buf, bar_id, prm.sweep_begin, s_th, prm, walker, active, lane, rc);
        deviates_s6<L>(ring, scratch, slots, buf, bar_id, s_th, prm.sweep_end, prm, walker, active, lane, rc);
    }
    __syncthreads();
    // ---- a4: merge the bins of the real rows into the global uint64 histogram
    if (prm.sweep_end > prm.therm)
        for (int jl = sent_lo + tid; jl < n_rows - sent_hi; jl += nthr) {
            const uint32_t v = *reinterpret_cast<uint32_t*>(tbl + (size_t)jl * S6_RS + S6_BIN_OFF);
            if (v) atomicAdd(prm.H + j_lo + jl, (unsigned long long)v);
        }
}

}  // namespace muca
