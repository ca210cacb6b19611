// paper_1707_00919_b200/csrc/muca_resident.cuh
// Resident sweep kernel v5 for L <= 32 (sm_100a): "state in the address", walker warps paired with deviate warps.
// Citations: "PAPER.md:<line>" = /root/reference/PAPER.md, "R<n>" = DESIGN.md section 3.
//
// The walker's dynamic state -- energy slot j AND the carry c = [previous site of this row flipped] -- is ONE
// shared-memory address S = rowaddr(j, c).  The table is stored twice: copy c at byte offset c*K (K a power of
// two above copy 0, the lattices and the deviate ring); copy 1 has its columns permuted (f -> f ^ 1: a flipped
// left neighbour toggles the [left != s] bit of the column index).  Row (j, c) is 68 bytes (17 words: consecutive
// rows rotate through all 32 banks):
//     +4f      t  = thresh[j][a],  a = a(f ^ c)          (PAPER.md:109 acceptance, R6/R7)
//     +32+4f   Sa = rowaddr(j + 2 - a, 1)                 (state an ACCEPTED move leads to; a rejected one leads
//                                                          to rowaddr(j, 0) = S & ~K)
//     +64      histogram bin of slot j (copy 0 only: both copies of a slot count into it)
// Two 32-bit loads instead of one 64-bit load: a random-row LDS.64 takes 34 cycles (two 16-lane phases, each with
// its own bank conflicts), a random-row LDS.32 27 (profiles/r01_ubench_chain.txt); Sa arrives 3 cycles behind t.
// Per site the serial chain is   LDS t -> ISETP -> SEL(Sa, S & ~K) -> IADD (+ column of the next site) -> LDS t'.
// Column extraction, flip mask and histogram increment are off the chain.  Philox runs in a paired "deviate" warp
// (same walkers) that feeds a double-buffered shared ring one row ahead: the hardware interleaves its instruction
// stream into the stalls of the walker warps (at 4 pairs per SM, walker warps share schedulers with walker warps and
// deviate warps with deviate warps).  What was measured and dropped: a single in-order
// warp doing both (75 cycles per site), selecting between two precomputed entry addresses (ptxas folds the add
// into an instruction predicated on the decision, +11 cycles), and speculative loads for both outcomes of the
// next site (the walker warp becomes issue-bound at the same 49 cycles).
#pragma once
#include "muca_device.cuh"

namespace muca {


template <int L>
struct V5 {
    static constexpr uint32_t BINS = L * L + 1;
    static constexpr uint32_t RS = 68;
    static constexpr uint32_t SA_OFF = 32, BIN_OFF = 64;
    static constexpr uint32_t TBL_BYTES = (BINS + 1) * RS;   // + one all-reject row: parking place of unused lanes
    static constexpr int KBIT = L == 32 ? 17 : (L == 16 ? 16 : 15);
    static constexpr uint32_t K = 1u << KBIT;
    static constexpr uint32_t LAT_OFF = (TBL_BYTES + 15u) & ~15u;
    static constexpr int MAX_WARPS = 4;                      // walker warps per block (+ as many deviate warps)
    static constexpr int SLOTS = 32 * MAX_WARPS;             // lattice / ring columns
    static constexpr int NC = Geo<L>::BITS / 4;              // Philox calls per row
    static constexpr uint32_t RING_OFF = LAT_OFF + (uint32_t)L * 4u * SLOTS;
    static constexpr uint32_t RING_BYTES = 2u * NC * 16u * SLOTS;
    static_assert(1024u + RING_OFF + RING_BYTES <= K, "copy 0 + lattices + ring must end below K");
    static constexpr size_t SMEM_BYTES = (size_t)K + TBL_BYTES;
};

// Static planes of a row, split so that the part that does not depend on the row ABOVE (which the walker has only
// just finished) can be prepared one row ahead, in the shadow of the current row's table loads:
//   partial_words: nibble q of P[r] = hl + 2*(vd + hr) of site 4q + r   (hl/hr: left/right bond, vd: bond to the row below)
//   finish_words : FW[r] = P[r] + 2*vu   (vu: bond to the row above)  =  column f = hl + 2*n3 of field_words()
template <int L>
__device__ __forceinline__ void partial_words(const uint32_t c, const uint32_t dn, uint32_t (&P)[4], uint32_t& patch) {
    using G = Geo<L>;
    constexpr int BITS = G::BITS;
    uint32_t rw, lw;
    if constexpr (L >= 32) {
        rw = (c >> 1) | (c << 31);
        lw = (c << 1) | (c >> 31);
    } else {
        rw = (c >> 1) | ((c & 1u) << (BITS - 1));
        lw = ((c << 1) | (c >> (BITS - 1))) & G::MASK;
    }
    const uint32_t vd = c ^ dn, hr = c ^ rw, hl = c ^ lw;
    const uint32_t m0 = vd ^ hr, m1 = vd & hr;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t A = hl >> r;
        const uint32_t B = r >= 1 ? m0 >> (r - 1) : m0 << 1;
        const uint32_t C = r >= 2 ? m1 >> (r - 2) : m1 << (2 - r);
        const uint32_t t1 = (A & 0x11111111u) | (B & 0x22222222u);
        P[r] = t1 | (C & 0x44444444u);
    }
    constexpr int QL = BITS / 4 - 1;
    const uint32_t hr_last = (hr >> (BITS - 1)) & 1u;
    patch = (1u << (4 * QL + 1)) - (hr_last << (4 * QL + 2));   // site 0 flipped: n3 of the LAST site +-1
}
template <int L>
__device__ __forceinline__ void finish_words(const uint32_t (&P)[4], const uint32_t vu, uint32_t (&FW)[4]) {
    constexpr uint32_t M = Geo<L>::BITS == 32 ? 0x11111111u : (Geo<L>::BITS == 16 ? 0x1111u : 0x11u);
#pragma unroll
    for (int r = 0; r < 4; ++r) FW[r] = P[r] + 2u * ((vu >> r) & M);
}

// One site of the walker chain, in PTX.  Three things ptxas does not do by itself:
//  * the decision must be consumed by a SEL: ISETP -> SEL -> (IADD ->) LDS costs 9 (13) cycles on sm_100a, ISETP ->
//    predicated instruction -> LDS about 20 (profiles/r01_ubench_chain.txt).  ptxas turns "S = p ? sa : S & ~K" into a
//    predicated AND unless the AND has a second, unconditional use: here it is the address of the histogram
//    increment (the bin of copy 0 serves both copies);
//  * the walker warp is a single in-order instruction stream whose ISETP blocks until the threshold arrives, so
//    everything that does not depend on the decision should be issued BEFORE the ISETP, in the shadow of the
//    27-cycle table load.  The predicate chain ps -> pg -> ISETP (LOP3 with a predicate output; both are true at
//    run time: sr is a non-zero address) pins the ISETP behind the column extraction of the next site;
//  * H[j]++ of the PREVIOUS attempt is issued behind this site's table loads (S still holds that state).
//   %0 S: state address (in/out)    %1 A: entry address of this site (in), of the next site (out)
//   %2 flips (in/out)   %3 FW[3] at site 0 (in/out)   %4 deviate   %5 field word of the NEXT site   %6 its shift
//   %7 flip mask of this site   %8 ~K   %9 patch (site 0)
// The flip mask is a predicated OR (one ALU instruction; collecting bit K of the new state with SHF + LOP3 instead
// costs 1.7 cycles per site once two walker warps share a scheduler and its ALU pipe).
#define MUCA_V5_SITE(SHIFT_OP, EXTRA_LINE)                                       \
    "{\n\t.reg .pred p, ps, pg;\n\t.reg .b32 t, sa, sr, g0, g;\n\t"               \
    "ld.shared.u32 t, [%1];\n\t"                                                 \
    "ld.shared.u32 sa, [%1+32];\n\t"                                             \
    "setp.eq.u32 ps, 0, 0;\n\t"                                                  \
    "lop3.and.b32 sr|ps, %0, %8, 0, 0xC0, ps;\n\t"                               \
    "red.shared.add.u32 [sr+64], 1;\n\t"                                         \
    SHIFT_OP " g0, %5, %6;\n\t"                                                  \
    "lop3.or.b32 g|pg, g0, 0x1C, 0, 0xC0, ps;\n\t"                               \
    "setp.le.and.u32 p, %4, t, pg;\n\t"                                          \
    "selp.u32 %0, sa, sr, p;\n\t"                                                \
    "add.u32 %1, %0, g;\n\t"                                                     \
    "@p or.b32 %2, %2, %7;\n\t" EXTRA_LINE "}"

// One row of the walker warp.  In: the row above (`up`, final), this row (`c`, `P`, `patch`, `rnd`: old values, partial
// planes, deviates).  Out: the same for row y + 1 in (c1, P1, patch1, rnd1), fetched / prepared while this row is
// processed (none of it depends on this row; only "FW = P + 2*vu" waits for the row above), and `up` = this row's new
// value.  Every site increments the bin of the state it STARTS from, i.e. of the state after the previous attempt.
template <int L>
__device__ __forceinline__ void row_v5(uint32_t* __restrict__ lat, uint32_t& S, const int y, const bool more, uint32_t& up,
                                       const uint32_t c, const uint32_t (&P)[4], const uint32_t patch,
                                       const uint32_t (&rnd)[Geo<L>::BITS], uint32_t& c1, uint32_t (&P1)[4], uint32_t& patch1,
                                       uint32_t (&rnd1)[Geo<L>::BITS], const uint4* __restrict__ ring, int& buf,
                                       const int bar_id) {
    using G = Geo<L>;
    using V = V5<L>;
    constexpr int BITS = G::BITS, NC = V::NC, SLOTS = V::SLOTS;
    // the deviates of row y + 1 are in ring[buf]; ring[buf ^ 1] (this row's, already in registers) may be refilled.
    // After the last row of a phase there is no such barrier (the deviate warp has left its loop) and what is
    // fetched below is not used.
    if (more) pair_barrier(bar_id);
    uint32_t FW[4];
    finish_words<L>(P, c ^ up, FW);
    const int y1 = (y + 1) & (L - 1), y2 = (y + 2) & (L - 1);
    c1 = lat[y1 * SLOTS];
    partial_words<L>(c1, lat[y2 * SLOTS], P1, patch1);   // row y + 2 is old (or row 0, final in this sweep, when y + 1 = L - 1)
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const uint4 v = ring[(buf * NC + k) * SLOTS];
        rnd1[4 * k] = v.x; rnd1[4 * k + 1] = v.y; rnd1[4 * k + 2] = v.z; rnd1[4 * k + 3] = v.w;
    }
    buf ^= (int)more;
    S &= ~V::K;                        // site 0: its left neighbour (site L-1) has not been visited in this sweep
    uint32_t A = S + ((FW[0] << 2) & 0x1Cu);
    uint32_t flips = 0, unused = 0;    // `unused` fills operand %3 of the site macro where site 0 has FW[3]
#pragma unroll
    for (int x = 0; x < BITS; ++x) {
        // column of the next site: nibble qn of FW[xn & 3], moved to bits 2..4 inside the site block
        const int xn = x + 1, qn = xn >> 2;
        const uint32_t fwn = xn < BITS ? FW[xn & 3] : 0u;
        const uint32_t sh = qn == 0 ? 2u : (uint32_t)(4 * qn - 2);
        if (x == 0)                    // site 0 also patches the last site's column: its right neighbour is site 0
            asm volatile(MUCA_V5_SITE("shl.b32", "@p add.u32 %3, %3, %9;\n\t")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(FW[3])
                         : "r"(rnd[x]), "r"(fwn), "r"(sh), "r"(1u), "n"(~V::K), "r"(patch) : "memory");
        else if (qn == 0)
            asm volatile(MUCA_V5_SITE("shl.b32", "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused)
                         : "r"(rnd[x]), "r"(fwn), "r"(sh), "r"(1u << (x & 31)), "n"(~V::K) : "memory");
        else
            asm volatile(MUCA_V5_SITE("shr.u32", "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused)
                         : "r"(rnd[x]), "r"(fwn), "r"(sh), "r"(1u << (x & 31)), "n"(~V::K) : "memory");
    }
    up = c ^ flips;
    lat[y * SLOTS] = up;
}

// Walker warp: sweeps s0 .. s1-1; `buf` is the ring buffer holding the deviates of the next row to fetch.  Rows are
// processed in pairs so that the two register sets (this row / next row) swap roles without copies.
// The caller compensates the first and the last attempt of the measured phase in the histogram (see row_v5).
template <int L>
__device__ __forceinline__ void sweeps_v5(uint32_t* __restrict__ lat, uint32_t& S, const uint32_t s0, const uint32_t s1,
                                          const uint4* __restrict__ ring, int& buf, const int bar_id) {
    using G = Geo<L>;
    using V = V5<L>;
    constexpr int BITS = G::BITS, NC = V::NC, SLOTS = V::SLOTS;
    if (s1 <= s0) return;
    uint32_t up = lat[(L - 1) * SLOTS], cA = lat[0], cB;
    uint32_t PA[4], PB[4], patchA, patchB, rndA[BITS], rndB[BITS];
    partial_words<L>(cA, lat[SLOTS], PA, patchA);
    pair_barrier(bar_id);                      // the deviates of the first row are in ring[buf]
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const uint4 v = ring[(buf * NC + k) * SLOTS];
        rndA[4 * k] = v.x; rndA[4 * k + 1] = v.y; rndA[4 * k + 2] = v.z; rndA[4 * k + 3] = v.w;
    }
    buf ^= 1;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; y += 2) {
            row_v5<L>(lat, S, y, true, up, cA, PA, patchA, rndA, cB, PB, patchB, rndB, ring, buf, bar_id);
            row_v5<L>(lat, S, y + 1, s + 1 < s1 || y + 2 < L, up, cB, PB, patchB, rndB, cA, PA, patchA, rndA, ring, buf, bar_id);
        }
    }
}

// Deviate warp: the NC Philox calls of one row advance round-major (NC independent IMAD.WIDE chains), results go to
// the double-buffered shared ring rnd[buf][call][slot] as one 16-byte store per call.  One barrier per row hands
// the buffer over.  R4: ctr = (i >> 2, sweep, iteration, walker).
template <int L>
__device__ __forceinline__ void deviates_v5(uint4* __restrict__ ring, const uint32_t s0, const uint32_t s1, int& buf,
                                            const int bar_id, const SweepParams& prm, const uint32_t walker) {
    constexpr int NC = V5<L>::NC, SLOTS = V5<L>::SLOTS;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            uint32_t st[NC][4];
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                st[k][0] = (uint32_t)(y * (L / 4) + k); st[k][1] = s; st[k][2] = prm.iteration; st[k][3] = walker;
            }
#pragma unroll
            for (int r = 0; r < 10; ++r)
#pragma unroll
                for (int k = 0; k < NC; ++k)
                    philox_round(st[k], prm.key0 + (uint32_t)r * 0x9E3779B9u, prm.key1 + (uint32_t)r * 0xBB67AE85u);
#pragma unroll
            for (int k = 0; k < NC; ++k) ring[(buf * NC + k) * SLOTS] = make_uint4(st[k][0], st[k][1], st[k][2], st[k][3]);
            pair_barrier(bar_id);
            buf ^= 1;
        }
    }
}

// Block = nw walker warps + nw deviate warps, nw <= 4; walker warp i and deviate warp i ("pair" i) serve the same
// wpw <= 32 walkers, (b*nw + i)*wpw .. +wpw-1, in their lanes 0 .. wpw-1 (see the warp -> role map in the kernel).
// The host spreads the walkers over all SMs (as few pairs per SM, then as few lanes per warp, as possible: fewer
// lanes collide in the banks).  Lanes without a walker are parked on the all-reject row and never leave it.
template <int L>
__global__ void __launch_bounds__(64 * V5<L>::MAX_WARPS, 1) sweep_kernel_v5(const SweepParams prm, const int wpw) {
    using G = Geo<L>;
    using V = V5<L>;
    constexpr int N = G::N, BINS = G::BINS, SLOTS = V::SLOTS;
    extern __shared__ __align__(16) uint32_t smem[];
    char* const sm = reinterpret_cast<char*>(smem);
    const int tid = threadIdx.x, nthr = blockDim.x, nw = nthr >> 6;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    // the window must end below K, and no row address may be 0 (the site macro uses "S & ~K != 0" as an always-true
    // predicate; dynamic shared memory starts behind the 1 KB the system reserves on sm_100)
    if (sbase == 0u || sbase + V::RING_OFF + V::RING_BYTES > V::K) __trap();

    // ---- both table copies: row (j, c) = t[8] | Sa[8] | bin
    for (int idx = tid; idx < BINS * 16; idx += nthr) {
        const int j = idx >> 4, cc = (idx >> 3) & 1, f = idx & 7;
        const int fe = f ^ cc, a = (fe >> 1) + (fe & 1);
        int jn = j + 2 - a;                                  // where an accepted move leads (dE = 8 - 4a)
        uint32_t t = prm.table[j * 8 + fe];
        if (jn < 0 || jn > N) { jn = j; t = 0u; }            // R17: cannot occur for a real configuration
        char* const row = sm + (size_t)cc * V::K + (size_t)j * V::RS;
        *reinterpret_cast<uint32_t*>(row + 4 * f) = t;
        *reinterpret_cast<uint32_t*>(row + V::SA_OFF + 4 * f) = sbase + V::K + (uint32_t)jn * V::RS;
    }
    for (int idx = tid; idx < BINS * 2; idx += nthr)
        *reinterpret_cast<uint32_t*>(sm + (size_t)(idx & 1) * V::K + (size_t)(idx >> 1) * V::RS + V::BIN_OFF) = 0u;
    if (tid < 17)  // row BINS of copy 0: t = 0 and Sa = itself in every column -- a lane parked here stays here
        *reinterpret_cast<uint32_t*>(sm + (size_t)BINS * V::RS + 4 * tid) = tid >= 8 && tid < 16 ? sbase + BINS * V::RS : 0u;

    // warp -> role.  A warp runs on scheduler (warp id % 4).  With 4 pairs per block the walker warps take warp ids
    // {0, 1, 4, 5} and the deviate warps {2, 3, 6, 7}: two walker warps share a scheduler (each is latency-bound and
    // leaves 60 % of the issue slots to the other) and two deviate warps share one; a walker sharing with its deviate
    // warp instead loses 12 cycles per site to the Philox stream (profiles/README.md).  With 1 or 2 pairs every warp
    // has a scheduler of its own (deviate ids 0 .. nw-1, walker ids nw .. 2nw-1).
    const int warp_id = tid >> 5;
    const bool is_walker = nw == 4 ? (warp_id & 2) == 0 : warp_id >= nw;
    const int pair = nw == 4 ? (warp_id & 1) | ((warp_id >> 2) << 1) : (is_walker ? warp_id - nw : warp_id);
    const int lane = tid & 31, slot = 32 * pair + lane;          // slot: lattice / ring column
    const int w = (blockIdx.x * nw + pair) * wpw + lane;
    const bool active = lane < wpw && w < prm.W;
    const int bar_id = 1 + pair;
    uint32_t* const lat = reinterpret_cast<uint32_t*>(sm + V::LAT_OFF) + slot;
    uint4* const ring = reinterpret_cast<uint4*>(sm + V::RING_OFF);

    // ---- lattice: one word per row, column `slot`
    if (is_walker) {
        if (!active) {
            for (int y = 0; y < L; ++y) lat[y * SLOTS] = 0u;
        } else if (L >= 32) {
            for (int y = 0; y < L; ++y) lat[y * SLOTS] = prm.spins[(size_t)y * prm.W + w];
        } else {
            constexpr int RPW = 32 / G::BITS;
            for (int t = 0; t < N / 32; ++t) {
                const uint32_t word = prm.spins[(size_t)t * prm.W + w];
#pragma unroll
                for (int q = 0; q < RPW; ++q) lat[(t * RPW + q) * SLOTS] = (word >> (q * G::BITS)) & G::MASK;
            }
        }
    }
    __syncthreads();

    const uint32_t walker = prm.walker_offset + (uint32_t)w;
    const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                          : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
    // slot j = (E + 2N)/4, copy 0
    uint32_t S = sbase + (is_walker && active ? (uint32_t)((prm.E[w] + 2 * N) >> 2) : (uint32_t)BINS) * V::RS;
    int buf = 0;
    // ---- thermalisation sweeps: same code, the bins are cleared afterwards
    if (is_walker) sweeps_v5<L>(lat, S, prm.sweep_begin, s_th, ring + slot, buf, bar_id);
    else deviates_v5<L>(ring + slot, prm.sweep_begin, s_th, buf, bar_id, prm, walker);
    __syncthreads();
    for (int j = tid; j <= BINS; j += nthr) *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF) = 0u;
    __syncthreads();
    // ---- measured sweeps: every site counts the state it starts from, so the state before the first measured
    //      attempt is taken out again here and the state after the last one is added below
    if (is_walker) {
        if (s_th < prm.sweep_end) atomicSub(reinterpret_cast<uint32_t*>(sm + ((S & ~V::K) - sbase) + V::BIN_OFF), 1u);
        sweeps_v5<L>(lat, S, s_th, prm.sweep_end, ring + slot, buf, bar_id);
        if (s_th < prm.sweep_end) atomicAdd(reinterpret_cast<uint32_t*>(sm + ((S & ~V::K) - sbase) + V::BIN_OFF), 1u);
    } else {
        deviates_v5<L>(ring + slot, s_th, prm.sweep_end, buf, bar_id, prm, walker);
    }
    if (is_walker) {
        if (active) {
            prm.E[w] = (int)(((S & ~V::K) - sbase) / V::RS) * 4 - 2 * N;
            if (L >= 32) {
                for (int y = 0; y < L; ++y) prm.spins[(size_t)y * prm.W + w] = lat[y * SLOTS];
            } else {
                constexpr int RPW = 32 / G::BITS;
                for (int t = 0; t < N / 32; ++t) {
                    uint32_t word = 0u;
#pragma unroll
                    for (int q = 0; q < RPW; ++q) word |= lat[(t * RPW + q) * SLOTS] << (q * G::BITS);
                    prm.spins[(size_t)t * prm.W + w] = word;
                }
            }
        }
    }
    __syncthreads();

    // ---- a4: merge the block's bins into the global uint64 histogram
    if (prm.sweep_end > prm.therm) {
        for (int j = tid; j < BINS; j += nthr) {
            const uint32_t v = *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF);
            if (v) atomicAdd(prm.H + j, (unsigned long long)v);
        }
    }
}

}  // namespace muca
