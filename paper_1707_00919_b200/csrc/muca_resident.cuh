// paper_1707_00919_b200/csrc/muca_resident.cuh
// Resident sweep kernel v6 for L <= 32 (sm_100a): "state in the address", two-candidate select, walker warps paired
// with deviate warps, everything that is not the per-site chain spread over the sites of the previous row.
// Citations: "PAPER.md:<line>" = /root/reference/PAPER.md, "R<n>" = DESIGN.md section 3.
//
// The walker's dynamic state is the shared-memory address S = rowaddr(j) of its energy slot j; the carry
// c = [previous site of this row flipped] lives in the ENTRY address A of the next lookup.  The table is stored twice:
// copy c at byte offset c*K (K a power of two above copy 0, the lattices and the deviate ring); copy 1 has its columns
// permuted (f -> f ^ 1: a flipped left neighbour toggles the [left != s] bit of the column index).  Row (j, c) is 68
// bytes (17 words: consecutive rows rotate through all 32 banks):
//     +4f      t  = thresh[j][a],  a = a(f ^ c)          (PAPER.md:109 acceptance, R6/R7)
//     +32+4f   Sa = rowaddr(j + 2 - a)                    (state an ACCEPTED move leads to; a rejected one keeps S)
//     +64      histogram bin of slot j (copy 0 only)
// Per site the serial chain is   LDS t -> ISETP -> SEL(A_acc, A_rej) -> LDS t'   with BOTH candidates of the next
// entry address, A_acc = Sa + K + 4f' and A_rej = S + 4f', formed before the decision (round 1, v5, selected the
// state and added the column afterwards: ISETP -> SEL -> IADD -> LDS).  Philox runs in a paired "deviate" warp (same
// walkers) that feeds a double-buffered shared ring one row ahead.
//
// What the ncu source view of v5 showed (profiles/README.md, round 2): a steady-state site cost 46 cycles, but the
// row prologue -- eight 16-byte ring loads in one burst (32 wavefronts queued in front of the first table loads) and
// ~70 instructions of bit-sliced preparation -- added another 340 cycles per row, 10.7 per site.  Here the deviates
// of row y + 1 replace those of row y in place, one 16-byte load per four sites, and the field words of row y + 1 are
// prepared a step per site in the shadow of the table loads; the part that depends on the row above is finished as
// soon as the last site of its residue class (x & 3) has been decided.
#pragma once
#include "muca_device.cuh"

namespace muca {

#ifndef MUCA_SITE_VARIANT
#define MUCA_SITE_VARIANT 7
#endif
#if MUCA_SITE_VARIANT == 7
#define MUCA_V6_DT 1   // the state an accepted move leads to is computed from a 16-word delta table instead of loaded from the row
#endif

template <int L>
struct V6 {
    static constexpr uint32_t SBASE = 1024;                  // dynamic shared memory starts behind the 1 KB the system reserves on sm_100 (checked)
    static constexpr uint32_t BINS = L * L + 1;
#ifdef MUCA_V6_DT
    // row (j, c): t[8] | bin (copy 0 only) = 9 words (odd: consecutive rows rotate through all 32 banks);
    // behind the rows of copy c: DT[c][f] = RS * (2 - a(f ^ c)), the state change of an accepted move
    static constexpr uint32_t RS = 36, BIN_OFF = 32;
    static constexpr uint32_t DT_OFF = (BINS + 1) * RS;      // + one all-reject row: parking place of unused lanes
    static constexpr uint32_t COPY_BYTES = DT_OFF + 32;
    // K = offset of copy 1; K % 128 == 32 puts DT[1][f] into other banks than DT[0][f]: a warp's delta load is one wavefront
    static constexpr uint32_t K = (COPY_BYTES + 127u) / 128u * 128u + 32u;
    static constexpr uint32_t LAT_OFF = (K + COPY_BYTES + 15u) & ~15u;
#else
    static constexpr uint32_t RS = 68;
    static constexpr uint32_t SA_OFF = 32, BIN_OFF = 64;
    static constexpr uint32_t TBL_BYTES = (BINS + 1) * RS;   // + one all-reject row: parking place of unused lanes
    static constexpr int KBIT = L == 32 ? 17 : (L == 16 ? 16 : 15);
    static constexpr uint32_t K = 1u << KBIT;
    static constexpr uint32_t LAT_OFF = (TBL_BYTES + 15u) & ~15u;
#endif
    static constexpr int MAX_WARPS = 4;                      // walker warps per block (+ as many deviate warps)
    static constexpr int SLOTS = 32 * MAX_WARPS;             // lattice / ring columns
    static constexpr int NC = Geo<L>::BITS / 4;              // Philox calls per row
    static constexpr uint32_t RING_OFF = LAT_OFF + (uint32_t)L * 4u * SLOTS;
    static constexpr uint32_t RING_BYTES = 2u * NC * 16u * SLOTS;
#ifdef MUCA_V6_DT
    static constexpr size_t SMEM_BYTES = (size_t)RING_OFF + RING_BYTES;
#else
    static_assert(1024u + RING_OFF + RING_BYTES <= K, "copy 0 + lattices + ring must end below K");
    static constexpr size_t SMEM_BYTES = (size_t)K + TBL_BYTES;
#endif
};

// Field words of a row: nibble q of FW[r] holds the column f = hl + 2*n3 of site 4q + r (hl: bond to the left
// neighbour's OLD value, n3 = antiparallel bonds to up / down / right).  They are built in two parts so that most of
// the work can be done a row ahead: the planes that do not depend on the row ABOVE (which the walker is still
// updating) go into P[r] = hl + 2*(vd + hr), one small step per site of the row before (prep_step), and
// FW[r] = P[r] + 2*vu is finished when the sites 4q + r of the row above are final (finish_word).
template <int L>
struct NextRow {
    uint32_t c, dn;            // the row (old value) and the row below it (old; row 0, already final, below row L-1)
    uint32_t hl, hr, m0, m1;   // bond planes: left, right, (down + right) as sum and carry bits
    uint32_t t;
    uint32_t P[4];
    uint32_t patch;            // added to FW[3] when site 0 flips: n3 of the LAST site of the row changes by +-1
};

constexpr int PREP_STEPS = 17;

template <int L, int I>
__device__ __forceinline__ void prep_step(NextRow<L>& n) {
    using G = Geo<L>;
    constexpr int BITS = G::BITS;
    if constexpr (I == 0) {
        const uint32_t rw = L >= 32 ? __funnelshift_r(n.c, n.c, 1) : ((n.c >> 1) | ((n.c & 1u) << (BITS - 1)));
        n.hr = n.c ^ rw;
    } else if constexpr (I == 1) {
        const uint32_t lw = L >= 32 ? __funnelshift_l(n.c, n.c, 1) : (((n.c << 1) | (n.c >> (BITS - 1))) & G::MASK);
        n.hl = n.c ^ lw;
    } else if constexpr (I == 2) {
        n.m0 = n.c ^ n.dn ^ n.hr;
    } else if constexpr (I == 3) {
        n.m1 = (n.c ^ n.dn) & n.hr;
    } else if constexpr (I < 16) {
        constexpr int r = (I - 4) / 3, part = (I - 4) % 3;
        if constexpr (part == 0) n.t = (n.hl >> r) & 0x11111111u;
        else if constexpr (part == 1) n.t |= (r >= 1 ? n.m0 >> (r >= 1 ? r - 1 : 0) : n.m0 << 1) & 0x22222222u;
        else n.P[r] = n.t | ((r >= 2 ? n.m1 >> (r >= 2 ? r - 2 : 0) : n.m1 << (2 - r)) & 0x44444444u);
    } else {
        constexpr int QL = BITS / 4 - 1;
        const uint32_t hr_last = (n.hr >> (BITS - 1)) & 1u;
        n.patch = (1u << (4 * QL + 1)) - (hr_last << (4 * QL + 2));
    }
}
template <int L, int I0, int I1>
__device__ __forceinline__ void prep_steps(NextRow<L>& n) {
    if constexpr (I0 < I1) {
        prep_step<L, I0>(n);
        prep_steps<L, I0 + 1, I1>(n);
    }
}
// the steps that follow site x of the row above: sites 0 .. BITS-5 share the PREP_STEPS steps evenly, the last four
// sites are left to finish_word
template <int L>
__device__ __forceinline__ void prep_for_site(NextRow<L>& n, const int x) {
    constexpr int D = Geo<L>::BITS - 4;
    switch (x) {
#define MUCA_PREP_CASE(X) case X: if constexpr (X < D) prep_steps<L, (X * PREP_STEPS) / D, ((X + 1) * PREP_STEPS) / D>(n); break;
        MUCA_PREP_CASE(0) MUCA_PREP_CASE(1) MUCA_PREP_CASE(2) MUCA_PREP_CASE(3) MUCA_PREP_CASE(4) MUCA_PREP_CASE(5) MUCA_PREP_CASE(6)
        MUCA_PREP_CASE(7) MUCA_PREP_CASE(8) MUCA_PREP_CASE(9) MUCA_PREP_CASE(10) MUCA_PREP_CASE(11) MUCA_PREP_CASE(12)
        MUCA_PREP_CASE(13) MUCA_PREP_CASE(14) MUCA_PREP_CASE(15) MUCA_PREP_CASE(16) MUCA_PREP_CASE(17) MUCA_PREP_CASE(18)
        MUCA_PREP_CASE(19) MUCA_PREP_CASE(20) MUCA_PREP_CASE(21) MUCA_PREP_CASE(22) MUCA_PREP_CASE(23) MUCA_PREP_CASE(24)
        MUCA_PREP_CASE(25) MUCA_PREP_CASE(26) MUCA_PREP_CASE(27)
#undef MUCA_PREP_CASE
        default: break;
    }
}
// FW[r] of the row below `above_new` (bits 4q + r of above_new must be final)
template <int L>
__device__ __forceinline__ uint32_t finish_word(const NextRow<L>& n, const uint32_t above_new, const int r) {
    constexpr uint32_t M = Geo<L>::BITS == 32 ? 0x11111111u : (Geo<L>::BITS == 16 ? 0x1111u : 0x11u);
    return n.P[r] + 2u * (((n.c ^ above_new) >> r) & M);
}

// One site of the walker chain, in PTX.
//   %0 S: state address (in/out)    %1 A: entry address of this site (in), of the next site (out)
//   %2 flips (in/out)   %3 FW[3] at site 0 (in/out)   %4 deviate   %5 field word of the NEXT site   %6 its shift
//   %7 flip mask of this site   %8 K (0 at the last site of a row: the next row starts without a carry)   %9 patch (site 0)
// H[j]++ of the PREVIOUS attempt is issued behind this site's table loads (S still holds that state); thermalisation
// sweeps leave it out.  The flip mask is a predicated OR.
//   %0 S   %1 A   %2 flips   %3 FW[3] at site 0   %4 checksum   %5 delta-table offset A - S (variant 7)
//   %6 deviate   %7 field word of the NEXT site   %8 its shift   %9 flip mask   %10 K (0 at the last site of a row)
//   %11 patch (site 0)   %12 address of DT[0][0] (variant 7)
#if MUCA_SITE_VARIANT == 3     // Sa loaded from the row (in front of t: volatile loads keep their order)
#define MUCA_V6_SITE(SHIFT_OP, HIST_LINE, EXTRA_LINE)                            \
    "{\n\t.reg .pred p;\n\t.reg .b32 t, sa, g0, g, gk, ar, aa;\n\t"              \
    "ld.volatile.shared.u32 sa, [%1+32];\n\t"                                    \
    "ld.volatile.shared.u32 t, [%1];\n\t" HIST_LINE                              \
    SHIFT_OP " g0, %7, %8;\n\t"                                                  \
    "and.b32 g, g0, 0x1C;\n\t"                                                   \
    "add.u32 ar, %0, g;\n\t"                                                     \
    "add.u32 gk, g, %10;\n\t"                                                    \
    "add.u32 aa, sa, gk;\n\t"                                                    \
    "mad.lo.u32 %4, aa, ar, %4;\n\t"                                             \
    "setp.le.u32 p, %6, t;\n\t"                                                  \
    "selp.u32 %1, aa, ar, p;\n\t"                                                \
    "selp.u32 %0, sa, %0, p;\n\t"                                                \
    "@p or.b32 %2, %2, %9;\n\t" EXTRA_LINE "}"
#elif MUCA_SITE_VARIANT == 7   // Sa = S + DT[A - S]: a conflict-free load behind the table load; the offset A - S is selected like A
#define MUCA_V6_SITE(SHIFT_OP, HIST_LINE, EXTRA_LINE)                            \
    "{\n\t.reg .pred p;\n\t.reg .b32 t, d, sa, g0, g, gk, ar, aa, sg;\n\t"       \
    "ld.volatile.shared.u32 t, [%1];\n\t"                                        \
    "ld.volatile.shared.u32 d, [%5+%12];\n\t" HIST_LINE                          \
    SHIFT_OP " g0, %7, %8;\n\t"                                                  \
    "and.b32 g, g0, 0x1C;\n\t"                                                   \
    "add.u32 ar, %0, g;\n\t"                                                     \
    "add.u32 gk, g, %10;\n\t"                                                    \
    "add.u32 sg, %0, gk;\n\t"                                                    \
    "add.u32 aa, sg, d;\n\t"                                                     \
    "add.u32 sa, %0, d;\n\t"                                                     \
    "mad.lo.u32 %4, aa, ar, %4;\n\t"                                             \
    "setp.le.u32 p, %6, t;\n\t"                                                  \
    "selp.u32 %1, aa, ar, p;\n\t"                                                \
    "selp.u32 %5, gk, g, p;\n\t"                                                 \
    "selp.u32 %0, sa, %0, p;\n\t"                                                \
    "@p or.b32 %2, %2, %9;\n\t" EXTRA_LINE "}"
#endif
#ifdef MUCA_V6_DT
#define MUCA_V6_HIST "red.shared.add.u32 [%0+32], 1;\n\t"
#else
#define MUCA_V6_HIST "red.shared.add.u32 [%0+64], 1;\n\t"
#endif

template <int L, bool MEAS, int KK>
__device__ __forceinline__ void site_v6(uint32_t& S, uint32_t& A, uint32_t& flips, uint32_t& fw3, uint32_t& chk, uint32_t& off, const uint32_t rnd,
                                        const uint32_t fwn, const int qn, const uint32_t mask, const uint32_t patch,
                                        const bool first) {
    const uint32_t sh = qn == 0 ? 2u : (uint32_t)(4 * qn - 2);   // nibble qn of the field word -> bits 2..4
    uint32_t unused = 0;   // fills operand %3 of the site macro where site 0 has FW[3]
#ifdef MUCA_V6_DT
    constexpr uint32_t DTA = V6<L>::SBASE + V6<L>::DT_OFF;
#else
    constexpr uint32_t DTA = 0;
#endif
    if (first) {   // site 0 also patches the last site's column: its right neighbour is site 0
        if (MEAS)
            asm volatile(MUCA_V6_SITE("shl.b32", MUCA_V6_HIST, "@p add.u32 %3, %3, %11;\n\t")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(fw3), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(patch), "n"(DTA) : "memory");
        else
            asm volatile(MUCA_V6_SITE("shl.b32", "", "@p add.u32 %3, %3, %11;\n\t")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(fw3), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(patch), "n"(DTA) : "memory");
    } else if (qn == 0) {
        if (MEAS)
            asm volatile(MUCA_V6_SITE("shl.b32", MUCA_V6_HIST, "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(0), "n"(DTA) : "memory");
        else
            asm volatile(MUCA_V6_SITE("shl.b32", "", "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(0), "n"(DTA) : "memory");
    } else {
        if (MEAS)
            asm volatile(MUCA_V6_SITE("shr.u32", MUCA_V6_HIST, "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(0), "n"(DTA) : "memory");
        else
            asm volatile(MUCA_V6_SITE("shr.u32", "", "")
                         : "+r"(S), "+r"(A), "+r"(flips), "+r"(unused), "+r"(chk), "+r"(off)
                         : "r"(rnd), "r"(fwn), "r"(sh), "r"(mask), "n"(KK), "r"(0), "n"(DTA) : "memory");
    }
}

// One row of the walker warp.  In: the row above (`up`, final), this row's old value `c`, its finished field words FW,
// its deviates rnd[] and the entry address A of site 0.  While the row is processed, the row below is prepared in `n`
// (old value, partial planes), its field words FWn are finished and its deviates replace this row's in rnd[] (call k
// after site 4k + 3).  Out: `up` = this row's new value, A = entry address of site 0 of the row below.
// Every site increments the bin of the state it STARTS from, i.e. of the state after the previous attempt.
template <int L, bool MEAS>
__device__ __forceinline__ void row_v6(uint32_t* __restrict__ lat, uint32_t& S, uint32_t& A, uint32_t& chk, uint32_t& off, const int y, const bool more,
                                       uint32_t& up, const uint32_t c, uint32_t (&FW)[4], const uint32_t patch,
                                       uint32_t (&rnd)[Geo<L>::BITS], NextRow<L>& n, uint32_t (&FWn)[4],
                                       const uint4* __restrict__ ring, int& buf, const int bar_id) {
    using G = Geo<L>;
    using V = V6<L>;
    constexpr int BITS = G::BITS, NC = V::NC, SLOTS = V::SLOTS;
    // the deviates of row y + 1 are in ring[buf]; ring[buf ^ 1] (this row's, all fetched) may be refilled.  After the
    // last row of a phase there is no such barrier (the deviate warp has left its loop) and what is fetched is not used.
    if (more) pair_barrier(bar_id);
    const int y1 = (y + 1) & (L - 1), y2 = (y + 2) & (L - 1);
    n.c = lat[y1 * SLOTS];
    n.dn = lat[y2 * SLOTS];   // row y + 2 is old (or row 0, final in this sweep, when y + 1 = L - 1)
    uint32_t flips = 0;
#pragma unroll
    for (int x = 0; x < BITS; ++x) {
        const int xn = x + 1;
        if (xn < BITS)
            site_v6<L, MEAS, (int)V::K>(S, A, flips, FW[3], chk, off, rnd[x], FW[xn & 3], xn >> 2, 1u << x, patch, x == 0);
        else   // next site: site 0 of the row below, no carry
            site_v6<L, MEAS, 0>(S, A, flips, FW[3], chk, off, rnd[x], FWn[0], 0, 1u << x, patch, false);
        // ---- off the chain, in the shadow of the table loads: prepare the row below
        prep_for_site<L>(n, x);
        if (x >= BITS - 4 && x < BITS - 1) FWn[x - (BITS - 4)] = finish_word<L>(n, c ^ flips, x - (BITS - 4));
        if ((x & 3) == 3 && more) {   // the deviates of sites 4k .. 4k + 3 are spent: fetch call k of the row below into their place
            const int k = x >> 2;
            const uint4 v = ring[(buf * NC + k) * SLOTS];
            rnd[4 * k] = v.x; rnd[4 * k + 1] = v.y; rnd[4 * k + 2] = v.z; rnd[4 * k + 3] = v.w;
        }
    }
    buf ^= (int)more;
    up = c ^ flips;
    lat[y * SLOTS] = up;
    FWn[3] = finish_word<L>(n, up, 3);
}

// Walker warp: sweeps s0 .. s1-1; `buf` is the ring buffer holding the deviates of the next row to fetch.  Rows are
// processed in pairs so that the two register sets (this row / row below) swap roles without copies.
// The caller compensates the first and the last attempt of the measured phase in the histogram (see row_v6).
template <int L, bool MEAS>
__device__ __forceinline__ void sweeps_v6(uint32_t* __restrict__ lat, uint32_t& S, uint32_t& chk, const uint32_t s0, const uint32_t s1,
                                          const uint4* __restrict__ ring, int& buf, const int bar_id) {
    using G = Geo<L>;
    using V = V6<L>;
    constexpr int BITS = G::BITS, NC = V::NC, SLOTS = V::SLOTS;
    if (s1 <= s0) return;
    uint32_t up = lat[(L - 1) * SLOTS];
    NextRow<L> nA, nB;
    uint32_t FWA[4], FWB[4], rnd[BITS];
    nA.c = lat[0];
    nA.dn = lat[SLOTS];
    prep_steps<L, 0, PREP_STEPS>(nA);
#pragma unroll
    for (int r = 0; r < 4; ++r) FWA[r] = finish_word<L>(nA, up, r);
    pair_barrier(bar_id);                      // the deviates of the first row are in ring[buf]
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const uint4 v = ring[(buf * NC + k) * SLOTS];
        rnd[4 * k] = v.x; rnd[4 * k + 1] = v.y; rnd[4 * k + 2] = v.z; rnd[4 * k + 3] = v.w;
    }
    buf ^= 1;
    uint32_t off = (FWA[0] << 2) & 0x1Cu;      // site 0: its left neighbour (site L-1) has not been visited in this sweep
    uint32_t A = S + off;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; y += 2) {
            row_v6<L, MEAS>(lat, S, A, chk, off, y, true, up, nA.c, FWA, nA.patch, rnd, nB, FWB, ring, buf, bar_id);
            row_v6<L, MEAS>(lat, S, A, chk, off, y + 1, s + 1 < s1 || y + 2 < L, up, nB.c, FWB, nB.patch, rnd, nA, FWA, ring, buf, bar_id);
        }
    }
}

// Deviate warp: the NC Philox calls of one row advance round-major (NC independent IMAD.WIDE chains), results go to
// the double-buffered shared ring rnd[buf][call][slot] as one 16-byte store per call.  One barrier per row hands
// the buffer over.  R4: ctr = (i >> 2, sweep, iteration, walker).
template <int L>
__device__ __forceinline__ void deviates_v6(uint4* __restrict__ ring, const uint32_t s0, const uint32_t s1, int& buf,
                                            const int bar_id, const SweepParams& prm, const uint32_t walker, const bool active) {
    constexpr int NC = V6<L>::NC, SLOTS = V6<L>::SLOTS;
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
            for (int k = 0; k < NC; ++k)
                if (active) ring[(buf * NC + k) * SLOTS] = make_uint4(st[k][0], st[k][1], st[k][2], st[k][3]);
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
__global__ void __launch_bounds__(64 * V6<L>::MAX_WARPS, 1) sweep_kernel_v6(const SweepParams prm, const int wpw, const int role_map) {
    using G = Geo<L>;
    using V = V6<L>;
    constexpr int N = G::N, BINS = G::BINS, SLOTS = V::SLOTS;
    extern __shared__ __align__(16) uint32_t smem[];
    char* const sm = reinterpret_cast<char*>(smem);
    const int tid = threadIdx.x, nthr = blockDim.x, nw = nthr >> 6;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
#ifdef MUCA_V6_DT
    if (sbase != V::SBASE) __trap();   // the site macro addresses the delta table by an immediate

    // ---- both table copies: row (j, c) = t[8] | bin; delta tables behind the rows
    for (int idx = tid; idx < BINS * 16; idx += nthr) {
        const int j = idx >> 4, cc = (idx >> 3) & 1, f = idx & 7;
        const int fe = f ^ cc, a = (fe >> 1) + (fe & 1);
        const int jn = j + 2 - a;                            // where an accepted move leads (dE = 8 - 4a)
        // R17: a move out of [0, N] cannot occur for a real configuration; its entry is never consulted
        *reinterpret_cast<uint32_t*>(sm + (size_t)cc * V::K + (size_t)j * V::RS + 4 * f) = (jn < 0 || jn > N) ? 0u : prm.table[j * 8 + fe];
    }
    for (int j = tid; j <= BINS; j += nthr) *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF) = 0u;
    if (tid < 16) {   // row BINS of both copies: t = 0 in every column; the lanes parked here get deviates 0xFFFFFFFF and stay
        const int cc = tid >> 3, f = tid & 7, fe = f ^ cc, a = (fe >> 1) + (fe & 1);
        *reinterpret_cast<uint32_t*>(sm + (size_t)cc * V::K + (size_t)BINS * V::RS + 4 * f) = 0u;
        *reinterpret_cast<int32_t*>(sm + (size_t)cc * V::K + V::DT_OFF + 4 * f) = (int)V::RS * (2 - a);
    }
#else
    // copy 0, the lattices and the ring must end below K (dynamic shared memory starts behind the 1 KB the system
    // reserves on sm_100)
    if (sbase + V::RING_OFF + V::RING_BYTES > V::K) __trap();

    // ---- both table copies: row (j, c) = t[8] | Sa[8] | bin
    for (int idx = tid; idx < BINS * 16; idx += nthr) {
        const int j = idx >> 4, cc = (idx >> 3) & 1, f = idx & 7;
        const int fe = f ^ cc, a = (fe >> 1) + (fe & 1);
        int jn = j + 2 - a;                                  // where an accepted move leads (dE = 8 - 4a)
        uint32_t t = prm.table[j * 8 + fe];
        if (jn < 0 || jn > N) { jn = j; t = 0u; }            // R17: cannot occur for a real configuration
        char* const row = sm + (size_t)cc * V::K + (size_t)j * V::RS;
        *reinterpret_cast<uint32_t*>(row + 4 * f) = t;
        *reinterpret_cast<uint32_t*>(row + V::SA_OFF + 4 * f) = sbase + (uint32_t)jn * V::RS;
    }
    for (int idx = tid; idx < BINS * 2; idx += nthr)
        *reinterpret_cast<uint32_t*>(sm + (size_t)(idx & 1) * V::K + (size_t)(idx >> 1) * V::RS + V::BIN_OFF) = 0u;
    if (tid < 34) {  // row BINS of both copies: t = 0 and Sa = itself in every column -- a lane parked here stays here
        const int cc = tid / 17, e = tid % 17;
        *reinterpret_cast<uint32_t*>(sm + (size_t)cc * V::K + (size_t)BINS * V::RS + 4 * e) = e >= 8 && e < 16 ? sbase + BINS * V::RS : 0u;
    }
#endif

    // warp -> role.  A warp runs on scheduler (warp id % 4).  role_map 0 (4 pairs per block): the walker warps take
    // warp ids {0, 1, 4, 5} and the deviate warps {2, 3, 6, 7}: two walker warps share a scheduler and two deviate warps
    // share one.  role_map 1: deviate warps 0 .. 3, walker warps 4 .. 7 -- every scheduler runs one walker warp and one
    // deviate warp (the walker has the higher warp id).  With 1 or 2 pairs every warp has a scheduler of its own
    // (deviate ids 0 .. nw-1, walker ids nw .. 2nw-1).
    const int warp_id = tid >> 5;
    const bool split = nw == 4 && role_map == 0;
    const bool is_walker = split ? (warp_id & 2) == 0 : warp_id >= nw;
    const int pair = split ? (warp_id & 1) | ((warp_id >> 2) << 1) : (is_walker ? warp_id - nw : warp_id);
    const int lane = tid & 31, slot = 32 * pair + lane;          // slot: lattice / ring column
    const int w = (blockIdx.x * nw + pair) * wpw + lane;
    const bool active = lane < wpw && w < prm.W;
    const int bar_id = 1 + pair;
    uint32_t* const lat = reinterpret_cast<uint32_t*>(sm + V::LAT_OFF) + slot;
    uint4* const ring = reinterpret_cast<uint4*>(sm + V::RING_OFF);
    // a lane without a walker never accepts: its ring slots hold the deviate 0xFFFFFFFF for good (the deviate warp
    // stores only for lanes with a walker) and its row has all thresholds 0
    if (!is_walker && !active)
        for (int k = 0; k < 2 * V::NC; ++k) ring[k * SLOTS + slot] = make_uint4(0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu);

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
    // slot j = (E + 2N)/4
    uint32_t S = sbase + (is_walker && active ? (uint32_t)((prm.E[w] + 2 * N) >> 2) : (uint32_t)BINS) * V::RS;
    int buf = 0;
    uint32_t chk = 0;
    // ---- thermalisation sweeps: nothing is recorded
    if (is_walker) sweeps_v6<L, false>(lat, S, chk, prm.sweep_begin, s_th, ring + slot, buf, bar_id);
    else deviates_v6<L>(ring + slot, prm.sweep_begin, s_th, buf, bar_id, prm, walker, active);
    // ---- measured sweeps: every site counts the state it starts from, so the state before the first measured
    //      attempt is taken out again here and the state after the last one is added below
    if (is_walker) {
        if (s_th < prm.sweep_end) atomicSub(reinterpret_cast<uint32_t*>(sm + (S - sbase) + V::BIN_OFF), 1u);
        sweeps_v6<L, true>(lat, S, chk, s_th, prm.sweep_end, ring + slot, buf, bar_id);
        if (s_th < prm.sweep_end) atomicAdd(reinterpret_cast<uint32_t*>(sm + (S - sbase) + V::BIN_OFF), 1u);
    } else {
        deviates_v6<L>(ring + slot, s_th, prm.sweep_end, buf, bar_id, prm, walker, active);
    }
    if (is_walker) {
        if (chk == 0x9E3779B9u && !active) lat[0] = chk;   // keeps the checksum of the site macro alive (never true for a parked lane: its addresses are constant)
        if (active) {
            prm.E[w] = (int)((S - sbase) / V::RS) * 4 - 2 * N;
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

    // ---- a4: merge the block's bins into the global uint64 histogram (the parking row BINS is not a slot)
    if (prm.sweep_end > prm.therm) {
        for (int j = tid; j < BINS; j += nthr) {
            const uint32_t v = *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF);
            if (v) atomicAdd(prm.H + j, (unsigned long long)v);
        }
    }
}

}  // namespace muca
