// paper_1707_00919_b200/csrc/muca_resident.cuh
// Resident sweep kernel v6 for L <= 32 (sm_100a): "state in the address", two-candidate select, walker warps paired
// with deviate warps, everything that is not the per-site chain spread over the sites of the previous row; the site
// macro in its PIPELINED form (the table load of the next site closes the macro, round 2).
// Citations: "PAPER.md:<line>" = /root/reference/PAPER.md, "R<n>" = DESIGN.md section 3.
//
// The walker's dynamic state is the shared-memory address S = rowaddr(j) of its energy slot j.  Row j is 36 bytes (9
// words: consecutive rows rotate through all 32 banks):
//     +4f      t = thresh[j][a(f)],  f = hl + 2*n3 the column of the site: n3 antiparallel bonds to up / down / right,
//              hl = [left neighbour != s]                                  (PAPER.md:109 acceptance, R6/R7)
//     +32      histogram bin of slot j
// and behind the rows the delta table DT[f] = RS * (2 - a(f)): an accepted move leads to S + DT[f].  The carry
// c = [previous site of this row flipped] toggles the hl bit of the column, f -> f ^ 1; it lives in the ENTRY address
// A = S + 4 (f ^ c) of the lookup, never in S.
// Per site the serial chain is   LDS t -> ISETP -> SEL(A_acc, A_rej) -> LDS t'   with BOTH candidates of the next
// entry address, A_acc = S + DT[f ^ c] + 4 (f' ^ 1) and A_rej = S + 4 f', formed before the decision (round 1, v5,
// selected the state and added the column afterwards, ISETP -> SEL -> IADD -> LDS, kept two copies of the table for
// the two values of the carry and loaded the next state from the row: a second load with ~3.3 bank-conflict
// wavefronts).  Philox runs in a paired "deviate" warp (same walkers) that feeds a double-buffered shared ring one
// row ahead.
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

template <int L>
struct V6 {
    static constexpr uint32_t SBASE = 1024;                  // dynamic shared memory starts behind the 1 KB the system reserves on sm_100 (checked)
    static constexpr uint32_t BINS = L * L + 1;
    static constexpr uint32_t RS = 36, BIN_OFF = 32;         // row j: t[8] | bin
    static constexpr uint32_t DT_OFF = (BINS + 1) * RS;      // + one all-reject row: parking place of unused lanes
    static constexpr uint32_t LAT_OFF = (DT_OFF + 32u + 15u) & ~15u;
    static constexpr int MAX_WARPS = 4;                      // walker warps per block (+ as many deviate warps)
    static constexpr int SLOTS = 32 * MAX_WARPS;             // lattice / ring columns
    static constexpr int NC = Geo<L>::BITS / 4;              // Philox calls per row
    static constexpr uint32_t RING_OFF = LAT_OFF + (uint32_t)L * 4u * SLOTS;
    static constexpr uint32_t RING_BYTES = 2u * NC * 16u * SLOTS;
    static constexpr uint32_t SCRATCH_OFF = RING_OFF + RING_BYTES;          // 16 bytes per call and deviate warp (philox_unit)
    static constexpr uint32_t TAG_OFF = SCRATCH_OFF + 16u * NC * MAX_WARPS;   // MUCA_CHECKED build: 2 x MAX_WARPS hand-over tags
    static constexpr size_t SMEM_BYTES = (size_t)TAG_OFF + 8u * MAX_WARPS;
};

// Field words of a row: nibble q of FW[r] holds the column f = hl + 2*n3 of site 4q + r (hl: bond to the left
// neighbour's OLD value, n3 = antiparallel bonds to up / down / right).  They are built in two parts so that most of
// the work can be done a row ahead: the planes that do not depend on the row ABOVE (which the walker is still
// updating) go into P[r] = hl + 2*(vd + hr), one small step per site of the row before (prep_step), and
// FW[r] = P[r] + 2*vu is finished when the sites 4q + r of the row above are final (finish_word).
template <int L>
struct NextRow {
    uint32_t c, dn;            // the row (old value) and the row below it (old; row 0, already final, below row L-1)
    uint32_t left, right;      // L >= 64: the words of the same row to the left / right of c (old values, periodic)
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
        const uint32_t rw = G::WPR > 1 ? __funnelshift_r(n.c, n.right, 1)
                            : L >= 32 ? __funnelshift_r(n.c, n.c, 1) : ((n.c >> 1) | ((n.c & 1u) << (BITS - 1)));
        n.hr = n.c ^ rw;
    } else if constexpr (I == 1) {
        const uint32_t lw = G::WPR > 1 ? __funnelshift_l(n.left, n.c, 1)
                            : L >= 32 ? __funnelshift_l(n.c, n.c, 1) : (((n.c << 1) | (n.c >> (BITS - 1))) & G::MASK);
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
// the value written by preparation step I (scheduling dependency of the pipelined site macro)
template <int L, int I>
__device__ __forceinline__ uint32_t prep_last(const NextRow<L>& n) {
    if constexpr (I == 0) return n.hr;
    else if constexpr (I == 1) return n.hl;
    else if constexpr (I == 2) return n.m0;
    else if constexpr (I == 3) return n.m1;
    else if constexpr (I < 16) return ((I - 4) % 3 == 2) ? n.P[(I - 4) / 3] : n.t;
    else return n.patch;
}
// FW[r] of the row below `above_new` (bits 4q + r of above_new must be final)
template <int L>
__device__ __forceinline__ uint32_t finish_word(const NextRow<L>& n, const uint32_t above_new, const int r) {
    constexpr uint32_t M = Geo<L>::BITS == 32 ? 0x11111111u : (Geo<L>::BITS == 16 ? 0x1111u : 0x11u);
    return n.P[r] + 2u * (((n.c ^ above_new) >> r) & M);
}

// One site of the walker chain, in PTX.  Operands:
//   %0 S: state address (in/out)      %1 A: entry address of this site (in), of the next site (out)
//   %2 flips (in/out)                 %3 FW[3] at site 0 (in/out)          %4 checksum (in/out, see below)
//   %5 off = A - S = 4 (f ^ c): offset into the delta table (in: this site, out: next site)
//   %6 g1 = 4f of the NEXT site (in), of the site after it (out)           %7 gx1 = g1 ^ 4 (same; g1 where a row starts)
//   %8 deviate   %9 field word of the site AFTER the next   %10 its shift   %11 flip mask of this site
//   %12 the constant 4 in a register   %13 patch (site 0)   %14 address of DT[0]
// What ptxas does not do by itself (profiles/README.md, round 2; SASS checked with cuobjdump):
//  * the decision must be consumed by SELs: ISETP -> SEL -> LDS costs ~9 cycles, ISETP -> predicated instruction ->
//    LDS about 20.  ptxas turns "A = p ? aa : ar" into "A = aa; @!p A = S + g" unless BOTH candidates have a second,
//    unconditional use: the multiply-add into the checksum %4 (FMA pipe, idle in a walker warp; the checksum is kept
//    alive by a store that never executes).  The state itself may be a predicated add: it is off the chain.
//  * the table load is issued in front of the (conflict-free, one-wavefront) delta load: volatile loads keep their order.
// The column of the site after the next is extracted here, a site early, so that both candidates can be formed as soon
// as the delta arrives.  H[j]++ of the PREVIOUS attempt is issued behind this site's loads (S still holds that state);
// thermalisation sweeps leave it out.  The flip mask is a predicated OR.
#define MUCA_V6_SITE(SHIFT_OP, HIST_LINE, GX_LINE, EXTRA_LINE)                   \
    "{\n\t.reg .pred p;\n\t.reg .b32 t, d, sa, gs, g2, gx2, ar, aa, sg;\n\t"     \
    "ld.volatile.shared.u32 t, [%1];\n\t"                                        \
    "ld.volatile.shared.u32 d, [%5+%14];\n\t" HIST_LINE                          \
    SHIFT_OP " gs, %9, %10;\n\t"                                                 \
    "add.u32 ar, %0, %6;\n\t"                                                    \
    "add.u32 sg, %0, %7;\n\t"                                                    \
    "and.b32 g2, gs, 0x1C;\n\t" GX_LINE                                          \
    "add.u32 aa, sg, d;\n\t"                                                     \
    "add.u32 sa, %0, d;\n\t"                                                     \
    "mad.lo.u32 %4, aa, ar, %4;\n\t"                                             \
    "setp.le.u32 p, %8, t;\n\t"                                                  \
    "selp.u32 %1, aa, ar, p;\n\t"                                                \
    "selp.u32 %5, %7, %6, p;\n\t"                                                \
    "selp.u32 %0, sa, %0, p;\n\t"                                                \
    "@p or.b32 %2, %2, %11;\n\t" EXTRA_LINE                                      \
    "mov.u32 %6, g2;\n\tmov.u32 %7, gx2;\n\t}"
#define MUCA_V6_HIST "red.shared.add.u32 [%0+32], 1;\n\t"
#define MUCA_V6_GX_CARRY "lop3.b32 gx2, gs, 0x1C, %12, 0x6A;\n\t"   /* (gs & 0x1C) ^ 4: the column if this site's left neighbour has flipped */
#define MUCA_V6_GX_ROWSTART "mov.u32 gx2, g2;\n\t"                  /* site 0 of a row: its left neighbour has not been visited in this sweep */
#define MUCA_V6_PATCH "@p add.u32 %3, %3, %13;\n\t"

// The PIPELINED form of the site (resident kernel; profiles/README.md, round 2).  Threshold t and delta d of THIS site
// were loaded by the previous macro (operands %8, %9); this one decides, selects and at once issues the loads of the
// NEXT site, directly behind the two selects:
//     ISETP -> SEL A' -> LDS t'         is all that is left between two table loads of the chain.
// In the form above the new state was "selp S, S + d, S", which ptxas turns into an add predicated on the decision; a
// predicate is consumed by a predicated instruction ~13 cycles after its ISETP, the warp issues in order, and the
// next table load sat behind it.  Here S' = A' - off' (both selected, no predicate), H[j]++ counts the state after
// the attempt where it is known, and the column extraction is a funnel shift whose other half (%16, shifted out of
// the bits kept by the mask) is the last value written by the preparation steps scheduled at this site: without
// that dependency ptxas sinks the ~35 preparation instructions of a row to its end, where no table load hides them.
//   %0 S  %1 A  %2 flips  %3 FW[3] (site 0)  %4 checksum  %5 off  %6 g1  %7 gx1  %8 t  %9 d       (all in/out)
//   %10 deviate  %11 field word of the site after the next  %12 its shift  %13 flip mask  %14 the constant 4
//   %15 patch  %16 scheduling dependency  %17 address of DT[0]
#define MUCA_V6P_SITE(SHIFT_LINE, HIST_LINE, GX_LINE, EXTRA_LINE)                \
    "{\n\t.reg .pred p;\n\t.reg .b32 gs, g2, gx2, ar, aa, sg;\n\t"               \
    SHIFT_LINE                                                                   \
    "add.u32 ar, %0, %6;\n\t"                                                    \
    "add.u32 sg, %0, %7;\n\t"                                                    \
    "and.b32 g2, gs, 0x1C;\n\t" GX_LINE                                          \
    "add.u32 aa, sg, %9;\n\t"                                                    \
    "mad.lo.u32 %4, aa, ar, %4;\n\t"                                             \
    "setp.le.u32 p, %10, %8;\n\t"                                                \
    "selp.u32 %1, aa, ar, p;\n\t"                                                \
    "selp.u32 %5, %7, %6, p;\n\t"                                                \
    "ld.volatile.shared.u32 %8, [%1];\n\t"                                       \
    "ld.volatile.shared.u32 %9, [%5+%17];\n\t"                                   \
    "sub.u32 %0, %1, %5;\n\t"                                                    \
    HIST_LINE                                                                    \
    "@p or.b32 %2, %2, %13;\n\t" EXTRA_LINE                                      \
    "mov.u32 %6, g2;\n\tmov.u32 %7, gx2;\n\t}"
#define MUCA_V6P_SHL "shf.l.clamp.b32 gs, %16, %11, %12;\n\t"       /* (fw << s) | (dep >> (32 - s)): s = 2, the mask keeps bits 2..4 */
#define MUCA_V6P_SHR "shf.r.clamp.b32 gs, %11, %16, %12;\n\t"       /* (fw >> s) | (dep << (32 - s)): s <= 26 */
#define MUCA_V6P_GX_CARRY "lop3.b32 gx2, gs, 0x1C, %14, 0x6A;\n\t"
#define MUCA_V6P_PATCH "@p add.u32 %3, %3, %15;\n\t"

// threshold and delta of the next site (pipelined form) and the scheduling dependency of its macro
struct SitePipe { uint32_t t, d, dep; };

enum { SITE_FIRST = 0, SITE_SHL = 1, SITE_SHR = 2, SITE_ROWSTART = 3 };   // flavour of the site macro

template <int L, bool MEAS, int FLAVOUR, uint32_t DTA, bool PIPE>
__device__ __forceinline__ void site_v6(uint32_t& S, uint32_t& A, uint32_t& flips, uint32_t& fw3, uint32_t& chk, uint32_t& off,
                                        uint32_t& g1, uint32_t& gx1, const uint32_t rnd, const uint32_t fw2, const uint32_t sh2,
                                        const uint32_t mask, const uint32_t patch, SitePipe& pp) {
    uint32_t unused = 0;   // fills operand %3 of the site macro where site 0 has FW[3]
    if constexpr (PIPE) {
#define MUCA_V6P_ASM(SHIFT, HIST, GX, EXTRA, FW3)                                                                      \
    asm volatile(MUCA_V6P_SITE(SHIFT, HIST, GX, EXTRA)                                                                 \
                 : "+r"(S), "+r"(A), "+r"(flips), "+r"(FW3), "+r"(chk), "+r"(off), "+r"(g1), "+r"(gx1), "+r"(pp.t), "+r"(pp.d) \
                 : "r"(rnd), "r"(fw2), "r"(sh2), "r"(mask), "r"(4u), "r"(patch), "r"(pp.dep), "n"(DTA) : "memory")
        if constexpr (FLAVOUR == SITE_FIRST) {
            if constexpr (MEAS) MUCA_V6P_ASM(MUCA_V6P_SHL, MUCA_V6_HIST, MUCA_V6P_GX_CARRY, MUCA_V6P_PATCH, fw3);
            else MUCA_V6P_ASM(MUCA_V6P_SHL, "", MUCA_V6P_GX_CARRY, MUCA_V6P_PATCH, fw3);
        } else if constexpr (FLAVOUR == SITE_SHL) {
            if constexpr (MEAS) MUCA_V6P_ASM(MUCA_V6P_SHL, MUCA_V6_HIST, MUCA_V6P_GX_CARRY, "", unused);
            else MUCA_V6P_ASM(MUCA_V6P_SHL, "", MUCA_V6P_GX_CARRY, "", unused);
        } else if constexpr (FLAVOUR == SITE_SHR) {
            if constexpr (MEAS) MUCA_V6P_ASM(MUCA_V6P_SHR, MUCA_V6_HIST, MUCA_V6P_GX_CARRY, "", unused);
            else MUCA_V6P_ASM(MUCA_V6P_SHR, "", MUCA_V6P_GX_CARRY, "", unused);
        } else {
            if constexpr (MEAS) MUCA_V6P_ASM(MUCA_V6P_SHL, MUCA_V6_HIST, MUCA_V6_GX_ROWSTART, "", unused);
            else MUCA_V6P_ASM(MUCA_V6P_SHL, "", MUCA_V6_GX_ROWSTART, "", unused);
        }
#undef MUCA_V6P_ASM
        return;
    }
#define MUCA_V6_ASM(SHIFT_OP, HIST, GX, EXTRA, FW3)                                                                    \
    asm volatile(MUCA_V6_SITE(SHIFT_OP, HIST, GX, EXTRA)                                                               \
                 : "+r"(S), "+r"(A), "+r"(flips), "+r"(FW3), "+r"(chk), "+r"(off), "+r"(g1), "+r"(gx1)                 \
                 : "r"(rnd), "r"(fw2), "r"(sh2), "r"(mask), "r"(4u), "r"(patch), "n"(DTA) : "memory")
    if constexpr (FLAVOUR == SITE_FIRST) {   // site 0 also patches the last site's column: its right neighbour is site 0
        if constexpr (MEAS) MUCA_V6_ASM("shl.b32", MUCA_V6_HIST, MUCA_V6_GX_CARRY, MUCA_V6_PATCH, fw3);
        else MUCA_V6_ASM("shl.b32", "", MUCA_V6_GX_CARRY, MUCA_V6_PATCH, fw3);
    } else if constexpr (FLAVOUR == SITE_SHL) {
        if constexpr (MEAS) MUCA_V6_ASM("shl.b32", MUCA_V6_HIST, MUCA_V6_GX_CARRY, "", unused);
        else MUCA_V6_ASM("shl.b32", "", MUCA_V6_GX_CARRY, "", unused);
    } else if constexpr (FLAVOUR == SITE_SHR) {
        if constexpr (MEAS) MUCA_V6_ASM("shr.u32", MUCA_V6_HIST, MUCA_V6_GX_CARRY, "", unused);
        else MUCA_V6_ASM("shr.u32", "", MUCA_V6_GX_CARRY, "", unused);
    } else {
        if constexpr (MEAS) MUCA_V6_ASM("shl.b32", MUCA_V6_HIST, MUCA_V6_GX_ROWSTART, "", unused);
        else MUCA_V6_ASM("shl.b32", "", MUCA_V6_GX_ROWSTART, "", unused);
    }
#undef MUCA_V6_ASM
}

// The deviate ring is written by another warp between two pair barriers: its pointers are NOT __restrict__ (with
// __restrict__ the compiler reused the values of an earlier load of the same ring slot across the barrier).
// Site X of a 32-site unit (a row for L <= 32, one word of a row for L >= 64); compile-time recursion: flavour, shifts
// and masks are constants.  FIRST / LASTW: the unit is the first / last one of its lattice row.  FW: the unit's
// field words; fw3t: FW[3] of the LAST unit of the row (site 0 of the row patches it); FWseq: the field words of the
// next unit in typewriter order (the columns of its sites 0 and 1 are extracted at the end of this unit); (n, FWp):
// the unit one lattice row below, prepared here.  DTA: address of the delta table; stride: uint4 elements between two
// calls in the ring.
template <int L, bool MEAS, int X, bool FIRST, bool LASTW, uint32_t DTA, bool PIPE>
struct RowSites {
    static __device__ __forceinline__ void run(uint32_t& S, uint32_t& A, uint32_t& flips, uint32_t& chk, uint32_t& off, uint32_t& g1,
                                               uint32_t& gx1, const uint32_t c, uint32_t (&FW)[4], uint32_t& fw3t, const uint32_t patch,
                                               uint32_t (&rnd)[Geo<L>::BITS], NextRow<L>& n, uint32_t (&FWp)[4],
                                               const uint32_t (&FWseq)[4], const uint4* ring, const int stride,
                                               const int buf, const bool more, SitePipe& pp) {
        constexpr int BITS = Geo<L>::BITS, NC = BITS / 4;
        constexpr int X2 = X + 2;                              // the site whose column is extracted now
        constexpr bool below = X2 >= BITS;                     // it belongs to the next unit
        constexpr int q2 = below ? 0 : X2 >> 2;
        constexpr uint32_t sh2 = q2 == 0 ? 2u : (uint32_t)(4 * q2 - 2);   // nibble q2 of the field word -> bits 2..4
        constexpr int FLAVOUR = (X == 0 && FIRST) ? SITE_FIRST : ((X2 == BITS && LASTW) ? SITE_ROWSTART : (q2 == 0 ? SITE_SHL : SITE_SHR));
        site_v6<L, MEAS, FLAVOUR, DTA, PIPE>(S, A, flips, fw3t, chk, off, g1, gx1, rnd[X], below ? FWseq[X2 - BITS] : FW[X2 & 3], sh2,
                                             1u << X, patch, pp);
        // ---- off the chain, in the shadow of the table loads: prepare the unit below
        constexpr int D = BITS - 4;
        if constexpr (X < D) {
            constexpr int I0 = (X * PREP_STEPS) / D, I1 = ((X + 1) * PREP_STEPS) / D;
            prep_steps<L, I0, I1>(n);
            if constexpr (PIPE && I1 > I0) pp.dep = prep_last<L, I1 - 1>(n);   // pins these steps in front of the next site
        }
        if constexpr (X >= BITS - 4 && X < BITS - 1) FWp[X - (BITS - 4)] = finish_word<L>(n, c ^ flips, X - (BITS - 4));
        if constexpr ((X & 3) == 3) {
            if (more) {   // the deviates of sites 4k .. 4k + 3 are spent: fetch call k of the next unit into their place
                constexpr int k = X >> 2;
                if constexpr (PIPE) {   // volatile: stays between the table loads of this site and of the next one
                    asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(rnd[4 * k]), "=r"(rnd[4 * k + 1]), "=r"(rnd[4 * k + 2]), "=r"(rnd[4 * k + 3])
                                 : "r"((uint32_t)__cvta_generic_to_shared(ring + (buf * NC + k) * stride)) : "memory");
                } else {
                    const uint4 v = ring[(buf * NC + k) * stride];
                    rnd[4 * k] = v.x; rnd[4 * k + 1] = v.y; rnd[4 * k + 2] = v.z; rnd[4 * k + 3] = v.w;
                }
            }
        }
        if constexpr (X + 1 < BITS)
            RowSites<L, MEAS, X + 1, FIRST, LASTW, DTA, PIPE>::run(S, A, flips, chk, off, g1, gx1, c, FW, fw3t, patch, rnd, n, FWp, FWseq,
                                                                  ring, stride, buf, more, pp);
    }
};

// One row of the walker warp.  In: the row above (`up`, final), this row's old value `c`, its finished field words FW,
// its deviates rnd[], the entry address A of site 0 (with off = A - S) and the column offsets g1, gx1 of site 1.  While
// the row is processed, the row below is prepared in `n` (old value, partial planes), its field words FWn are finished
// (FWn[r] as soon as the sites 4q + r of this row are final) and its deviates replace this row's in rnd[] (call k after
// site 4k + 3).  Out: `up` = this row's new value, A / off / g1 / gx1 for the row below.
// Every site increments the bin of the state its attempt leads to (pipelined site macro).
template <int L, bool MEAS>
__device__ __forceinline__ void row_v6(uint32_t* __restrict__ lat, uint32_t& S, uint32_t& A, uint32_t& chk, uint32_t& off, uint32_t& g1,
                                       uint32_t& gx1, const int y, const bool more, uint32_t& up, const uint32_t c, uint32_t (&FW)[4],
                                       const uint32_t patch, uint32_t (&rnd)[Geo<L>::BITS], NextRow<L>& n, uint32_t (&FWn)[4],
                                       const uint4* ring, int& buf, const int bar_id, SitePipe& pp, RingCheck& rc) {
    using V = V6<L>;
    constexpr int SLOTS = V::SLOTS;
    // the deviates of row y + 1 are in ring[buf]; ring[buf ^ 1] (this row's, all fetched) may be refilled.  After the
    // last row of a phase there is no such barrier (the deviate warp has left its loop) and nothing is fetched.
    if (more) {
        pair_barrier(bar_id);
        ring_expect(rc, buf, CHK_RING_EARLY);
    }
    const int y1 = (y + 1) & (L - 1), y2 = (y + 2) & (L - 1);
    n.c = lat[y1 * SLOTS];
    n.dn = lat[y2 * SLOTS];   // row y + 2 is old (or row 0, final in this sweep, when y + 1 = L - 1)
    uint32_t flips = 0;
    RowSites<L, MEAS, 0, true, true, V::SBASE + V::DT_OFF, true>::run(S, A, flips, chk, off, g1, gx1, c, FW, FW[3], patch, rnd, n, FWn, FWn,
                                                                      ring, SLOTS, buf, more, pp);
    if (more) ring_fetched(rc, buf);
    state_check(rc, S >= V::SBASE && S <= V::SBASE + V::BINS * V::RS && (S - V::SBASE) % V::RS == 0u);
    buf ^= (int)more;
    up = c ^ flips;
    lat[y * SLOTS] = up;
    FWn[3] = finish_word<L>(n, up, 3);
}

// Walker warp: sweeps s0 .. s1-1; `buf` is the ring buffer holding the deviates of the next row to fetch.  Rows are
// processed in pairs so that the two register sets (this row / row below) swap roles without copies.
template <int L, bool MEAS>
__device__ __forceinline__ void sweeps_v6(uint32_t* __restrict__ lat, uint32_t& S, uint32_t& chk, const uint32_t s0, const uint32_t s1,
                                          const uint4* ring, int& buf, const int bar_id, RingCheck& rc) {
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
    ring_expect(rc, buf, CHK_RING_EARLY);
#pragma unroll
    for (int k = 0; k < NC; ++k) {
        const uint4 v = ring[(buf * NC + k) * SLOTS];
        rnd[4 * k] = v.x; rnd[4 * k + 1] = v.y; rnd[4 * k + 2] = v.z; rnd[4 * k + 3] = v.w;
    }
    ring_fetched(rc, buf);
    buf ^= 1;
    uint32_t off = (FWA[0] << 2) & 0x1Cu;      // site 0: its left neighbour (site L-1) has not been visited in this sweep
    uint32_t A = S + off;
    uint32_t g1 = (FWA[1] << 2) & 0x1Cu, gx1 = g1 ^ 4u;
    SitePipe pp;
    pp.dep = 0u;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(pp.t) : "r"(A) : "memory");                            // threshold and
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(pp.d) : "r"(off + V::SBASE + V::DT_OFF) : "memory");   // delta of site 0
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; y += 2) {
            row_v6<L, MEAS>(lat, S, A, chk, off, g1, gx1, y, true, up, nA.c, FWA, nA.patch, rnd, nB, FWB, ring, buf, bar_id, pp, rc);
            row_v6<L, MEAS>(lat, S, A, chk, off, g1, gx1, y + 1, s + 1 < s1 || y + 2 < L, up, nB.c, FWB, nB.patch, rnd, nA, FWA, ring, buf,
                            bar_id, pp, rc);
        }
    }
}

// Deviate warp: the NC Philox calls of one row advance round-major (NC independent IMAD.WIDE chains, philox_unit), results
// go to the double-buffered shared ring rnd[buf][call][slot] as one 16-byte store per call (lanes without a walker
// store nothing: their slots hold 0xFFFFFFFF for good).  One barrier per row hands the buffer over.
// R4: ctr = (i >> 2, sweep, iteration, walker).
template <int L>
__device__ __forceinline__ void deviates_v6(uint4* ring, uint4* scratch, const uint32_t s0, const uint32_t s1, int& buf,
                                            const int bar_id, const SweepParams& prm, const uint32_t walker, const bool active, const int lane,
                                            RingCheck& rc) {
    constexpr int NC = V6<L>::NC, SLOTS = V6<L>::SLOTS;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
        const PhiloxSweep pc = philox_sweep_consts(s, prm.iteration, prm.key0, prm.key1);
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            uint32_t st[NC][4];
            philox_unit<NC>(st, scratch, (uint32_t)(y * (L / 4)), pc, walker, lane);
#pragma unroll
            for (int k = 0; k < NC; ++k)
                if (active) ring[(buf * NC + k) * SLOTS] = make_uint4(st[k][0], st[k][1], st[k][2], st[k][3]);
            ring_publish(rc, buf, lane);
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
    if (!smem_base_ok(prm, sbase, V::SBASE)) return;   // the site macro addresses the delta table by an immediate

    // ---- table: row j = t[8] | bin; delta table behind the rows
    for (int idx = tid; idx < BINS * 8; idx += nthr) {
        const int j = idx >> 3, f = idx & 7, a = (f >> 1) + (f & 1);
        const int jn = j + 2 - a;                            // where an accepted move leads (dE = 8 - 4a)
        // R17: a move out of [0, N] cannot occur for a real configuration; its entry is never consulted
        *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + 4 * f) = (jn < 0 || jn > N) ? 0u : prm.table[idx];
    }
    for (int j = tid; j <= BINS; j += nthr) *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF) = 0u;
    if (tid < 8) {   // row BINS: t = 0 in every column; the lanes parked here get deviates 0xFFFFFFFF and stay
        const int f = tid, a = (f >> 1) + (f & 1);
        *reinterpret_cast<uint32_t*>(sm + (size_t)BINS * V::RS + 4 * f) = 0u;
        *reinterpret_cast<int32_t*>(sm + V::DT_OFF + 4 * f) = (int)V::RS * (2 - a);
    }

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
    uint4* const scratch = reinterpret_cast<uint4*>(sm + V::SCRATCH_OFF) + pair * V::NC;
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
    RingCheck rc;
#ifdef MUCA_CHECKED
    rc.tags = reinterpret_cast<volatile uint32_t*>(sm + V::TAG_OFF) + pair;
    rc.stride = V::MAX_WARPS;
    rc.flag = prm.check;
    rc.fault = blockIdx.x == 0 && pair == 0 ? prm.fault : 0u;
#endif
    // ---- thermalisation sweeps: nothing is recorded
    if (is_walker) sweeps_v6<L, false>(lat, S, chk, prm.sweep_begin, s_th, ring + slot, buf, bar_id, rc);
    else deviates_v6<L>(ring + slot, scratch, prm.sweep_begin, s_th, buf, bar_id, prm, walker, active, lane, rc);
    // ---- measured sweeps: every attempt counts the state it leads to
    if (is_walker) {
        sweeps_v6<L, true>(lat, S, chk, s_th, prm.sweep_end, ring + slot, buf, bar_id, rc);
    } else {
        deviates_v6<L>(ring + slot, scratch, s_th, prm.sweep_end, buf, bar_id, prm, walker, active, lane, rc);
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
