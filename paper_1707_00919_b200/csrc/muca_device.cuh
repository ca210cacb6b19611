// paper_1707_00919_b200/csrc/muca_device.cuh
// Device code of libmuca_b200 (sm_100a): Philox4x32-10, the packed-lattice layout helpers, the
// init / energy / pack / unpack kernels and the Metropolis sweep kernel (the hot path).
// Citations: "PAPER.md:<line>" = /root/reference/PAPER.md, "R<n>" = DESIGN.md section 3.
// Shares nothing with oracle/ (which is byte-per-spin, modulo arithmetic, no bit tricks).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace muca {

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 ("counter-based RNG Philox", Ref. [41]; R4: 4x32, 10 rounds).
// One round: (c0,c1,c2,c3) -> (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)); keys bumped by the
// Weyl constants after every round.  In the sweep kernel only c3 (the walker id) differs between the
// lanes of a warp, so ptxas moves the key schedule and the first round onto the uniform datapath.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ------------------------------------------------------------------------------------------------
// Packed lattice layout in HBM.  Spin bit 1 <-> spin -1.  "Typewriter word" t of a
// walker holds sites 32t .. 32t+31 (site i = y*L + x at bit i & 31).
//   L <  32 : word t of walker w at spins[t*W + w]                       (walker-interleaved words)
//   L >= 32 : row y = WPR = L/32 consecutive words; row y of walker w at spins[(y*W + w)*WPR .. +WPR)
//             (walker-interleaved ROWS: one 4/8/16-byte vector per thread, coalesced across the warp).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ size_t word_index(int L, int W, int w, int t) {
    if (L < 32) return (size_t)t * W + w;
    const int wpr = L >> 5;
    const int y = t / wpr, k = t - y * wpr;
    return ((size_t)y * W + w) * wpr + k;
}

// Row y of walker w as up to 4 words (bits 0..L-1 of the row, low word first); generic-L helper for the
// one-off kernels.
__device__ __forceinline__ void load_row(const uint32_t* spins, int L, int W, int w, int y,
                                         uint32_t (&row)[4]) {
    row[0] = row[1] = row[2] = row[3] = 0u;
    if (L < 32) {
        const int bit0 = y * L;
        const uint32_t word = spins[word_index(L, W, w, bit0 >> 5)];
        row[0] = (word >> (bit0 & 31)) & ((1u << L) - 1u);
    } else {
        const int wpr = L >> 5;
        for (int k = 0; k < wpr; ++k) row[k] = spins[word_index(L, W, w, y * wpr + k)];
    }
}

// Number of antiparallel bonds A of walker w; E = 2A - 2N (Eq. (5): every bond once,
// -1 if parallel, +1 if antiparallel), slot j = (E + 2N)/4 = A/2.
__device__ int antiparallel_bonds(const uint32_t* spins, int L, int W, int w) {
    int A = 0;
    uint32_t first[4], cur[4], nxt[4];
    load_row(spins, L, W, w, 0, first);
    for (int k = 0; k < 4; ++k) cur[k] = first[k];
    const int wpr = L < 32 ? 1 : (L >> 5);
    for (int y = 0; y < L; ++y) {
        if (y + 1 < L) load_row(spins, L, W, w, y + 1, nxt);
        else for (int k = 0; k < 4; ++k) nxt[k] = first[k];
        for (int k = 0; k < wpr; ++k) {
            uint32_t right;  // right neighbour of every site of word k (periodic in the row)
            if (L < 32) right = (cur[0] >> 1) | ((cur[0] & 1u) << (L - 1));
            else right = (cur[k] >> 1) | (cur[(k + 1) % wpr] << 31);
            A += __popc(cur[k] ^ right) + __popc(cur[k] ^ nxt[k]);
        }
        for (int k = 0; k < 4; ++k) cur[k] = nxt[k];
    }
    return A;
}

// ------------------------------------------------------------------------------------------------
// a0 -- initial configuration (R1, R5): typewriter word t = 4q + m of global walker g is word m of
// Philox(ctr = (q, 0, 0xFFFFFFFF, g), key).  One thread per walker.
// ------------------------------------------------------------------------------------------------
__global__ void init_kernel(uint32_t* spins, int32_t* E, int L, int W,
                            uint32_t walker_offset, uint32_t key0, uint32_t key1) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    const int N = L * L, n_words = N >> 5;
    for (int q = 0; 4 * q < n_words; ++q) {
        uint32_t r[4];
        philox4x32_10((uint32_t)q, 0u, 0xFFFFFFFFu, walker_offset + (uint32_t)w, key0, key1, r);
        for (int m = 0; m < 4 && 4 * q + m < n_words; ++m) spins[word_index(L, W, w, 4 * q + m)] = r[m];
    }
    E[w] = 2 * antiparallel_bonds(spins, L, W, w) - 2 * N;
}

__global__ void energy_kernel(const uint32_t* __restrict__ spins, int32_t* __restrict__ E, int L, int W) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= W) return;
    E[w] = 2 * antiparallel_bonds(spins, L, W, w) - 2 * L * L;
}

// a6 -- read-back: one thread per (walker, typewriter word) writes 32 int8 spins, out[w*N + i] = 1 - 2*bit.
__global__ void unpack_kernel(const uint32_t* __restrict__ spins, int8_t* __restrict__ out, int L, int W) {
    const int n_words = (L * L) >> 5;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)W * n_words) return;
    const int w = (int)(idx / n_words), t = (int)(idx - (size_t)w * n_words);
    const uint32_t word = spins[word_index(L, W, w, t)];
    uint4* dst = reinterpret_cast<uint4*>(out + idx * 32);  // 32-byte aligned: idx*32
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        uint32_t v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint32_t nib = (word >> (16 * h + 4 * q)) & 0xFu;
            // byte b = +1 (0x01) if bit clear, -1 (0xFF) if set
            uint32_t bytes = 0x01010101u;
#pragma unroll
            for (int b = 0; b < 4; ++b)
                if (nib & (1u << b)) bytes |= 0xFFu << (8 * b);
            v[q] = bytes;
        }
        dst[h] = make_uint4(v[0], v[1], v[2], v[3]);
    }
}

// inverse of unpack_kernel (muca_set_spins): in[w*N + i] < 0  <->  bit set.
__global__ void pack_kernel(const int8_t* __restrict__ in, uint32_t* __restrict__ spins, int L, int W) {
    const int n_words = (L * L) >> 5;
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)W * n_words) return;
    const int w = (int)(idx / n_words), t = (int)(idx - (size_t)w * n_words);
    const int8_t* src = in + idx * 32;
    uint32_t word = 0u;
    for (int b = 0; b < 32; ++b) word |= (src[b] < 0 ? 1u : 0u) << b;
    spins[word_index(L, W, w, t)] = word;
}

__global__ void philox_debug_kernel(const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key,
                                    uint32_t* __restrict__ out, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t r[4];
    philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], r);
    for (int m = 0; m < 4; ++m) out[4 * i + m] = r[m];
}

// ------------------------------------------------------------------------------------------------
// a2/a3/a4 -- the sweep kernel.
//
// Device threshold table "T8" (built on the host from omega, muca.cu): row j holds 8 words indexed by
//   f = 4*hi + 2*lo + g,   n3 = lo + 2*hi = antiparallel count over {up, down, right},  g = [left antiparallel],
//   T8[j][f] = thresh[j][a = n3 + g]     (PAPER.md:109 acceptance, R6/R7 integer form).
// The left neighbour is the site visited just before (typewriter order, R3), so g = hl ^ D where hl is the
// static bit (old left value) and D says whether the previous site flipped: the lookup address is
// (row + 4*f_static) ^ (D << 2) -- one XOR on the serial chain instead of a recount.
//
// Variants (template MODE):
//   0  TBL_SMEM   table AND histogram interleaved in shared memory (row stride 40 B: 8 thresholds, 1 bin, pad),
//                 lattices resident in shared memory                     (L <= 32)
//   1  TBL_L1     table read from global through L1 (32 B rows), histogram + lattices in shared memory (L = 64)
//   2  STREAMED   table through L1, histogram in shared memory, lattice rows streamed from HBM with a
//                 three-row register window and one-row-ahead prefetch    (L = 128; any L >= 32)
// ------------------------------------------------------------------------------------------------
struct SweepParams {
    uint32_t* spins;            // packed lattices (layout above)
    int32_t* E;                 // per-walker energy
    const uint32_t* table;      // T8, (N+1)*8 words, global
    unsigned long long* H;      // global histogram, N+1 bins
    int W;                      // walkers in this context
    uint32_t walker_offset;     // global id of walker 0 (R16)
    uint32_t key0, key1;        // Philox key = seed split low/high (R4)
    uint32_t iteration;         // n (R4: ctr.z)
    uint32_t sweep_begin;       // first sweep index of this launch (ctr.y)
    uint32_t sweep_end;         // one past the last
    uint32_t therm;             // sweeps with index < therm are not recorded
};

enum { MODE_TBL_SMEM = 0, MODE_TBL_L1 = 1, MODE_STREAMED = 2, MODE_V3 = 3, MODE_V5 = 4, MODE_STREAMED_SMEM = 5 };
//   5  STREAMED_SMEM  table + histogram in shared memory as in 0, lattice rows streamed as in 2: the lattices no longer
//                     limit the walkers per SM, so that 8 warps share an SM at L = 64 (164 KB of table) (L = 64)
__host__ __device__ constexpr bool tbl_in_smem(int mode) { return mode == MODE_TBL_SMEM || mode == MODE_STREAMED_SMEM; }
__host__ __device__ constexpr bool lat_streamed(int mode) { return mode == MODE_STREAMED || mode == MODE_STREAMED_SMEM; }

template <int L>
struct Geo {
    static constexpr int N = L * L;
    static constexpr int BINS = N + 1;
    static constexpr int WPR = L >= 32 ? L / 32 : 1;   // words per row
    static constexpr int BITS = L >= 32 ? 32 : L;      // valid bits per row word
    static constexpr uint32_t MASK = L >= 32 ? 0xFFFFFFFFu : ((1u << (L & 31)) - 1u);
};

constexpr int ROW_SMEM_WORDS = 10;  // MODE 0 row: 8 thresholds + 1 histogram bin + 1 pad (stride 40 B, multiple of 8)
constexpr int ROW_L1_WORDS = 8;     // MODE 1/2 row: 8 thresholds (32 B)

// Four consecutive sites (one Philox call) of the shared-memory-table variant, written in PTX so that the
// decision stays in a predicate along the serial chain (no SEL / 0-1 materialisation between sites):
//   pD -> @pD xor (column f ^ 1) -> address -> ld.shared -> setp -> pD ...
// o is the ABSOLUTE shared-memory address of the walker's table row.  (rp, tp) are the deviate and threshold
// of the previous site: re-evaluating rp <= tp recreates the predicate that cannot cross an asm boundary.
// t0: threshold used by the first site of the group (the row loop needs site 0's decision for the wrap patch).
#define MUCA_SITE_PTX(FWOP, ROP, MOP, MEAS_LINE)                                   \
    "shr.u32 f, " FWOP ", %16;\n\t"                                              \
    "and.b32 f, f, 7;\n\t"                                                         \
    "@pD xor.b32 f, f, 1;\n\t"                                                     \
    "shl.b32 ad, f, 2;\n\t"                                                        \
    "add.u32 ad, ad, %0;\n\t"                                                    \
    "ld.shared.u32 t, [ad];\n\t"                                                   \
    "prmt.b32 d, %14, %15, f;\n\t"                                       \
    "sub.u32 oa, %0, d;\n\t"                                                     \
    "add.u32 oa, oa, %17;\n\t"                                                  \
    "setp.le.u32 pD, " ROP ", t;\n\t"                                              \
    "@pD mov.u32 %0, oa;\n\t"                                                    \
    "@pD xor.b32 %1, %1, " MOP ";\n\t" MEAS_LINE

template <int Q, bool MEAS, uint32_t RS>
__device__ __forceinline__ void site_group_smem(const uint32_t fw0, const uint32_t fw1, const uint32_t fw2,
                                                const uint32_t fw3, uint32_t& o, uint32_t& c,
                                                const uint32_t (&rnd)[4], uint32_t& rp, uint32_t& tp, uint32_t& t0) {
    constexpr uint32_t LUT_LO = (RS * 0) | (RS * 1) << 8 | (RS * 1) << 16 | (RS * 2) << 24;
    constexpr uint32_t LUT_HI = (RS * 2) | (RS * 3) << 8 | (RS * 3) << 16 | (RS * 4) << 24;
    uint32_t t_first, t_last;
    if (MEAS) {
        asm volatile(
            "{\n\t.reg .pred pD;\n\t.reg .b32 f, ad, d, oa, t;\n\t"
            "setp.le.u32 pD, %12, %13;\n\t"
            MUCA_SITE_PTX("%4", "%8", "%18", "red.shared.add.u32 [%0+32], 1;\n\t")
            "mov.u32 %2, t;\n\t"
            MUCA_SITE_PTX("%5", "%9", "%19", "red.shared.add.u32 [%0+32], 1;\n\t")
            MUCA_SITE_PTX("%6", "%10", "%20", "red.shared.add.u32 [%0+32], 1;\n\t")
            MUCA_SITE_PTX("%7", "%11", "%21", "red.shared.add.u32 [%0+32], 1;\n\t")
            "mov.u32 %3, t;\n\t}"
            : "+r"(o), "+r"(c), "=r"(t_first), "=r"(t_last)
            : "r"(fw0), "r"(fw1), "r"(fw2), "r"(fw3), "r"(rnd[0]), "r"(rnd[1]),
              "r"(rnd[2]), "r"(rnd[3]), "r"(rp), "r"(tp), "r"(LUT_LO), "r"(LUT_HI),
              "n"(4 * Q), "n"(2 * RS), "n"(1u << (4 * Q)), "n"(1u << (4 * Q + 1)),
              "n"(1u << (4 * Q + 2)), "n"(1u << (4 * Q + 3))
            : "memory");
    } else {
        asm volatile(
            "{\n\t.reg .pred pD;\n\t.reg .b32 f, ad, d, oa, t;\n\t"
            "setp.le.u32 pD, %12, %13;\n\t"
            MUCA_SITE_PTX("%4", "%8", "%18", "")
            "mov.u32 %2, t;\n\t"
            MUCA_SITE_PTX("%5", "%9", "%19", "")
            MUCA_SITE_PTX("%6", "%10", "%20", "")
            MUCA_SITE_PTX("%7", "%11", "%21", "")
            "mov.u32 %3, t;\n\t}"
            : "+r"(o), "+r"(c), "=r"(t_first), "=r"(t_last)
            : "r"(fw0), "r"(fw1), "r"(fw2), "r"(fw3), "r"(rnd[0]), "r"(rnd[1]),
              "r"(rnd[2]), "r"(rnd[3]), "r"(rp), "r"(tp), "r"(LUT_LO), "r"(LUT_HI),
              "n"(4 * Q), "n"(2 * RS), "n"(1u << (4 * Q)), "n"(1u << (4 * Q + 1)),
              "n"(1u << (4 * Q + 2)), "n"(1u << (4 * Q + 3)));
    }
    rp = rnd[3];
    tp = t_last;
    t0 = t_first;
}

// The same four sites with the decision consumed by SELs instead of predicated instructions (measured recorded
// sweeps only; used by the paired streamed kernels, where a warp has a scheduler to itself or shares it with one other
// chain and the length of the chain is what counts):
//   pD -> SEL (carry 0/1) -> XOR (column) -> IMAD (address) -> ld.shared -> setp -> pD     and     pD -> SEL (state)
// ISETP -> SEL -> next instruction costs 9 cycles, ISETP -> predicated instruction -> next one about 17
// (profiles/r01_ubench_chain.txt).  The accept candidate oa passes through a LOP3 with a predicate output (true at run
// time: oa is a non-zero address): without a second, unconditional consumer ptxas folds "sub/add + selp" into an add
// predicated on the decision.
#define MUCA_SITE_SEL(FWOP, ROP, MOP)                                              \
    "shr.u32 f0, " FWOP ", %16;\n\t"                                             \
    "and.b32 f0, f0, 7;\n\t"                                                       \
    "selp.u32 cy, 1, 0, pD;\n\t"                                                   \
    "xor.b32 f, f0, cy;\n\t"                                                       \
    "mad.lo.u32 ad, f, 4, %0;\n\t"                                               \
    "ld.shared.u32 t, [ad];\n\t"                                                   \
    "prmt.b32 d, %14, %15, f;\n\t"                                     \
    "sub.u32 oa, %0, d;\n\t"                                                     \
    "add.u32 oa, oa, %17;\n\t"                                                  \
    "lop3.and.b32 oa|pq, oa, oa, oa, 0xF0, pt;\n\t"                                \
    "setp.le.and.u32 pD, " ROP ", t, pq;\n\t"                                      \
    "selp.u32 %0, oa, %0, pD;\n\t"                                             \
    "@pD xor.b32 %1, %1, " MOP ";\n\t"                                             \
    "red.shared.add.u32 [%0+32], 1;\n\t"

template <int Q, uint32_t RS>
__device__ __forceinline__ void site_group_smem_sel(const uint32_t fw0, const uint32_t fw1, const uint32_t fw2,
                                                    const uint32_t fw3, uint32_t& o, uint32_t& c,
                                                    const uint32_t (&rnd)[4], uint32_t& rp, uint32_t& tp, uint32_t& t0) {
    constexpr uint32_t LUT_LO = (RS * 0) | (RS * 1) << 8 | (RS * 1) << 16 | (RS * 2) << 24;
    constexpr uint32_t LUT_HI = (RS * 2) | (RS * 3) << 8 | (RS * 3) << 16 | (RS * 4) << 24;
    uint32_t t_first, t_last;
    asm volatile(
        "{\n\t.reg .pred pD, pq, pt;\n\t.reg .b32 f0, cy, f, ad, d, oa, t;\n\t"
        "setp.eq.u32 pt, 0, 0;\n\t"
        "setp.le.u32 pD, %12, %13;\n\t"
        MUCA_SITE_SEL("%4", "%8", "%18")
        "mov.u32 %2, t;\n\t"
        MUCA_SITE_SEL("%5", "%9", "%19")
        MUCA_SITE_SEL("%6", "%10", "%20")
        MUCA_SITE_SEL("%7", "%11", "%21")
        "mov.u32 %3, t;\n\t}"
        : "+r"(o), "+r"(c), "=r"(t_first), "=r"(t_last)
        : "r"(fw0), "r"(fw1), "r"(fw2), "r"(fw3), "r"(rnd[0]), "r"(rnd[1]),
          "r"(rnd[2]), "r"(rnd[3]), "r"(rp), "r"(tp), "r"(LUT_LO), "r"(LUT_HI),
          "n"(4 * Q), "n"(2 * RS), "n"(1u << (4 * Q)), "n"(1u << (4 * Q + 1)),
          "n"(1u << (4 * Q + 2)), "n"(1u << (4 * Q + 3))
        : "memory");
    rp = rnd[3];
    tp = t_last;
    t0 = t_first;
}

template <int Q, int QN, int L, bool MEAS, uint32_t RS>
struct GroupLoop {
    // groups Q .. QN-1 of word k of a row (compile-time recursion: the shifts and flip masks are immediates)
    static __device__ __forceinline__ void run(uint32_t (&FWk)[4], uint32_t* FWlast3, const uint32_t patch, const bool first_word,
                                               uint32_t& o, uint32_t& c, uint32_t& rp, uint32_t& tp, const uint32_t ctr0,
                                               const uint32_t sweep, const uint32_t iteration, const uint32_t walker,
                                               const uint32_t key0, const uint32_t key1) {
        uint32_t rnd[4], t0;
        philox4x32_10(ctr0 + (uint32_t)Q, sweep, iteration, walker, key0, key1, rnd);
        site_group_smem<Q, MEAS, RS>(FWk[0], FWk[1], FWk[2], FWk[3], o, c, rnd, rp, tp, t0);
        if (Q == 0 && first_word) {
            // the right neighbour of the LAST site of the row is site 0, which has just been decided
            if (rnd[0] <= t0) *FWlast3 += patch;
        }
        GroupLoop<Q + 1, QN, L, MEAS, RS>::run(FWk, FWlast3, patch, first_word, o, c, rp, tp, ctr0, sweep, iteration, walker,
                                               key0, key1);
    }
};
template <int QN, int L, bool MEAS, uint32_t RS>
struct GroupLoop<QN, QN, L, MEAS, RS> {
    static __device__ __forceinline__ void run(uint32_t (&)[4], uint32_t*, const uint32_t, const bool, uint32_t&, uint32_t&,
                                               uint32_t&, uint32_t&, const uint32_t, const uint32_t, const uint32_t,
                                               const uint32_t, const uint32_t, const uint32_t) {}
};

// Deviates handed over by a paired deviate warp through a double-buffered shared ring (muca_window.cuh,
// sweep_kernel_wpair): ring[(buf * 8 + call) * slots], one uint4 per call and walker, one barrier per 32-site word.
struct DeviateFeed {
    const uint4* ring;   // + this walker's slot
    int slots, buf, bar_id;
};

// as GroupLoop, with the deviates of the word in rnd[32] instead of a Philox call per group
template <int Q, int QN, int L, bool MEAS, uint32_t RS>
struct GroupLoopExt {
    static __device__ __forceinline__ void run(uint32_t (&FWk)[4], uint32_t* FWlast3, const uint32_t patch, const bool first_word,
                                               uint32_t& o, uint32_t& c, uint32_t& rp, uint32_t& tp, const uint32_t (&rndw)[32]) {
        uint32_t t0;
        const uint32_t rnd[4] = {rndw[4 * Q], rndw[4 * Q + 1], rndw[4 * Q + 2], rndw[4 * Q + 3]};
        // SEL form where the chain length counts (L = 128: every warp has a scheduler to itself, c_flip 55.9 -> 53.2);
        // at L = 64 (7 pairs per SM, ALU pipe 59 % busy) the predicate-carried form is 2 % faster
        if constexpr (MEAS && L >= 128) site_group_smem_sel<Q, RS>(FWk[0], FWk[1], FWk[2], FWk[3], o, c, rnd, rp, tp, t0);
        else site_group_smem<Q, MEAS, RS>(FWk[0], FWk[1], FWk[2], FWk[3], o, c, rnd, rp, tp, t0);
        if (Q == 0 && first_word) {
            if (rnd[0] <= t0) *FWlast3 += patch;
        }
        GroupLoopExt<Q + 1, QN, L, MEAS, RS>::run(FWk, FWlast3, patch, first_word, o, c, rp, tp, rndw);
    }
};
template <int QN, int L, bool MEAS, uint32_t RS>
struct GroupLoopExt<QN, QN, L, MEAS, RS> {
    static __device__ __forceinline__ void run(uint32_t (&)[4], uint32_t*, const uint32_t, const bool, uint32_t&, uint32_t&,
                                               uint32_t&, uint32_t&, const uint32_t (&)[32]) {}
};

// One typewriter pass over row y of one walker.  up/dn: rows above/below (current values), cur: the row,
// updated in place.  o: byte offset of the walker's energy row in the table (= j * row stride), updated.
//
// Per row (bit-sliced, ~30 instructions for 32 sites): the three static planes
//   lo, hi = the two bits of n3 = [up != s] + [down != s] + [right != s],   hl = [left(old) != s]
// are interleaved into four "field words" FW[r] (r = x & 3): nibble q of FW[r] holds the table column
// f = hl + 2*lo + 4*hi of site x = 4q + r, so the per-site extraction is one shift and one mask.
// Per site the serial chain is  D(prev) -> f ^= D -> address -> LDS -> compare -> D:
//   fw   = f ^ D                     D: previous site flipped, which toggles the [left != s] bit (column f ^ 1)
//   t    = T8[row o][fw]             one 4-byte load (shared memory or L1)
//   D    = r <= t                    R6/R7
//   o   += D ? RS*(2 - a(fw)) : 0    RS*a(fw) comes from an 8-entry byte table in two registers (PRMT)
//   s_x ^= D                         predicated XOR with an immediate
//   H[row o] += 1                    shared-memory atomic, measured sweeps only
template <int L, int MODE, bool MEAS, bool EXT = false>
__device__ __forceinline__ void process_row(const uint32_t (&up)[Geo<L>::WPR], uint32_t (&cur)[Geo<L>::WPR],
                                            const uint32_t (&dn)[Geo<L>::WPR], uint32_t& o,
                                            const uint32_t ctr0_row, const uint32_t sweep, const uint32_t iteration,
                                            const uint32_t walker, const uint32_t key0, const uint32_t key1,
                                            const char* __restrict__ tbl_smem, const char* __restrict__ tbl_glob,
                                            uint32_t* __restrict__ hist, DeviateFeed* feed = nullptr) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, BITS = G::BITS;
    constexpr uint32_t RS = (tbl_in_smem(MODE) ? ROW_SMEM_WORDS : ROW_L1_WORDS) * 4;  // row stride in bytes
    // byte f of (LUT_HI:LUT_LO) = RS * a(f), a(f) = (f >> 1) + (f & 1) = antiparallel neighbours of column f
    constexpr uint32_t LUT_LO = (RS * 0) | (RS * 1) << 8 | (RS * 1) << 16 | (RS * 2) << 24;
    constexpr uint32_t LUT_HI = (RS * 2) | (RS * 3) << 8 | (RS * 3) << 16 | (RS * 4) << 24;
    static_assert(RS * 4 < 256, "row stride must keep RS*a in a byte");

    uint32_t FW[WPR][4];
    uint32_t patch = 0;   // added to FW[WPR-1][3] when site 0 flips: n3 of the LAST site changes by +-1
#pragma unroll
    for (int k = 0; k < WPR; ++k) {
        const uint32_t c = cur[k];
        uint32_t rw, lw;
        if constexpr (L >= 32) {
            rw = (c >> 1) | (cur[(k + 1) % WPR] << 31);          // right neighbours (old; last site patched)
            lw = (c << 1) | (cur[(k + WPR - 1) % WPR] >> 31);    // left neighbours (old)
        } else {
            rw = (c >> 1) | ((c & 1u) << (BITS - 1));
            lw = ((c << 1) | (c >> (BITS - 1))) & G::MASK;
        }
        const uint32_t vu = c ^ up[k], vd = c ^ dn[k], hr = c ^ rw;
        const uint32_t hl = c ^ lw;
        const uint32_t lo = vu ^ vd ^ hr;
        const uint32_t hi = (vu & vd) | (vu & hr) | (vd & hr);
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t A = hl >> r;                                   // bit 4q+r -> 4q
            const uint32_t B = r >= 1 ? lo >> (r - 1) : lo << 1;          //          -> 4q+1
            const uint32_t C = r >= 2 ? hi >> (r - 2) : hi << (2 - r);    //          -> 4q+2
            const uint32_t t1 = (A & 0x11111111u) | (B & ~0x11111111u);
            FW[k][r] = (t1 & 0x33333333u) | (C & ~0x33333333u);           // bit 4q+3 is junk, masked at extraction
        }
        if (k == WPR - 1) {
            constexpr int QL = BITS / 4 - 1;                              // nibble of the last site in FW[.][3]
            const uint32_t hr_last = (hr >> (BITS - 1)) & 1u;
            patch = (1u << (4 * QL + 1)) - (hr_last << (4 * QL + 2));     // +1 on n3 if the bond was parallel, else -1
        }
    }

    if constexpr (tbl_in_smem(MODE)) {
        // o is the absolute shared-memory address of the walker's table row (see site_group_smem)
        uint32_t rp = 1u, tp = 0u;   // "previous site did not flip": site 0's left neighbour is site L-1, not yet visited
#pragma unroll
        for (int k = 0; k < WPR; ++k) {
            uint32_t c = cur[k];
            if constexpr (EXT) {
                static_assert(BITS == 32, "external deviates: one ring hand-over per 32-site word");
                asm volatile("bar.sync %0, 64;" ::"r"(feed->bar_id) : "memory");   // the deviates of this word are in ring[buf]
                uint32_t rndw[32];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    const uint4 v = feed->ring[(feed->buf * 8 + q) * feed->slots];
                    rndw[4 * q] = v.x; rndw[4 * q + 1] = v.y; rndw[4 * q + 2] = v.z; rndw[4 * q + 3] = v.w;
                }
                feed->buf ^= 1;
                GroupLoopExt<0, BITS / 4, L, MEAS, RS>::run(FW[k], &FW[WPR - 1][3], patch, k == 0, o, c, rp, tp, rndw);
            } else {
                GroupLoop<0, BITS / 4, L, MEAS, RS>::run(FW[k], &FW[WPR - 1][3], patch, k == 0, o, c, rp, tp,
                                                         ctr0_row + (uint32_t)(k * 8), sweep, iteration, walker, key0, key1);
            }
            cur[k] = c;
        }
    } else {
        bool D = false;  // did the previous site of this row flip?
#pragma unroll
        for (int k = 0; k < WPR; ++k) {
            uint32_t c = cur[k];
#pragma unroll
            for (int q = 0; q < BITS / 4; ++q) {
                uint32_t rnd[4];
                philox4x32_10(ctr0_row + (uint32_t)(k * 8 + q), sweep, iteration, walker, key0, key1, rnd);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int x = q * 4 + r;
                    uint32_t fw = (FW[k][r] >> (4 * q)) & 7u;
                    if (D) fw ^= 1u;
                    const uint32_t t = __ldg(reinterpret_cast<const uint32_t*>(tbl_glob + (o + 4u * fw)));
                    const uint32_t o_acc = o + 2u * RS - __byte_perm(LUT_LO, LUT_HI, fw);   // j + 2 - a  (dE = 8 - 4a)
                    D = rnd[r] <= t;                                       // R6/R7: accept iff r <= t
                    if (D) {
                        o = o_acc;
                        c ^= 1u << x;
                    }
                    if (MEAS) atomicAdd(hist + (o >> 5), 1u);              // H[j]++ after EVERY attempt
                    if (k == 0 && x == 0) {
                        // the right neighbour of the LAST site of the row is site 0, which has just been decided
                        if (D) FW[WPR - 1][3] += patch;
                    }
                }
            }
            cur[k] = c;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// v3 resident kernel for L <= 32: "state in the address".
//
// The walker's whole dynamic state -- energy slot j AND the carry c = [previous site of this row flipped] --
// is ONE shared-memory address P = rowaddr(j, c).  The table is stored twice: copy c at byte offset c*K (K a
// power of two above copy 0 and the lattices), and copy 1 has its columns permuted (f -> f ^ 1: a flipped
// left neighbour toggles the [left != s] bit).  Entry (j, c, f) is 8 bytes {t, dP}:
//     t  = thresh[j][a],  a = a(f ^ c)                 (PAPER.md:109 acceptance, R6/R7)
//     dP = rowaddr(j + 2 - a, 1) - rowaddr(j, c)        (where an ACCEPTED move leads; a rejected one leads to
//                                                        rowaddr(j, 0) = P & ~K)
// so the per-site serial chain is   P -> IMAD (P + 8f) -> LDS.64 -> {ISETP | IADD} -> SEL -> P'
// with no predicated instruction on it (ISETP -> predicated op costs ~13 cycles more than ISETP -> SEL on
// sm_100a, profiles/r01_ubench_pipes.txt) and no PRMT / column fix-up.  Row j of a copy is 72 bytes:
// 8 entries, the histogram bin of (j, c) at +64, 4 bytes of padding; the two bins of a slot are added at the merge.
// ------------------------------------------------------------------------------------------------
template <int L>
struct V3 {
    static constexpr uint32_t BINS = L * L + 1;
    static constexpr uint32_t RS = 72;
    static constexpr uint32_t BIN_OFF = 64;
    static constexpr uint32_t TBL_BYTES = (BINS + 1) * RS;   // + one all-reject row for the unused slots of the last block
    static constexpr uint32_t K = L == 32 ? 131072u : (L == 16 ? 65536u : 32768u);
    static constexpr uint32_t LAT_OFF = (TBL_BYTES + 15u) & ~15u;
    static constexpr int MAX_TPB = 128;                      // walkers per block; lattices + deviate ring must fit between copy 0 and K
    static_assert(1024u + LAT_OFF + 16u + ((uint32_t)L * 4u + 2u * (L / 4) * 16u) * MAX_TPB <= K, "copy 0 + lattices + ring must end below K");
    static constexpr size_t SMEM_BYTES = (size_t)K + TBL_BYTES;
};

// static planes of one row (single word, L <= 32): nibble q of FW[r] = column f = hl + 2*lo + 4*hi of site 4q + r
template <int L>
__device__ __forceinline__ void field_words(const uint32_t up, const uint32_t c, const uint32_t dn, uint32_t (&FW)[4],
                                            uint32_t& patch) {
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
    const uint32_t vu = c ^ up, vd = c ^ dn, hr = c ^ rw, hl = c ^ lw;
    const uint32_t lo = vu ^ vd ^ hr;
    const uint32_t hi = (vu & vd) | (vu & hr) | (vd & hr);
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const uint32_t A = hl >> r;
        const uint32_t B = r >= 1 ? lo >> (r - 1) : lo << 1;
        const uint32_t C = r >= 2 ? hi >> (r - 2) : hi << (2 - r);
        const uint32_t t1 = (A & 0x11111111u) | (B & ~0x11111111u);
        FW[r] = (t1 & 0x33333333u) | (C & ~0x33333333u);
    }
    constexpr int QL = BITS / 4 - 1;
    const uint32_t hr_last = (hr >> (BITS - 1)) & 1u;
    patch = (1u << (4 * QL + 1)) - (hr_last << (4 * QL + 2));   // site 0 flipped: n3 of the LAST site +-1
}

// One Philox4x32-10 round on the state of one call (see philox4x32_10 above).
__device__ __forceinline__ void philox_round(uint32_t (&c)[4], const uint32_t k0, const uint32_t k1) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
    c[1] = (uint32_t)p1;
    c[3] = (uint32_t)p0;
    c[0] = n0;
    c[2] = n2;
}

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 for the deviate warps, with everything that does not depend on the walker taken out of the lanes.
// R4: ctr = (c0 = i >> 2, sweep, iteration, walker): only ctr.w differs between the lanes of a warp, so round 0 needs no
// per-lane multiply at all, rounds 1 and 2 need one each, rounds 3 .. 9 two each: 16 of the 20 wide multiplies of a call
// (nvcc, left to itself, keeps 18 in the lanes).  The four others give values that are the same for all walkers:
//   per kernel : (hi1, lo1) = M1 * iteration;                 Y2 = lo1 ^ K0[1]
//   per sweep  : (hi_s, lo_s) = M0 * (hi1 ^ sweep ^ K0[0]);   W3 = lo_s ^ K1[2]
//   per call   : (hi0, lo0) = M0 * c0,  (hi3, lo3) = M1 * (hi_s ^ lo0 ^ K1[1]):
//                U1 = hi0 ^ K1[0],  X3 = hi3 ^ K0[2],  L3k = lo3 ^ K0[3]
// (K0[r], K1[r]: the round keys key + r * Weyl constant).  The per-call values of the NC calls of a unit are computed by
// the lanes 0 .. NC-1 of the deviate warp (lane q: call q) into a warp-private scratch of 16 bytes per call and read back
// by all lanes with one broadcast load per call.
// ------------------------------------------------------------------------------------------------
struct PhiloxSweep { uint32_t hi_s, W3, Y2, k0, k1; };   // per-sweep / per-kernel values and the key

__device__ __forceinline__ PhiloxSweep philox_sweep_consts(const uint32_t sweep, const uint32_t iteration, const uint32_t k0, const uint32_t k1) {
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * iteration;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint64_t ps = (uint64_t)0xD2511F53u * (hi1 ^ sweep ^ k0);
    PhiloxSweep c;
    c.hi_s = (uint32_t)(ps >> 32);
    c.W3 = (uint32_t)ps ^ (k1 + 2u * 0xBB67AE85u);
    c.Y2 = lo1 ^ (k0 + 0x9E3779B9u);
    c.k0 = k0; c.k1 = k1;
    return c;
}
// lane q < ncalls: the walker-independent values of call c0_base + q -> scratch[q]
__device__ __forceinline__ void philox_call_consts(uint4* scratch, const int ncalls, const uint32_t c0_base, const PhiloxSweep& c, const int lane) {
    if (lane < ncalls) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (c0_base + (uint32_t)lane);
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint64_t p3 = (uint64_t)0xCD9E8D57u * (c.hi_s ^ lo0 ^ (c.k1 + 0xBB67AE85u));
        scratch[lane] = make_uint4(hi0 ^ c.k1, (uint32_t)(p3 >> 32) ^ (c.k0 + 2u * 0x9E3779B9u), (uint32_t)p3 ^ (c.k0 + 3u * 0x9E3779B9u), 0u);
    }
    __syncwarp();
}
// rounds 0 .. 2 of one call for this lane's walker, from the values above; the state is ready for round 3
__device__ __forceinline__ void philox_head(uint32_t (&st)[4], const uint4 u, const PhiloxSweep& c, const uint32_t walker) {
    const uint32_t c2 = u.x ^ walker;                                   // round 0: c2 = hi0 ^ walker ^ K1[0]
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;                     // round 1: the only per-lane product
    const uint32_t c0 = (uint32_t)(p1 >> 32) ^ c.Y2, c1 = (uint32_t)p1;
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;                     // round 2: the only per-lane product
    st[0] = u.y ^ c1;                                                   // hi3 ^ c1 ^ K0[2]
    st[1] = u.z;                                                        // lo3 ^ K0[3]: round 3 uses it as (c1 ^ K0[3])
    st[2] = (uint32_t)(p0 >> 32) ^ c.W3;                                // hi(p0) ^ lo_s ^ K1[2]
    st[3] = (uint32_t)p0;
}
// round 3: as philox_round, with c1 ^ K0[3] already folded into st[1]
__device__ __forceinline__ void philox_round3(uint32_t (&st)[4], const uint32_t k1_3) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * st[0];
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * st[2];
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ st[1];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ st[3] ^ k1_3;
    st[1] = (uint32_t)p1;
    st[3] = (uint32_t)p0;
    st[0] = n0;
    st[2] = n2;
}
// the NC calls c0_base .. c0_base + NC - 1 of one unit, round-major (NC independent multiply chains)
template <int NC>
__device__ __forceinline__ void philox_unit(uint32_t (&st)[NC][4], uint4* scratch, const uint32_t c0_base, const PhiloxSweep& c,
                                            const uint32_t walker, const int lane) {
    philox_call_consts(scratch, NC, c0_base, c, lane);
#pragma unroll
    for (int q = 0; q < NC; ++q) philox_head(st[q], scratch[q], c, walker);
    __syncwarp();   // the scratch may be rewritten for the next unit
#pragma unroll
    for (int q = 0; q < NC; ++q) philox_round3(st[q], c.k1 + 3u * 0xBB67AE85u);
#pragma unroll
    for (int r = 4; r < 10; ++r)
#pragma unroll
        for (int q = 0; q < NC; ++q) philox_round(st[q], c.k0 + (uint32_t)r * 0x9E3779B9u, c.k1 + (uint32_t)r * 0xBB67AE85u);
}

__device__ __forceinline__ void pair_barrier(const int id) {   // named barrier of one walker warp + its deviate warp
    asm volatile("bar.sync %0, 64;" ::"r"(id) : "memory");
}

// Deviate warp: the BITS/4 Philox calls of one row advance round-major (16 independent IMAD.WIDE chains at L = 32:
// a lone dependent chain issues one instruction per ~5 cycles), results go to the double-buffered shared ring
// rnd[buf][call][walker] as one 16-byte store per call.  One barrier per row hands the buffer over.
template <int L>
__device__ __forceinline__ void deviate_rows(uint4* __restrict__ ring, const int WB, const int ptid, const int bar_id,
                                             const SweepParams& prm, const uint32_t walker) {
    constexpr int NC = Geo<L>::BITS / 4;
    int buf = 0;
#pragma unroll 1
    for (uint32_t s = prm.sweep_begin; s < prm.sweep_end; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            uint32_t st[NC][4];
#pragma unroll
            for (int k = 0; k < NC; ++k) {     // R4: ctr = (i >> 2, sweep, iteration, walker)
                st[k][0] = (uint32_t)(y * (L / 4) + k); st[k][1] = s; st[k][2] = prm.iteration; st[k][3] = walker;
            }
#pragma unroll
            for (int r = 0; r < 10; ++r)
#pragma unroll
                for (int k = 0; k < NC; ++k)
                    philox_round(st[k], prm.key0 + (uint32_t)r * 0x9E3779B9u, prm.key1 + (uint32_t)r * 0xBB67AE85u);
#pragma unroll
            for (int k = 0; k < NC; ++k) ring[(buf * NC + k) * WB + ptid] = make_uint4(st[k][0], st[k][1], st[k][2], st[k][3]);
            pair_barrier(bar_id);
            buf ^= 1;
        }
    }
}

// Walker warp: sweeps s0 .. s1-1; `buf` is the ring buffer holding the deviates of the next row to process.
template <int L, bool MEAS>
__device__ __forceinline__ void sweeps_v3(uint32_t* __restrict__ lat, const int WB, uint32_t& P, const uint32_t s0,
                                          const uint32_t s1, const uint4* __restrict__ ring, int& buf, const int bar_id) {
    using G = Geo<L>;
    using V = V3<L>;
    constexpr int BITS = G::BITS, NC = BITS / 4;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            const int ym = (y + L - 1) & (L - 1), yp = (y + 1) & (L - 1);
            const uint32_t up = lat[ym * WB], dn = lat[yp * WB];
            const uint32_t c = lat[y * WB];
            uint32_t FW[4], patch;
            field_words<L>(up, c, dn, FW, patch);
            pair_barrier(bar_id);              // the deviates of this row are in ring[buf]; ring[buf ^ 1] may be refilled
            uint32_t rnd[BITS];
#pragma unroll
            for (int k = 0; k < NC; ++k) {
                const uint4 v = ring[(buf * NC + k) * WB];
                rnd[4 * k] = v.x; rnd[4 * k + 1] = v.y; rnd[4 * k + 2] = v.z; rnd[4 * k + 3] = v.w;
            }
            buf ^= 1;
            P &= ~V::K;                        // site 0: its left neighbour (site L-1) has not been visited in this sweep
            uint32_t A = P + ((FW[0] << 3) & 0x38u);
            uint32_t hpend = 0, flips = 0;
#pragma unroll
            for (int x = 0; x < BITS; ++x) {
                uint32_t t, dP;
                asm("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(t), "=r"(dP) : "r"(A));
                if (MEAS && x > 0)                 // H[j]++ of the PREVIOUS site, issued behind this site's table load
                    asm volatile("red.shared.add.u32 [%0+64], 1;" ::"r"(hpend) : "memory");
                const bool D = rnd[x] <= t;        // R6/R7: accept iff r <= t
                if (x == 0 && D) FW[3] += patch;
                // column offset of the next site; both candidates of its entry address are ready before D is known
                const int xn = x + 1;
                const uint32_t f8n = xn >= BITS ? 0u
                                     : (xn >> 2) == 0 ? (FW[xn & 3] << 3) & 0x38u
                                                      : (FW[xn & 3] >> ((xn >> 2) > 0 ? 4 * (xn >> 2) - 3 : 0)) & 0x38u;
                // A_acc feeds both the select below and P_acc, which keeps ptxas from folding the add into a predicated
                // instruction (ISETP -> predicated op costs ~9 cycles more than ISETP -> SEL on the serial chain)
                const uint32_t P_rej = P & ~V::K, A_rej = P_rej + f8n, Q = P + f8n;
                uint32_t A_acc;
                asm("add.u32 %0, %1, %2;" : "=r"(A_acc) : "r"(Q), "r"(dP));
                A = D ? A_acc : A_rej;
                P = D ? A_acc - f8n : P_rej;
                if (D) flips |= 1u << x;
                hpend = P;
            }
            if (MEAS)
                asm volatile("red.shared.add.u32 [%0+64], 1;" ::"r"(hpend) : "memory");
            lat[y * WB] = c ^ flips;
        }
    }
}

// Block = WB deviate threads (warps 0 .. WB/32-1) + WB walker threads (the next WB/32 warps); walker warp i and
// deviate warp i serve the same 32 walkers and, at WB = 128, share one scheduler (warp ids i and i + 4), so the
// hardware interleaves the Philox instruction stream into the stalls of the walker warp's serial chain.
template <int L>
__global__ void __launch_bounds__(2 * V3<L>::MAX_TPB, 1) sweep_kernel_v3(const SweepParams prm) {
    using G = Geo<L>;
    using V = V3<L>;
    constexpr int N = G::N, BINS = G::BINS, NC = G::BITS / 4;
    extern __shared__ __align__(16) uint32_t smem[];
    char* const sm = reinterpret_cast<char*>(smem);
    const int tid = threadIdx.x, nthr = blockDim.x, WB = nthr >> 1;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t ring_off = (V::LAT_OFF + (uint32_t)L * 4u * (uint32_t)WB + 15u) & ~15u;
    if (sbase + ring_off + 2u * NC * 16u * (uint32_t)WB > V::K) __trap();

    // ---- both table copies: entry (j, c, f) = {t, dP}; bins zeroed
    for (int idx = tid; idx < BINS * 16; idx += nthr) {
        const int j = idx >> 4, cc = (idx >> 3) & 1, f = idx & 7;
        const int fe = f ^ cc, a = (fe >> 1) + (fe & 1);
        uint2 e;
        e.x = prm.table[j * 8 + fe];
        e.y = (uint32_t)((int)V::RS * (2 - a)) + (cc ? 0u : V::K);
        *reinterpret_cast<uint2*>(sm + (size_t)cc * V::K + (size_t)j * V::RS + 8 * f) = e;
    }
    for (int idx = tid; idx < BINS * 2; idx += nthr) {
        const int j = idx >> 1, cc = idx & 1;
        *reinterpret_cast<uint2*>(sm + (size_t)cc * V::K + (size_t)j * V::RS + V::BIN_OFF) = make_uint2(0u, 0u);
    }
    if (tid < 9)   // row BINS of copy 0: {t = 0, dP = 0} in every column -- a walker parked here stays here; its bin is never merged
        *reinterpret_cast<uint2*>(sm + (size_t)BINS * V::RS + 8 * tid) = make_uint2(0u, 0u);

    const bool is_walker = tid >= WB;                          // higher warp ids win the scheduler's arbitration: give them the serial chain
    const int lt = is_walker ? tid - WB : tid;                 // walker slot in the block
    const int w = blockIdx.x * WB + lt;
    const bool active = w < prm.W;                             // unused slots of the last block are parked on the all-reject row
    const int bar_id = 1 + (lt >> 5);
    uint32_t* const lat = reinterpret_cast<uint32_t*>(sm + V::LAT_OFF) + lt;
    uint4* const ring = reinterpret_cast<uint4*>(sm + ring_off);

    // ---- lattice: one word per row
    if (is_walker) {
        if (!active) {
            for (int y = 0; y < L; ++y) lat[y * WB] = 0u;
        } else if (L >= 32) {
            for (int y = 0; y < L; ++y) lat[y * WB] = prm.spins[(size_t)y * prm.W + w];
        } else {
            constexpr int RPW = 32 / G::BITS;
            for (int t = 0; t < N / 32; ++t) {
                const uint32_t word = prm.spins[(size_t)t * prm.W + w];
#pragma unroll
                for (int q = 0; q < RPW; ++q) lat[(t * RPW + q) * WB] = (word >> (q * G::BITS)) & G::MASK;
            }
        }
    }
    __syncthreads();

    const uint32_t walker = prm.walker_offset + (uint32_t)w;
    if (!is_walker) {
        deviate_rows<L>(ring, WB, lt, bar_id, prm, walker);
    } else {
        // slot j = (E + 2N)/4, copy 0
        uint32_t P = sbase + (active ? (uint32_t)((prm.E[w] + 2 * N) >> 2) : (uint32_t)BINS) * V::RS;
        const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                              : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
        int buf = 0;
        sweeps_v3<L, false>(lat, WB, P, prm.sweep_begin, s_th, ring + lt, buf, bar_id);
        sweeps_v3<L, true>(lat, WB, P, s_th, prm.sweep_end, ring + lt, buf, bar_id);
        if (active) {
            prm.E[w] = (int)(((P & ~V::K) - sbase) / V::RS) * 4 - 2 * N;
            if (L >= 32) {
                for (int y = 0; y < L; ++y) prm.spins[(size_t)y * prm.W + w] = lat[y * WB];
            } else {
                constexpr int RPW = 32 / G::BITS;
                for (int t = 0; t < N / 32; ++t) {
                    uint32_t word = 0u;
#pragma unroll
                    for (int q = 0; q < RPW; ++q) word |= lat[(t * RPW + q) * WB] << (q * G::BITS);
                    prm.spins[(size_t)t * prm.W + w] = word;
                }
            }
        }
    }
    __syncthreads();

    // ---- a4: merge the two bins of every slot into the global uint64 histogram
    if (prm.sweep_end > prm.therm) {
        for (int j = tid; j < BINS; j += nthr) {
            const uint32_t v = *reinterpret_cast<uint32_t*>(sm + (size_t)j * V::RS + V::BIN_OFF) +
                               *reinterpret_cast<uint32_t*>(sm + (size_t)V::K + (size_t)j * V::RS + V::BIN_OFF);
            if (v) atomicAdd(prm.H + j, (unsigned long long)v);
        }
    }
}

template <int WPR> struct RowVec;
template <> struct RowVec<1> { using type = uint32_t; };
template <> struct RowVec<2> { using type = uint2; };
template <> struct RowVec<4> { using type = uint4; };

template <int WPR>
__device__ __forceinline__ void ld_row(const uint32_t* p, uint32_t (&r)[WPR]) {
    const typename RowVec<WPR>::type v = *reinterpret_cast<const typename RowVec<WPR>::type*>(p);
    const uint32_t* s = reinterpret_cast<const uint32_t*>(&v);
#pragma unroll
    for (int k = 0; k < WPR; ++k) r[k] = s[k];
}
template <int WPR>
__device__ __forceinline__ void st_row(uint32_t* p, const uint32_t (&r)[WPR]) {
    typename RowVec<WPR>::type v;
    uint32_t* s = reinterpret_cast<uint32_t*>(&v);
#pragma unroll
    for (int k = 0; k < WPR; ++k) s[k] = r[k];
    *reinterpret_cast<typename RowVec<WPR>::type*>(p) = v;
}

// shared-memory footprint of one block (bytes)
template <int L, int MODE>
__host__ __device__ constexpr size_t sweep_smem_bytes(int tpb) {
    using G = Geo<L>;
    const size_t tbl = tbl_in_smem(MODE) ? (size_t)G::BINS * ROW_SMEM_WORDS * 4 : (size_t)G::BINS * 4;
    const size_t tbl_al = (tbl + 15) & ~(size_t)15;
    const size_t lat = lat_streamed(MODE) ? 0 : (size_t)L * G::WPR * 4 * tpb;
    return tbl_al + lat;
}

template <int L, int MODE, bool MEAS>
__device__ __forceinline__ void resident_sweeps(uint32_t* __restrict__ lat, const int tpb, uint32_t& o,
                                                const uint32_t s0, const uint32_t s1, const SweepParams& prm,
                                                const uint32_t walker, const char* tbl_smem, const char* tbl_glob,
                                                uint32_t* hist) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            const int ym = (y + L - 1) & (L - 1), yp = (y + 1) & (L - 1);
            uint32_t up[WPR], cur[WPR], dn[WPR];
#pragma unroll
            for (int k = 0; k < WPR; ++k) {
                up[k] = lat[(ym * WPR + k) * tpb];
                cur[k] = lat[(y * WPR + k) * tpb];
                dn[k] = lat[(yp * WPR + k) * tpb];
            }
            process_row<L, MODE, MEAS>(up, cur, dn, o, (uint32_t)(y * (L / 4)), s, prm.iteration, walker, prm.key0,
                                       prm.key1, tbl_smem, tbl_glob, hist);
#pragma unroll
            for (int k = 0; k < WPR; ++k) lat[(y * WPR + k) * tpb] = cur[k];
        }
    }
}

template <int L, int MODE, bool MEAS, bool EXT = false>
__device__ __forceinline__ void streamed_sweeps(uint32_t* __restrict__ rows, const size_t row_stride, uint32_t& o,
                                                const uint32_t s0, const uint32_t s1, const SweepParams& prm,
                                                const uint32_t walker, const char* tbl_glob, uint32_t* hist,
                                                DeviateFeed* feed = nullptr, const bool store = true) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR;
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
        uint32_t first[WPR] = {}, up[WPR], cur[WPR], dn[WPR], pre[WPR] = {};
        ld_row<WPR>(rows + (size_t)(L - 1) * row_stride, up);   // row L-1, value of the previous sweep
        ld_row<WPR>(rows, cur);
        ld_row<WPR>(rows + row_stride, dn);
#pragma unroll 1
        for (int y = 0; y < L; ++y) {
            if (y + 2 < L) ld_row<WPR>(rows + (size_t)(y + 2) * row_stride, pre);   // prefetch one row ahead
            if (y == L - 1) {
#pragma unroll
                for (int k = 0; k < WPR; ++k) dn[k] = first[k];                     // row 0, already updated
            }
            process_row<L, MODE, MEAS, EXT>(up, cur, dn, o, (uint32_t)(y * (L / 4)), s, prm.iteration, walker,
                                            prm.key0, prm.key1, nullptr, tbl_glob, hist, feed);
            if (store) st_row<WPR>(rows + (size_t)y * row_stride, cur);   // store == false: a lane without a walker (pair kernel)
#pragma unroll
            for (int k = 0; k < WPR; ++k) {
                if (y == 0) first[k] = cur[k];
                up[k] = cur[k];
                cur[k] = dn[k];
                dn[k] = pre[k];
            }
        }
    }
}

template <int L, int MODE>
__global__ void sweep_kernel(const SweepParams prm) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, N = G::N, BINS = G::BINS;
    constexpr int RSW = tbl_in_smem(MODE) ? ROW_SMEM_WORDS : ROW_L1_WORDS;
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, tpb = blockDim.x;
    const int w = blockIdx.x * tpb + tid;
    const bool active = w < prm.W;

    // ---- shared memory: [table+bins | bins] [lattices]
    constexpr size_t TBL_WORDS = tbl_in_smem(MODE) ? (size_t)BINS * ROW_SMEM_WORDS : (size_t)BINS;
    constexpr size_t TBL_WORDS_AL = (TBL_WORDS + 3) & ~(size_t)3;
    uint32_t* const tbl_s = smem;
    uint32_t* const lat = smem + TBL_WORDS_AL + tid;   // this thread's column: lat[r * tpb]
    if (tbl_in_smem(MODE)) {
        for (int idx = tid; idx < BINS * ROW_SMEM_WORDS; idx += tpb) {
            const int j = idx / ROW_SMEM_WORDS, e = idx - j * ROW_SMEM_WORDS;
            tbl_s[idx] = e < 8 ? prm.table[j * 8 + e] : 0u;   // e == 8: histogram bin, e == 9: pad
        }
    } else {
        for (int idx = tid; idx < BINS; idx += tpb) tbl_s[idx] = 0u;
    }

    // ---- lattice into shared memory (unpacked to one word per row for L < 32)
    if (!lat_streamed(MODE)) {
        if (active) {
            if (L >= 32) {
                for (int y = 0; y < L; ++y) {
                    uint32_t r[WPR];
                    ld_row<WPR>(prm.spins + ((size_t)y * prm.W + w) * WPR, r);
#pragma unroll
                    for (int k = 0; k < WPR; ++k) lat[(y * WPR + k) * tpb] = r[k];
                }
            } else {
                constexpr int RPW = 32 / G::BITS;  // rows per packed word
                for (int t = 0; t < N / 32; ++t) {
                    const uint32_t word = prm.spins[(size_t)t * prm.W + w];
#pragma unroll
                    for (int q = 0; q < RPW; ++q) lat[(t * RPW + q) * tpb] = (word >> (q * G::BITS)) & G::MASK;
                }
            }
        }
    }
    __syncthreads();

    if (active) {
        const int E = prm.E[w];
        const uint32_t o_base = tbl_in_smem(MODE) ? (uint32_t)__cvta_generic_to_shared(tbl_s) : 0u;
        uint32_t o = o_base + (uint32_t)((E + 2 * N) >> 2) * (uint32_t)(RSW * 4);   // slot j = (E + 2N)/4
        const uint32_t walker = prm.walker_offset + (uint32_t)w;
        const char* tbl_smem = reinterpret_cast<const char*>(tbl_s);
        const char* tbl_glob = reinterpret_cast<const char*>(prm.table);
        const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                              : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
        if (lat_streamed(MODE)) {
            uint32_t* rows = prm.spins + (size_t)w * WPR;
            const size_t row_stride = (size_t)prm.W * WPR;
            streamed_sweeps<L, MODE, false>(rows, row_stride, o, prm.sweep_begin, s_th, prm, walker, tbl_glob, tbl_s);
            streamed_sweeps<L, MODE, true>(rows, row_stride, o, s_th, prm.sweep_end, prm, walker, tbl_glob, tbl_s);
        } else {
            resident_sweeps<L, MODE, false>(lat, tpb, o, prm.sweep_begin, s_th, prm, walker, tbl_smem, tbl_glob, tbl_s);
            resident_sweeps<L, MODE, true>(lat, tpb, o, s_th, prm.sweep_end, prm, walker, tbl_smem, tbl_glob, tbl_s);
        }
        prm.E[w] = (int)((o - o_base) / (uint32_t)(RSW * 4)) * 4 - 2 * N;

        if (!lat_streamed(MODE)) {
            if (L >= 32) {
                for (int y = 0; y < L; ++y) {
                    uint32_t r[WPR];
#pragma unroll
                    for (int k = 0; k < WPR; ++k) r[k] = lat[(y * WPR + k) * tpb];
                    st_row<WPR>(prm.spins + ((size_t)y * prm.W + w) * WPR, r);
                }
            } else {
                constexpr int RPW = 32 / G::BITS;
                for (int t = 0; t < N / 32; ++t) {
                    uint32_t word = 0u;
#pragma unroll
                    for (int q = 0; q < RPW; ++q) word |= lat[(t * RPW + q) * tpb] << (q * G::BITS);
                    prm.spins[(size_t)t * prm.W + w] = word;
                }
            }
        }
    }
    __syncthreads();

    // ---- a4: merge the block's bins into the global uint64 histogram
    if (prm.sweep_end > prm.therm) {
        for (int j = tid; j < BINS; j += tpb) {
            const uint32_t v = tbl_in_smem(MODE) ? tbl_s[j * ROW_SMEM_WORDS + 8] : tbl_s[j];
            if (v) atomicAdd(prm.H + j, (unsigned long long)v);
        }
    }
}

}  // namespace muca
