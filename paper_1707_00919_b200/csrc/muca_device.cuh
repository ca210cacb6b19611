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
// a2/a3/a4 -- the sweep kernels.
//
// Device threshold table "T8" (built on the host from omega, muca.cu): row j holds 8 words indexed by
//   f = 4*hi + 2*lo + g,   n3 = lo + 2*hi = antiparallel count over {up, down, right},  g = [left antiparallel],
//   T8[j][f] = thresh[j][a = n3 + g]     (PAPER.md:109 acceptance, R6/R7 integer form).
// The left neighbour is the site visited just before (typewriter order, R3), so g = hl ^ D where hl is the
// static bit (old left value) and D says whether the previous site flipped: the lookup column is f_static ^ D --
// one XOR on the serial chain instead of a recount.
//
// Kernels: sweep_kernel_v6 (muca_resident.cuh; L <= 32: table, histogram and lattices in shared memory),
// sweep_kernel_s6 (muca_streamed.cuh; L >= 32: table or a window of it and the histogram in shared memory, lattice
// rows streamed) and sweep_kernel_l1 below (L >= 32: table read through L1, histogram in shared memory, lattice rows
// streamed): the plain one, which needs no table in shared memory and therefore serves as the fallback of the
// windowed kernel at L = 128.
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
    int* check;                 // device word the violations are OR-ed into (CHK_SMEM_BASE in every build, the rest MUCA_CHECKED)
    uint32_t fault;             // MUCA_CHECKED build, tests: 1 + the hand-over that pair 0 of block 0 tags wrongly; 0 = none
};

// ------------------------------------------------------------------------------------------------
// Self-checks of the MUCA_CHECKED build (libmuca_b200_checked.so; paper_1707_00919_b200/build.py).  compute-sanitizer
// is not available on the GPU pool this library is developed on (profiles/r02_sanitizer.txt), so the two things its
// racecheck / memcheck tools would watch in these kernels are checked by the kernels themselves:
//  * the hand-over of deviates from a deviate warp to its walker warp through the double-buffered shared ring (named
//    barriers): the deviate warp tags every buffer it fills with a running number, the walker warp compares the tag with
//    its own count when it starts to fetch from a buffer (CHK_RING_EARLY: read before written) and when it has fetched
//    the last call (CHK_RING_LATE: overwritten while being read);
//  * the shared-memory address that IS the walker's state (every table load and histogram increment is relative to
//    it): after every row it must be the address of a table row (CHK_STATE).
// A violation sets a bit in a device word; muca_run_iteration then fails with MUCA_ECUDA.  In the normal build all of
// this compiles to nothing.
// ------------------------------------------------------------------------------------------------
enum { CHK_STATE = 1, CHK_RING_EARLY = 2, CHK_RING_LATE = 4, CHK_SMEM_BASE = 8 };
struct RingCheck {
#ifdef MUCA_CHECKED
    uint32_t ctr = 0;                     // hand-overs so far (deviate warp: published, walker warp: fetched)
    volatile uint32_t* tags = nullptr;    // tags[buf * stride]: number of the hand-over whose deviates are in ring[buf]
    int stride = 1;
    int* flag = nullptr;
    uint32_t fault = 0;
#endif
};
__device__ __forceinline__ void ring_publish(RingCheck& rc, const int buf, const int lane) {   // deviate warp, in front of the barrier
#ifdef MUCA_CHECKED
    if (lane == 0) rc.tags[buf * rc.stride] = rc.ctr + (rc.fault == rc.ctr + 1u ? 1u : 0u);
    rc.ctr += 1u;
#endif
}
__device__ __forceinline__ void ring_expect(RingCheck& rc, const int buf, const int code) {    // walker warp, behind the barrier
#ifdef MUCA_CHECKED
    if (rc.tags[buf * rc.stride] != rc.ctr) atomicOr(rc.flag, code);
#endif
}
__device__ __forceinline__ void ring_fetched(RingCheck& rc, const int buf) {                   // walker warp: last call of a buffer fetched
#ifdef MUCA_CHECKED
    ring_expect(rc, buf, CHK_RING_LATE);
    rc.ctr += 1u;
#endif
}
__device__ __forceinline__ void state_check(RingCheck& rc, const bool ok) {
#ifdef MUCA_CHECKED
    if (!ok) atomicOr(rc.flag, CHK_STATE);
#endif
}

// Checked in EVERY build: the site macros of the paired kernels address the delta table by an immediate, so the dynamic
// shared memory must start at the offset they were written for (the driver's reserved area, no static __shared__ in
// front).  Where it does not, the block sets CHK_SMEM_BASE and returns before touching anything, and muca_run_iteration
// fails with MUCA_ECUDA -- an ordinary error the caller can handle.  (A __trap() here would leave a sticky error behind
// that takes the caller's whole CUDA context down, torch's included.)  The condition is the same for every thread of
// the launch.  MUCA_CHECKED build, tests: prm.fault = 0xFFFFFFFF pretends a mismatch.
__device__ __forceinline__ bool smem_base_ok(const SweepParams& prm, const uint32_t base, const uint32_t expected) {
    bool ok = base == expected;
#ifdef MUCA_CHECKED
    if (prm.fault == 0xFFFFFFFFu) ok = false;
#endif
    if (!ok && threadIdx.x == 0) atomicOr(prm.check, CHK_SMEM_BASE);
    return ok;
}

template <int L>
struct Geo {
    static constexpr int N = L * L;
    static constexpr int BINS = N + 1;
    static constexpr int WPR = L >= 32 ? L / 32 : 1;   // words per row
    static constexpr int BITS = L >= 32 ? 32 : L;      // valid bits per row word
    static constexpr uint32_t MASK = L >= 32 ? 0xFFFFFFFFu : ((1u << (L & 31)) - 1u);
};

constexpr int ROW_L1_WORDS = 8;     // T8 row in global memory: 8 thresholds (32 B)

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

// One typewriter pass over row y of one walker (sweep_kernel_l1).  up/dn: rows above/below (current values), cur: the
// row, updated in place.  o: byte offset of the walker's energy row in T8 (= j * 32), updated.
//
// Per row (bit-sliced, ~30 instructions for 32 sites): the three static planes
//   lo, hi = the two bits of n3 = [up != s] + [down != s] + [right != s],   hl = [left(old) != s]
// are interleaved into four "field words" FW[r] (r = x & 3): nibble q of FW[r] holds the table column
// f = hl + 2*lo + 4*hi of site x = 4q + r, so the per-site extraction is one shift and one mask.
// Per site the serial chain is  D(prev) -> f ^= D -> address -> LDG -> compare -> D:
//   fw   = f ^ D                     D: previous site flipped, which toggles the [left != s] bit (column f ^ 1)
//   t    = T8[row o][fw]             one 4-byte load through L1
//   D    = r <= t                    R6/R7
//   o   += D ? 32*(2 - a(fw)) : 0    32*a(fw) comes from an 8-entry byte table in two registers (PRMT)
//   s_x ^= D
//   H[row o] += 1                    shared-memory atomic, measured sweeps only
template <int L, bool MEAS>
__device__ __forceinline__ void process_row(const uint32_t (&up)[Geo<L>::WPR], uint32_t (&cur)[Geo<L>::WPR],
                                            const uint32_t (&dn)[Geo<L>::WPR], uint32_t& o,
                                            const uint32_t ctr0_row, const uint32_t sweep, const uint32_t iteration,
                                            const uint32_t walker, const uint32_t key0, const uint32_t key1,
                                            const char* __restrict__ tbl_glob, uint32_t* __restrict__ hist) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, BITS = G::BITS;
    constexpr uint32_t RS = ROW_L1_WORDS * 4;  // row stride in bytes
    // byte f of (LUT_HI:LUT_LO) = RS * a(f), a(f) = (f >> 1) + (f & 1) = antiparallel neighbours of column f
    constexpr uint32_t LUT_LO = (RS * 0) | (RS * 1) << 8 | (RS * 1) << 16 | (RS * 2) << 24;
    constexpr uint32_t LUT_HI = (RS * 2) | (RS * 3) << 8 | (RS * 3) << 16 | (RS * 4) << 24;
    static_assert(RS * 4 < 256, "row stride must keep RS*a in a byte");

    uint32_t FW[WPR][4];
    uint32_t patch = 0;   // added to FW[WPR-1][3] when site 0 flips: n3 of the LAST site changes by +-1
#pragma unroll
    for (int k = 0; k < WPR; ++k) {
        const uint32_t c = cur[k];
        const uint32_t rw = (c >> 1) | (cur[(k + 1) % WPR] << 31);          // right neighbours (old; last site patched)
        const uint32_t lw = (c << 1) | (cur[(k + WPR - 1) % WPR] >> 31);    // left neighbours (old)
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

template <int L, bool MEAS>
__device__ __forceinline__ void streamed_sweeps(uint32_t* __restrict__ rows, const size_t row_stride, uint32_t& o,
                                                const uint32_t s0, const uint32_t s1, const SweepParams& prm,
                                                const uint32_t walker, const char* tbl_glob, uint32_t* hist) {
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
            process_row<L, MEAS>(up, cur, dn, o, (uint32_t)(y * (L / 4)), s, prm.iteration, walker, prm.key0, prm.key1, tbl_glob, hist);
            st_row<WPR>(rows + (size_t)y * row_stride, cur);
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

// shared-memory footprint of one block of sweep_kernel_l1 (bytes): the uint32 bins
template <int L>
__host__ __device__ constexpr size_t l1_smem_bytes() {
    return ((size_t)Geo<L>::BINS * 4 + 15) & ~(size_t)15;
}

// L >= 32: one thread per walker, Philox in the walker thread, thresholds through L1, a three-row register window
// over the streamed lattice rows (one vector load per row one row ahead, one store per row).
template <int L>
__global__ void sweep_kernel_l1(const SweepParams prm) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, N = G::N, BINS = G::BINS;
    static_assert(L >= 32, "streamed rows are whole 32-site words");
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, tpb = blockDim.x;
    const int w = blockIdx.x * tpb + tid;
    for (int idx = tid; idx < BINS; idx += tpb) smem[idx] = 0u;
    __syncthreads();
    if (w < prm.W) {
        uint32_t o = (uint32_t)((prm.E[w] + 2 * N) >> 2) * (uint32_t)(ROW_L1_WORDS * 4);   // slot j = (E + 2N)/4
        const uint32_t walker = prm.walker_offset + (uint32_t)w;
        const char* tbl_glob = reinterpret_cast<const char*>(prm.table);
        const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                              : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
        uint32_t* rows = prm.spins + (size_t)w * WPR;
        const size_t row_stride = (size_t)prm.W * WPR;
        streamed_sweeps<L, false>(rows, row_stride, o, prm.sweep_begin, s_th, prm, walker, tbl_glob, smem);
        streamed_sweeps<L, true>(rows, row_stride, o, s_th, prm.sweep_end, prm, walker, tbl_glob, smem);
        prm.E[w] = (int)(o / (uint32_t)(ROW_L1_WORDS * 4)) * 4 - 2 * N;
    }
    __syncthreads();
    // ---- a4: merge the block's bins into the global uint64 histogram
    if (prm.sweep_end > prm.therm) {
        for (int j = tid; j < BINS; j += tpb) {
            const uint32_t v = smem[j];
            if (v) atomicAdd(prm.H + j, (unsigned long long)v);
        }
    }
}

// smallest and largest energy slot of the walkers (host picks the window from them)
__global__ void slot_range_kernel(const int32_t* __restrict__ E, int W, int N, int* __restrict__ range) {
    int lo = 0x7FFFFFFF, hi = -1;
    for (int w = blockIdx.x * blockDim.x + threadIdx.x; w < W; w += gridDim.x * blockDim.x) {
        const int j = (E[w] + 2 * N) >> 2;
        lo = min(lo, j); hi = max(hi, j);
    }
    for (int d = 16; d > 0; d >>= 1) {
        lo = min(lo, __shfl_xor_sync(0xFFFFFFFFu, lo, d));
        hi = max(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, d));
    }
    if ((threadIdx.x & 31) == 0) { atomicMin(range, lo); atomicMax(range + 1, hi); }
}

}  // namespace muca
