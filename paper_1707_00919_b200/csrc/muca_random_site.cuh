// paper_1707_00919_b200/csrc/muca_random_site.cuh
// The paper's own update scheme: every update proposes the SAME random
// site in all walkers (one shared Philox stream), the acceptance deviate comes from a stream of the walker's own.
// DESIGN.md R22: update u of iteration n proposes site i_u = word (u & 3) of Philox(ctr = (u >> 2 mod 2^32, u >> 34,
// n, 0xFFFFFFFF), key) mod N; global walker g accepts iff word (u & 3) of Philox(ctr = (u >> 2 mod 2^32, u >> 34, n, g),
// key) <= thresh[j][a].  Work is counted in updates (attempted flips per walker), the paper's own unit.
// One thread per walker.  Shared memory (L <= 64): the threshold table as rows of 5 words thresh[j][a] (odd stride:
// consecutive rows rotate through all banks), the bins, the lattice words (lat[word * tpb + tid]: the site is
// warp-uniform, so every lattice access is conflict-free -- the paper's coalescing argument) and, for the
// next RS_CHUNK updates, a DESCRIPTOR of the update that the block computes once for all its walkers: the shared site
// stream (one Philox call gives four sites) turned into the five (word offset, bit) pairs of the site and its
// neighbours, plus a flag saying whether the update touches the word the update before may have changed.  So a thread
// does no index arithmetic at all, and -- the sites of successive updates being the same for all walkers and rarely
// adjacent -- it fetches the neighbourhood of update u + 1 BEFORE it decides update u unless that flag is set (a
// warp-uniform branch): the per-update chain is   j -> LDS thresh[j][a] -> compare -> j'   as in the typewriter kernels.
// The acceptance deviates come from one Philox call per four updates in the walker's thread.  At L = 128 the table
// (320 KB) does not fit: thresholds are read through L1 there.
#pragma once
#include "muca_device.cuh"

namespace muca {

struct RandomSiteParams {
    uint32_t* spins;
    int32_t* E;
    const uint32_t* table;          // T8 (muca_device.cuh)
    unsigned long long* H;
    int W;
    uint32_t walker_offset, key0, key1, iteration;
    unsigned long long u_begin, u_end, therm;   // updates [u_begin, u_end); updates with index < therm are not recorded
};

constexpr int RS_CHUNK = 256;     // updates described ahead, per block

// ACC: how a proposal is decided.  0 = integer thresholds thresh[j][a] (R6/R7, the library's own form); 1 = the paper's
// single-precision form U < exp32(omega_f[j'] - omega_f[j]) (R23), with omega_f as BINS floats in
// shared memory for every L.
enum { RS_ACC_THRESHOLD = 0, RS_ACC_EXPF32 = 1 };

// R23: the Philox word mapped to (0, 1] as cuRAND's curand_uniform does, and exp for arguments <= 0 as a fixed sequence
// of IEEE fp32 operations (the paper's requirement of identical results on CPU and GPU; restated, not
// shared, by the CPU implementation the tests compare with)
__device__ __forceinline__ float rs_uniform32(const uint32_t x) {
    return __fmaf_rn(__uint2float_rn(x), 2.3283064365386963e-10f, 1.1641532182693481e-10f);
}
__device__ __forceinline__ float rs_exp32(const float d) {
    if (d < -24.0f) return 0.0f;                                 // exp(-24) < 2^-33 <= U: never accepted
    const int n = __float2int_rn(__fmul_rn(d, 1.4426950408889634f));
    const float fn = __int2float_rn(n);
    float r = __fmaf_rn(fn, -0.693145751953125f, d);
    r = __fmaf_rn(fn, -1.428606765330187e-06f, r);
    float p = 1.0f / 720.0f;
    p = __fmaf_rn(p, r, 1.0f / 120.0f);
    p = __fmaf_rn(p, r, 1.0f / 24.0f);
    p = __fmaf_rn(p, r, 1.0f / 6.0f);
    p = __fmaf_rn(p, r, 0.5f);
    p = __fmaf_rn(p, r, 1.0f);
    p = __fmaf_rn(p, r, 1.0f);
    return __fmul_rn(p, __int_as_float((n + 127) << 23));
}

template <int L, int ACC = RS_ACC_THRESHOLD>
struct RandomSite {
    static constexpr int N = L * L, BINS = N + 1, NW = N / 32;
    static constexpr bool TBL_SMEM = L <= 64 || ACC == RS_ACC_EXPF32;
    // L <= 32: rows of thresh[j][0..4] | bin of slot j | pad (7 words, odd stride: all banks): threshold and bin are one
    // add away from the row address.  L = 64: rows of 5 thresholds and the bins apart (beside 208 walkers' lattices a
    // 7-word table would not fit).  L = 128: bins only.
    static constexpr bool BIN_IN_ROW = L <= 32 && ACC == RS_ACC_THRESHOLD;
    static constexpr int ROW_WORDS = ACC == RS_ACC_EXPF32 ? 1 : (BIN_IN_ROW ? 7 : 5);
    static constexpr int TBL_WORDS = TBL_SMEM ? ((BINS * ROW_WORDS + 3) & ~3) : 0;
    static constexpr int BIN_WORDS = BIN_IN_ROW ? 0 : ((BINS + 3) & ~3);
    static constexpr int DESC_WORDS = 8 * (RS_CHUNK + 2);      // two uint4 per update + two entries behind the chunk
    static constexpr int SITE_WORDS = RS_CHUNK + 4;            // the sites of the chunk, [0] = last site of the chunk before
    __host__ __device__ static constexpr size_t smem_bytes(int tpb) {
        return ((size_t)TBL_WORDS + BIN_WORDS + DESC_WORDS + SITE_WORDS + (size_t)NW * tpb) * 4;
    }
};

// The five lattice words of an update as loaded (RsWords) and what the decision needs from them (RsHood).  Loading and
// evaluating are two steps so that the threshold load of the update before can be issued between them: a warp issues
// in order, and the evaluation would otherwise wait for the words in front of that load.
struct RsWords { uint32_t wc, wr, wl, wd, wu; };
struct RsHood { uint32_t a, wc, addr_c, mask; };   // mask: bit of the site in its word (from the descriptor)

// descriptor word p = (byte offset of the lattice word in this thread's column << 5) | bit
template <int L>
__device__ __forceinline__ RsWords rs_load(const char* lat, const uint4 d0, const uint4 d1) {
    RsWords r;
    r.wc = *reinterpret_cast<const volatile uint32_t*>(lat + (d0.x >> 5));
    if constexpr (L <= 32) {   // a row lies within one word: left and right neighbour are bits of the site's own word
        r.wr = r.wc; r.wl = r.wc;
    } else {
        r.wr = *reinterpret_cast<const volatile uint32_t*>(lat + (d0.y >> 5));
        r.wl = *reinterpret_cast<const volatile uint32_t*>(lat + (d0.z >> 5));
    }
    r.wd = *reinterpret_cast<const volatile uint32_t*>(lat + (d0.w >> 5));
    r.wu = *reinterpret_cast<const volatile uint32_t*>(lat + (d1.x >> 5));
    return r;
}
__device__ __forceinline__ RsHood rs_eval(const RsWords& r, const uint4 d0, const uint4 d1) {
    const uint32_t s = __funnelshift_r(r.wc, r.wc, d0.x);       // rotate by the low 5 bits: bit 0 = the spin
    RsHood h;
    h.a = ((__funnelshift_r(r.wr, r.wr, d0.y) ^ s) & 1u) + ((__funnelshift_r(r.wl, r.wl, d0.z) ^ s) & 1u) +
          ((__funnelshift_r(r.wd, r.wd, d0.w) ^ s) & 1u) + ((__funnelshift_r(r.wu, r.wu, d1.x) ^ s) & 1u);   // antiparallel neighbours
    h.wc = r.wc;
    h.addr_c = d0.x >> 5;
    h.mask = d1.z;
    return h;
}

// Updates k .. k + 3 of the chunk (one acceptance call).  MEAS: 0 = none of the four is recorded, 1 = all are,
// 2 = the group straddles the begin / end of the launch or the end of the thermalisation (k0, k1, kth decide per update).
// In: cur = neighbourhood of update k, (d0, d1) = descriptor of update k + 1.  Per update: the words of the NEXT update
// are loaded at once, then the threshold of this one, then the descriptor of the update after the next; only then is
// anything evaluated -- three independent loads in flight, one round trip per update.  If the next update touches the
// word this one may change (flag in its descriptor, warp-uniform, ~5 / number of words of the time) its words are
// loaded again behind the store.
template <int L, int MEAS, int ACC>
__device__ __forceinline__ void rs_group(char* lat, const uint4* desc, const uint32_t* tbl, uint32_t* bins, const RandomSiteParams& prm,
                                         const int k, const int k0, const int k1, const int kth, const uint32_t (&ra)[4], int& j, RsHood& cur,
                                         uint4& d0, uint4& d1, uint32_t (&st)[4]) {
    constexpr bool TBL_SMEM = RandomSite<L, ACC>::TBL_SMEM, BIN_IN_ROW = RandomSite<L, ACC>::BIN_IN_ROW;
    constexpr int N = L * L;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        RsWords nw = rs_load<L>(lat, d0, d1);
        // the acceptance call of the NEXT four updates, 3 + 2 + 3 + 2 of its ten rounds per update, behind the loads: a call
        // is one dependent chain of wide multiplies, which a warp that issues in order cannot hide when it comes as a block
#pragma unroll
        for (int r = (m >> 1) * 5 + (m & 1) * 3; r < (m >> 1) * 5 + (m & 1) * 3 + ((m & 1) ? 2 : 3); ++r)
            philox_round(st, prm.key0 + (uint32_t)r * 0x9E3779B9u, prm.key1 + (uint32_t)r * 0xBB67AE85u);
        const bool live = MEAS != 2 || (k + m >= k0 && k + m < k1);
        uint32_t t = 0u;   // BIN_IN_ROW: j is the BYTE offset of the walker's table row (28 j), so that threshold and bin need one add
        float w_here = 0.0f, w_there = 0.0f;
        const int jn = j + 2 - (int)cur.a;                      // ACC = 1: j is the slot itself
        if constexpr (ACC == RS_ACC_EXPF32) {
            if (live) {
                w_here = __uint_as_float(*reinterpret_cast<const volatile uint32_t*>(tbl + j));
                w_there = __uint_as_float(*reinterpret_cast<const volatile uint32_t*>(tbl + (jn < 0 ? 0 : jn > N ? N : jn)));
            }
        } else {
            if (live) t = BIN_IN_ROW ? *reinterpret_cast<const volatile uint32_t*>(reinterpret_cast<const char*>(tbl) + j + 4 * (int)cur.a)
                        : TBL_SMEM ? *reinterpret_cast<const volatile uint32_t*>(tbl + 5 * j + (int)cur.a)
                                   : __ldg(prm.table + (size_t)j * 8 + (cur.a ? 2u * cur.a - 1u : 0u));
        }
        const uint4 e0 = desc[2 * (k + m) + 4], e1 = desc[2 * (k + m) + 5];   // descriptor of update k + m + 2 (two dummies behind the chunk)
        RsHood nxt = rs_eval(nw, d0, d1);
        if (live) {
            bool accept;
            if constexpr (ACC == RS_ACC_EXPF32) {                            // R23
                const float D = __fsub_rn(w_there, w_here);
                accept = cur.a == 2u || (jn >= 0 && jn <= N && (D >= 0.0f || rs_uniform32(ra[m]) < rs_exp32(D)));
            } else {
                accept = ra[m] <= t;                                         // R6/R7
            }
            if (accept) {
                *reinterpret_cast<volatile uint32_t*>(lat + cur.addr_c) = cur.wc ^ cur.mask;
                j += (BIN_IN_ROW ? 4 * RandomSite<L, ACC>::ROW_WORDS : 1) * (2 - (int)cur.a);   // dE = 8 - 4a
            }
            if (MEAS == 1 || (MEAS == 2 && k + m >= kth))                    // H[j]++ after EVERY measured attempt
                atomicAdd(BIN_IN_ROW ? reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(bins) + j + 20) : bins + j, 1u);
        }
        if (d1.y != 0u) {                                                    // warp-uniform
            nw = rs_load<L>(lat, d0, d1);
            nxt = rs_eval(nw, d0, d1);
        }
        cur = nxt; d0 = e0; d1 = e1;
    }
}

template <int L, int ACC>
__global__ void random_site_kernel(const RandomSiteParams prm) {
    using R = RandomSite<L, ACC>;
    constexpr int N = R::N, BINS = R::BINS, NW = R::NW;
    constexpr int LOG_L = L == 8 ? 3 : L == 16 ? 4 : L == 32 ? 5 : L == 64 ? 6 : 7;
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, tpb = blockDim.x;
    const int w = blockIdx.x * tpb + tid;
    const bool active = w < prm.W;
    uint32_t* const tbl = smem;                                 // row j: thresh[j][0..4] | bin | pad
    uint32_t* const bins = R::BIN_IN_ROW ? smem : smem + R::TBL_WORDS;   // BIN_IN_ROW: bin of slot j at tbl[7 j + 5]
    uint4* const desc = reinterpret_cast<uint4*>(smem + R::TBL_WORDS + R::BIN_WORDS);
    uint32_t* const sites = smem + R::TBL_WORDS + R::BIN_WORDS + R::DESC_WORDS;
    uint32_t* const latw = sites + R::SITE_WORDS + tid;         // typewriter word t of this walker at latw[t * tpb]
    char* const lat = reinterpret_cast<char*>(latw);
    if (ACC == RS_ACC_EXPF32) {
        for (int j = tid; j < BINS; j += tpb) tbl[j] = prm.table[j];       // omega_f[j] (float bits; the host rounded omega)
    } else if (R::TBL_SMEM) {
        for (int idx = tid; idx < BINS * R::ROW_WORDS; idx += tpb) {
            const int j = idx / R::ROW_WORDS, a = idx - R::ROW_WORDS * j;
            tbl[idx] = a < 5 ? prm.table[j * 8 + (a ? 2 * a - 1 : 0)] : 0u;   // a column of T8 with a(f) = a; bin and pad: 0
        }
    }
    if (!R::BIN_IN_ROW)
        for (int j = tid; j < BINS; j += tpb) bins[j] = 0u;
    if (tid == 0) {
        sites[0] = 0xFFFFFFFFu;                                 // no update before the first one of this launch
        for (int e = 0; e < 2; ++e) {                           // the entries behind the chunk: word 0, "load again"
            desc[2 * (RS_CHUNK + e)] = make_uint4(0u, 0u, 0u, 0u);
            desc[2 * (RS_CHUNK + e) + 1] = make_uint4(0u, 1u, 0u, 0u);
        }
    }
    if (active)
        for (int t = 0; t < NW; ++t) latw[t * tpb] = prm.spins[word_index(L, prm.W, w, t)];
    constexpr int JS = R::BIN_IN_ROW ? 4 * R::ROW_WORDS : 1;   // j is kept times JS (rs_group)
    int j = active ? ((prm.E[w] + 2 * N) >> 2) * JS : 0;       // slot
    const uint32_t g = prm.walker_offset + (uint32_t)w;
    for (unsigned long long u0 = prm.u_begin & ~3ull; u0 < prm.u_end; u0 += RS_CHUNK) {   // chunks start at a multiple of 4
        __syncthreads();                                        // the descriptors of the chunk before have been used
        for (int c = tid; c < RS_CHUNK / 4; c += tpb) {         // site stream, shared by all walkers (R22): one call gives 4 sites
            const unsigned long long uc = u0 + 4ull * c;
            uint32_t rs[4];
            philox4x32_10((uint32_t)((uc >> 2) & 0xFFFFFFFFull), (uint32_t)(uc >> 34), prm.iteration, 0xFFFFFFFFu, prm.key0, prm.key1, rs);
#pragma unroll
            for (int m = 0; m < 4; ++m) sites[1 + 4 * c + m] = rs[m] & (uint32_t)(N - 1);   // mod N, N a power of two
        }
        __syncthreads();
        for (int k = tid; k < RS_CHUNK; k += tpb) {             // descriptors
            const int i = (int)sites[1 + k];
            const int x = i & (L - 1), y = i >> LOG_L;
            const int ir = y * L + ((x + 1) & (L - 1)), il = y * L + ((x + L - 1) & (L - 1));
            const int id = ((y + 1) & (L - 1)) * L + x, iu = ((y + L - 1) & (L - 1)) * L + x;
            auto pk = [&](int s) { return (uint32_t)(((s >> 5) * tpb * 4) << 5) | (uint32_t)(s & 31); };
            const uint32_t prev = sites[k];                     // the site of the update before (0xFFFFFFFF: none)
            const uint32_t pw = prev >> 5;                      // the word it may have changed
            const bool hazard = prev == 0xFFFFFFFFu || pw == (uint32_t)(i >> 5) || pw == (uint32_t)(ir >> 5) || pw == (uint32_t)(il >> 5) ||
                                pw == (uint32_t)(id >> 5) || pw == (uint32_t)(iu >> 5);
            desc[2 * k] = make_uint4(pk(i), pk(ir), pk(il), pk(id));
            desc[2 * k + 1] = make_uint4(pk(iu), hazard ? 1u : 0u, 1u << (i & 31), 0u);
        }
        __syncthreads();
        if (tid == 0) sites[0] = sites[RS_CHUNK];               // read again only behind the next barrier
        if (!active) continue;
        // the chunk in 32-bit numbers: updates k0 .. k1-1 of it belong to this launch, those from kth on are recorded
        const int k0 = prm.u_begin > u0 ? (int)(prm.u_begin - u0) : 0;
        const int k1 = prm.u_end - u0 < (unsigned long long)RS_CHUNK ? (int)(prm.u_end - u0) : RS_CHUNK;
        const int kth = prm.therm <= u0 ? 0 : (prm.therm - u0 < (unsigned long long)RS_CHUNK ? (int)(prm.therm - u0) : RS_CHUNK);
        RsHood cur = rs_eval(rs_load<L>(lat, desc[0], desc[1]), desc[0], desc[1]);   // the first update of a chunk: fetched behind the store before it
        uint4 d0 = desc[2], d1 = desc[3];
        // acceptance stream of this walker (R22): one call per four updates; the call of the first group of the chunk here,
        // the call of every further group inside the group before it (rs_group)
        uint32_t st[4];
        philox4x32_10((uint32_t)((u0 >> 2) & 0xFFFFFFFFull), (uint32_t)(u0 >> 34), prm.iteration, g, prm.key0, prm.key1, st);
        for (int k = 0; k < k1; k += 4) {
            const uint32_t ra[4] = {st[0], st[1], st[2], st[3]};
            const unsigned long long un = u0 + (unsigned long long)k + 4ull;   // counter of the next group
            st[0] = (uint32_t)((un >> 2) & 0xFFFFFFFFull); st[1] = (uint32_t)(un >> 34); st[2] = prm.iteration; st[3] = g;
            if (k >= k0 && k + 4 <= k1 && k >= kth) rs_group<L, 1, ACC>(lat, desc, tbl, bins, prm, k, k0, k1, kth, ra, j, cur, d0, d1, st);
            else if (k >= k0 && k + 4 <= k1 && k + 4 <= kth) rs_group<L, 0, ACC>(lat, desc, tbl, bins, prm, k, k0, k1, kth, ra, j, cur, d0, d1, st);
            else rs_group<L, 2, ACC>(lat, desc, tbl, bins, prm, k, k0, k1, kth, ra, j, cur, d0, d1, st);
        }
    }
    if (active) {
        prm.E[w] = 4 * (j / JS) - 2 * N;
        for (int t = 0; t < NW; ++t) prm.spins[word_index(L, prm.W, w, t)] = latw[t * tpb];
    }
    __syncthreads();
    if (prm.u_end > prm.therm)
        for (int jj = tid; jj < BINS; jj += tpb) {
            const uint32_t v = R::BIN_IN_ROW ? tbl[jj * R::ROW_WORDS + 5] : bins[jj];
            if (v) atomicAdd(prm.H + jj, (unsigned long long)v);
        }
}

template <int L, int ACC>
__host__ __device__ constexpr size_t random_site_smem_bytes(int tpb) {
    return RandomSite<L, ACC>::smem_bytes(tpb);
}

}  // namespace muca
