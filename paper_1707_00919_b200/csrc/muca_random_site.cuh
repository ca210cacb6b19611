// paper_1707_00919_b200/csrc/muca_random_site.cuh
// The paper's own update scheme: every update proposes the SAME random
// site in all walkers (one shared Philox stream), the acceptance deviate comes from a stream of the walker's own.
// DESIGN.md R22: update u of iteration n proposes site i_u = word (u & 3) of Philox(ctr = (u >> 2 mod 2^32, u >> 34,
// n, 0xFFFFFFFF), key) mod N; global walker g accepts iff word (u & 3) of Philox(ctr = (u >> 2 mod 2^32, u >> 34, n, g),
// key) <= thresh[j][a].  Work is counted in updates (attempted flips per walker), the paper's own unit.
// Straightforward kernel (not the tuned path): one thread per walker, lattice words and bins in shared memory
// (lat[word * tpb + tid]: the site is warp-uniform, so every access is conflict-free -- the paper's coalescing
// argument), thresholds through L1, Philox in the thread.
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

template <int L>
__global__ void random_site_kernel(const RandomSiteParams prm) {
    constexpr int N = L * L, BINS = N + 1, NW = N / 32;
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, tpb = blockDim.x;
    const int w = blockIdx.x * tpb + tid;
    const bool active = w < prm.W;
    uint32_t* const bins = smem;
    uint32_t* const lat = smem + ((BINS + 3) & ~3) + tid;      // typewriter word t of this walker at lat[t * tpb]
    for (int j = tid; j < BINS; j += tpb) bins[j] = 0u;
    if (active)
        for (int t = 0; t < NW; ++t) lat[t * tpb] = prm.spins[word_index(L, prm.W, w, t)];
    __syncthreads();
    if (active) {
        int j = (prm.E[w] + 2 * N) >> 2;                       // slot
        const uint32_t g = prm.walker_offset + (uint32_t)w;
        uint32_t rs[4] = {0, 0, 0, 0}, ra[4] = {0, 0, 0, 0};
        for (unsigned long long u = prm.u_begin; u < prm.u_end; ++u) {
            if ((u & 3ull) == 0ull || u == prm.u_begin) {
                const uint32_t c0 = (uint32_t)((u >> 2) & 0xFFFFFFFFull), c1 = (uint32_t)(u >> 34);
                philox4x32_10(c0, c1, prm.iteration, 0xFFFFFFFFu, prm.key0, prm.key1, rs);   // site stream, shared by all walkers
                philox4x32_10(c0, c1, prm.iteration, g, prm.key0, prm.key1, ra);             // acceptance stream of this walker
            }
            const int i = (int)(rs[u & 3ull] & (uint32_t)(N - 1));   // mod N, N a power of two
            const int x = i & (L - 1), y = i / L;
            const int ir = y * L + ((x + 1) & (L - 1)), il = y * L + ((x + L - 1) & (L - 1));
            const int id = ((y + 1) & (L - 1)) * L + x, iu = ((y + L - 1) & (L - 1)) * L + x;
            const uint32_t wc = lat[(i >> 5) * tpb];
            const uint32_t s = (wc >> (i & 31)) & 1u;
            const uint32_t a = (((lat[(ir >> 5) * tpb] >> (ir & 31)) & 1u) ^ s) + (((lat[(il >> 5) * tpb] >> (il & 31)) & 1u) ^ s) +
                               (((lat[(id >> 5) * tpb] >> (id & 31)) & 1u) ^ s) + (((lat[(iu >> 5) * tpb] >> (iu & 31)) & 1u) ^ s);
            const uint32_t f = a ? 2u * a - 1u : 0u;             // a column of T8 with a(f) = a
            const uint32_t t = __ldg(prm.table + (size_t)j * 8 + f);
            if (ra[u & 3ull] <= t) {                             // R6/R7
                lat[(i >> 5) * tpb] = wc ^ (1u << (i & 31));
                j += 2 - (int)a;                                 // dE = 8 - 4a
            }
            if (u >= prm.therm) atomicAdd(bins + j, 1u);        // H[j]++ after EVERY measured attempt
        }
        prm.E[w] = 4 * j - 2 * N;
        for (int t = 0; t < NW; ++t) prm.spins[word_index(L, prm.W, w, t)] = lat[t * tpb];
    }
    __syncthreads();
    if (prm.u_end > prm.therm)
        for (int j = tid; j < BINS; j += tpb)
            if (bins[j]) atomicAdd(prm.H + j, (unsigned long long)bins[j]);
}

template <int L>
__host__ __device__ constexpr size_t random_site_smem_bytes(int tpb) {
    return ((size_t)((L * L + 1 + 3) & ~3) + (size_t)(L * L / 32) * tpb) * 4;
}

}  // namespace muca
