// paper_1707_00919_b200/csrc/muca_window.cuh
// Sweep kernel for lattices whose threshold table does not fit in shared memory (L = 128: 16385 rows): the lattice
// rows are streamed as in sweep_kernel<L, STREAMED> and shared memory holds a WINDOW of the table, rows
// [j_lo, j_lo + n_rows), around the energies the walkers have at the start of the iteration -- a shared-memory
// threshold load on the per-site chain (27 cycles) instead of a divergent L1 load (61, profiles/README.md).
// A walker may leave the window during the iteration.  That cannot be excluded beforehand, so it is DETECTED and
// the host repeats the iteration with the L1 kernel from a snapshot (muca.cu): the two outermost rows on a side
// that is not the end of the real table are sentinels with all thresholds 0 -- a walker that enters one cannot
// move on (up to an r = 0 deviate, probability 2^-32 per attempt, which two zeroed pad rows beyond absorb) -- and
// every sweep, thermalisation included, counts into the row's bin, so that a non-zero sentinel bin at the end of a
// phase says "the window was left" whatever happened afterwards.  Site code: process_row<L, STREAMED_SMEM>.
#pragma once
#include "muca_device.cuh"

namespace muca {

constexpr int WINDOW_PAD_ROWS = 2;   // zeroed rows before and behind the window

__host__ __device__ constexpr size_t window_smem_bytes(int n_rows) {
    return (size_t)(n_rows + 2 * WINDOW_PAD_ROWS) * ROW_SMEM_WORDS * 4;
}

template <int L>
__global__ void sweep_kernel_window(const SweepParams prm, const int j_lo, const int n_rows, const int sent_lo,
                                    const int sent_hi, int* __restrict__ overflow) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, N = G::N;
    constexpr uint32_t RS = ROW_SMEM_WORDS * 4;
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, tpb = blockDim.x;
    const int w = blockIdx.x * tpb + tid;
    const bool active = w < prm.W;
    uint32_t* const tbl_s = smem + WINDOW_PAD_ROWS * ROW_SMEM_WORDS;   // row 0 of the window
    for (int idx = tid; idx < (n_rows + 2 * WINDOW_PAD_ROWS) * ROW_SMEM_WORDS; idx += tpb) {
        const int jl = idx / ROW_SMEM_WORDS - WINDOW_PAD_ROWS, e = idx - (jl + WINDOW_PAD_ROWS) * ROW_SMEM_WORDS;
        const bool real = jl >= sent_lo && jl < n_rows - sent_hi;      // neither pad nor sentinel
        smem[idx] = (e < 8 && real) ? prm.table[(size_t)(j_lo + jl) * 8 + e] : 0u;   // e == 8: bin, e == 9: pad word
    }
    __syncthreads();

    const uint32_t o_base = (uint32_t)__cvta_generic_to_shared(tbl_s);
    const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                          : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
    uint32_t o = o_base;
    uint32_t* rows = prm.spins + (size_t)w * WPR;
    const size_t row_stride = (size_t)prm.W * WPR;
    const uint32_t walker = prm.walker_offset + (uint32_t)w;
    if (active) {
        o = o_base + (uint32_t)(((prm.E[w] + 2 * N) >> 2) - j_lo) * RS;          // the host put every walker inside the window
        streamed_sweeps<L, MODE_STREAMED_SMEM, true>(rows, row_stride, o, prm.sweep_begin, s_th, prm, walker, nullptr, tbl_s);
    }
    __syncthreads();
    // ---- thermalisation done: was a sentinel row entered?  then clear the bins for the measured sweeps
    bool left = false;
    for (int jl = tid; jl < n_rows; jl += tpb) {
        uint32_t& bin = tbl_s[jl * ROW_SMEM_WORDS + 8];
        if ((jl < sent_lo || jl >= n_rows - sent_hi) && bin) left = true;
        bin = 0u;
    }
    __syncthreads();
    if (active) {
        streamed_sweeps<L, MODE_STREAMED_SMEM, true>(rows, row_stride, o, s_th, prm.sweep_end, prm, walker, nullptr, tbl_s);
        prm.E[w] = ((int)((o - o_base) / RS) + j_lo) * 4 - 2 * N;
    }
    __syncthreads();
    // ---- a4: merge the window's bins into the global uint64 histogram; sentinel bins only report
    for (int jl = tid; jl < n_rows; jl += tpb) {
        const uint32_t v = tbl_s[jl * ROW_SMEM_WORDS + 8];
        if (jl < sent_lo || jl >= n_rows - sent_hi) {
            if (v) left = true;
        } else if (v && prm.sweep_end > prm.therm) {
            atomicAdd(prm.H + j_lo + jl, (unsigned long long)v);
        }
    }
    if (left) atomicOr(overflow, 1);
}

// ------------------------------------------------------------------------------------------------
// The same with Philox moved to paired deviate warps (as in the resident kernel, muca_resident.cuh): block =
// npairs walker warps (even warp ids) + npairs deviate warps (odd ids); pair p = warps 2p and 2p + 1 serve the 32
// walkers blockIdx.x * 32 * npairs + 32 p ...  A warp runs on scheduler (warp id % 4), so walker warps share
// schedulers with walker warps and deviate warps with deviate warps.  The deviate warp computes the 8 Philox calls
// of a 32-site word round-major and hands them over through a double-buffered ring, one named barrier per word
// (at most 8 pairs per block: barrier ids 1 .. 8, 128 registers per thread).  Shared memory: ring (npairs * 8 KB) | table window.
// ------------------------------------------------------------------------------------------------
constexpr int WPAIR_MAX_PAIRS = 8;   // 512 threads: 128 registers per thread
__host__ __device__ constexpr size_t wpair_ring_bytes(int npairs) { return (size_t)npairs * 2 * 8 * 32 * 16; }
__host__ __device__ constexpr size_t wpair_smem_bytes(int n_rows, int npairs) {
    return wpair_ring_bytes(npairs) + window_smem_bytes(n_rows);
}

template <int L>
__device__ __forceinline__ void wpair_deviates(uint4* __restrict__ ring, const int slots, int& buf, const int bar_id,
                                               const uint32_t s0, const uint32_t s1, const SweepParams& prm,
                                               const uint32_t walker, const bool active) {
    constexpr int WPR = Geo<L>::WPR;
    const uint32_t force = active ? 0u : 0xFFFFFFFFu;   // lanes without a walker get deviates that no threshold of a pad row accepts
#pragma unroll 1
    for (uint32_t s = s0; s < s1; ++s) {
#pragma unroll 1
        for (int word = 0; word < L * WPR; ++word) {      // typewriter word: sites 32 word .. 32 word + 31, calls 8 word .. + 7
            uint32_t st[8][4];
#pragma unroll
            for (int q = 0; q < 8; ++q) {                  // R4: ctr = (i >> 2, sweep, iteration, walker)
                st[q][0] = (uint32_t)(word * 8 + q); st[q][1] = s; st[q][2] = prm.iteration; st[q][3] = walker;
            }
#pragma unroll
            for (int r = 0; r < 10; ++r)
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    philox_round(st[q], prm.key0 + (uint32_t)r * 0x9E3779B9u, prm.key1 + (uint32_t)r * 0xBB67AE85u);
#pragma unroll
            for (int q = 0; q < 8; ++q)
                ring[(buf * 8 + q) * slots] = make_uint4(st[q][0] | force, st[q][1] | force, st[q][2] | force, st[q][3] | force);
            asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory");
            buf ^= 1;
        }
    }
}

template <int L>
__global__ void __launch_bounds__(64 * WPAIR_MAX_PAIRS, 1)
sweep_kernel_wpair(const SweepParams prm, const int j_lo, const int n_rows, const int sent_lo, const int sent_hi,
                   int* __restrict__ overflow) {
    using G = Geo<L>;
    constexpr int WPR = G::WPR, N = G::N;
    constexpr uint32_t RS = ROW_SMEM_WORDS * 4;
    extern __shared__ __align__(16) uint32_t smem[];
    const int tid = threadIdx.x, nthr = blockDim.x, npairs = nthr >> 6;
    const int warp_id = tid >> 5, lane = tid & 31, pair = warp_id >> 1;
    const bool is_walker = (warp_id & 1) == 0;
    const int slot = 32 * pair + lane, slots = 32 * npairs;
    const int w = blockIdx.x * slots + slot;
    const bool active = w < prm.W;
    uint4* const ring = reinterpret_cast<uint4*>(smem) + slot;
    uint32_t* const win = smem + wpair_ring_bytes(npairs) / 4;
    uint32_t* const tbl_s = win + WINDOW_PAD_ROWS * ROW_SMEM_WORDS;    // row 0 of the window
    for (int idx = tid; idx < (n_rows + 2 * WINDOW_PAD_ROWS) * ROW_SMEM_WORDS; idx += nthr) {
        const int jl = idx / ROW_SMEM_WORDS - WINDOW_PAD_ROWS, e = idx - (jl + WINDOW_PAD_ROWS) * ROW_SMEM_WORDS;
        const bool real = jl >= sent_lo && jl < n_rows - sent_hi;
        win[idx] = (e < 8 && real) ? prm.table[(size_t)(j_lo + jl) * 8 + e] : 0u;
    }
    __syncthreads();

    const uint32_t o_base = (uint32_t)__cvta_generic_to_shared(tbl_s);
    const uint32_t s_th = prm.therm < prm.sweep_begin ? prm.sweep_begin
                          : (prm.therm > prm.sweep_end ? prm.sweep_end : prm.therm);
    // Lanes without a walker must take part in the pair barriers of their warp, so they run the same code: they read
    // the rows of the last walker, store nothing, sit on pad row -1 (all thresholds 0) and receive deviates 0xFFFFFFFF.
    const int wl = active ? w : prm.W - 1;
    uint32_t* rows = prm.spins + (size_t)wl * WPR;
    const size_t row_stride = (size_t)prm.W * WPR;
    const uint32_t walker = prm.walker_offset + (uint32_t)w;
    uint32_t o = active && is_walker ? o_base + (uint32_t)(((prm.E[w] + 2 * N) >> 2) - j_lo) * RS : o_base - RS;
    int buf = 0;
    DeviateFeed feed{ring, slots, 0, 1 + pair};
    if (is_walker)
        streamed_sweeps<L, MODE_STREAMED_SMEM, true, true>(rows, row_stride, o, prm.sweep_begin, s_th, prm, walker, nullptr, tbl_s,
                                                           &feed, active);
    else
        wpair_deviates<L>(ring, slots, buf, 1 + pair, prm.sweep_begin, s_th, prm, walker, active);
    __syncthreads();
    bool left = false;
    for (int jl = tid; jl < n_rows; jl += nthr) {
        uint32_t& bin = tbl_s[jl * ROW_SMEM_WORDS + 8];
        if ((jl < sent_lo || jl >= n_rows - sent_hi) && bin) left = true;
        bin = 0u;
    }
    __syncthreads();
    if (is_walker) {
        streamed_sweeps<L, MODE_STREAMED_SMEM, true, true>(rows, row_stride, o, s_th, prm.sweep_end, prm, walker, nullptr, tbl_s, &feed,
                                                           active);
        if (active) prm.E[w] = ((int)((o - o_base) / RS) + j_lo) * 4 - 2 * N;
    } else {
        wpair_deviates<L>(ring, slots, buf, 1 + pair, s_th, prm.sweep_end, prm, walker, active);
    }
    __syncthreads();
    for (int jl = tid; jl < n_rows; jl += nthr) {
        const uint32_t v = tbl_s[jl * ROW_SMEM_WORDS + 8];
        if (jl < sent_lo || jl >= n_rows - sent_hi) {
            if (v) left = true;
        } else if (v && prm.sweep_end > prm.therm) {
            atomicAdd(prm.H + j_lo + jl, (unsigned long long)v);
        }
    }
    if (left) atomicOr(overflow, 1);
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
