// tb_reduce.cuh -- candidate reduction on the device ("a candidate
// reduction algorithm by grouping together multiple detections of the same candidate"; the paper
// gives no algorithm: reading G24 of DESIGN.md section 3).
//
//   R1  detections sorted by (template, fold, bin); a maximal run of adjacent bins within one
//       (template, fold) is one peak = its detection of highest sigma (ties: lowest bin)
//   R2  peaks ranked by (sigma descending, template, fold, bin)
//   R3  greedy distillation in rank order: an unabsorbed peak heads a group and absorbs every
//       weaker unabsorbed peak b with |q F_b - p F_h| <= tol16 for some 1 <= p, q <= 16, where
//       F = bin << (4 - fold) is the fundamental frequency in 1/16 bins (exact integers)
//   R4  groups numbered in head order, with peak / detection / distinct-template counts
//
// The list is small next to the search (10^2..10^6 rows of 24 bytes), so the kernels are simple:
// a bitonic sort (shared-memory tiles + global merge steps), a run scan, and R3 as rounds of a
// data-parallel rule that reaches the sequential greedy result: a peak is decided once its
// strongest related peak that has not been absorbed is decided (a head absorbs it; none -> it is a
// head itself).  The related peaks of a peak b are found, not scanned for: |q F_b - p F_a| <= tol
// means F_a lies in [(q F_b - tol)/p, (q F_b + tol)/p], so with the peaks also sorted by F each of
// the 159 coprime (p, q) pairs (a pair with a common factor g asks for tol/g: a subset) is one
// binary search plus a walk over the window: O(159 log np + matches) per peak and round instead of
// a walk over every stronger peak (O(np) each, O(np^2) per round, minutes at 10^5 peaks).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tb_kernels.cuh"

namespace tb {

struct SortRec {                 // 16 bytes: 96-bit key + payload
    uint64_t hi;
    uint32_t lo;
    uint32_t val;
};
__device__ __forceinline__ bool rec_less(const SortRec& a, const SortRec& b)
{
    return a.hi < b.hi || (a.hi == b.hi && (a.lo < b.lo || (a.lo == b.lo && a.val < b.val)));
}
__device__ __forceinline__ void rec_cas(SortRec& a, SortRec& b, bool up)
{
    if (rec_less(b, a) == up) { const SortRec t = a; a = b; b = t; }
}

constexpr int BS_TILE = 2048;    // records per shared-memory tile (32 KB)
constexpr int BS_THREADS = 1024;

// full bitonic sort of every BS_TILE-record tile (ascending in even tiles, descending in odd ones,
// i.e. the state of the network after the stage of size BS_TILE); n is a multiple of BS_TILE
__global__ void __launch_bounds__(BS_THREADS) k_bitonic_tiles(SortRec* __restrict__ r)
{
    __shared__ SortRec s[BS_TILE];
    SortRec* g = r + (size_t)blockIdx.x * BS_TILE;
    s[threadIdx.x] = g[threadIdx.x];
    s[threadIdx.x + BS_THREADS] = g[threadIdx.x + BS_THREADS];
    for (unsigned size = 2; size <= BS_TILE; size <<= 1) {
        for (unsigned j = size >> 1; j > 0; j >>= 1) {
            __syncthreads();
            const unsigned i = 2 * threadIdx.x - (threadIdx.x & (j - 1));           // lower index of the pair
            const size_t gi = (size_t)blockIdx.x * BS_TILE + i;
            rec_cas(s[i], s[i + j], (gi & size) == 0);
        }
    }
    __syncthreads();
    g[threadIdx.x] = s[threadIdx.x];
    g[threadIdx.x + BS_THREADS] = s[threadIdx.x + BS_THREADS];
}

// one compare-exchange step (distance j >= BS_TILE) of the stage of size `size`
__global__ void __launch_bounds__(256) k_bitonic_step(SortRec* __restrict__ r, size_t n, size_t size, size_t j)
{
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n / 2) return;
    const size_t i = 2 * t - (t & (j - 1));
    SortRec a = r[i], b = r[i + j];
    if (rec_less(b, a) == ((i & size) == 0)) { r[i] = b; r[i + j] = a; }
}

// the steps j = BS_TILE/2 .. 1 of the stage of size `size` (>= BS_TILE), inside shared memory
__global__ void __launch_bounds__(BS_THREADS) k_bitonic_finish(SortRec* __restrict__ r, size_t size)
{
    __shared__ SortRec s[BS_TILE];
    SortRec* g = r + (size_t)blockIdx.x * BS_TILE;
    s[threadIdx.x] = g[threadIdx.x];
    s[threadIdx.x + BS_THREADS] = g[threadIdx.x + BS_THREADS];
    const bool up = (((size_t)blockIdx.x * BS_TILE) & size) == 0;                    // size >= BS_TILE: uniform per tile
    for (unsigned j = BS_TILE >> 1; j > 0; j >>= 1) {
        __syncthreads();
        const unsigned i = 2 * threadIdx.x - (threadIdx.x & (j - 1));
        rec_cas(s[i], s[i + j], up);
    }
    __syncthreads();
    g[threadIdx.x] = s[threadIdx.x];
    g[threadIdx.x + BS_THREADS] = s[threadIdx.x + BS_THREADS];
}

// sort keys of the raw detections: (template, fold, bin); padding records sort last
__global__ void __launch_bounds__(256) k_red_det_keys(const Candidate* __restrict__ c, size_t n, size_t npad, SortRec* __restrict__ r)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npad) return;
    SortRec o;
    if (i < n) { o.hi = ((uint64_t)c[i].template_id << 32) | ((uint64_t)c[i].fold << 28) | c[i].bin; o.lo = 0; o.val = (uint32_t)i; }
    else       { o.hi = ~0ull; o.lo = ~0u; o.val = ~0u; }
    r[i] = o;
}

struct Peak {                    // 32 bytes
    uint32_t template_id, fold, bin;
    float    power, sigma;
    uint32_t n_det;              // detections in the run
    uint32_t first;              // position of the run's first detection in the sorted list
    uint32_t pad;
};

// R1: thread i = sorted detection i; the first detection of a run walks it and emits the peak
__global__ void __launch_bounds__(256)
k_red_peaks(const Candidate* __restrict__ c, const SortRec* __restrict__ srt, size_t n, Peak* __restrict__ peaks,
            uint32_t* __restrict__ peak_of, unsigned int* __restrict__ n_peaks)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint64_t key = srt[i].hi;
    if (i > 0 && srt[i - 1].hi + 1 == key && (uint32_t)(key & 0x0fffffffu) != 0u) return;   // continues its predecessor's run (same template and fold, next bin)
    size_t j = i;
    Candidate best = c[srt[i].val];
    while (j + 1 < n && srt[j + 1].hi == srt[j].hi + 1 && (uint32_t)(srt[j + 1].hi & 0x0fffffffu) != 0u) {
        ++j;
        const Candidate d = c[srt[j].val];
        if (d.sigma > best.sigma) best = d;
    }
    const unsigned int id = atomicAdd(n_peaks, 1u);
    Peak p;
    p.template_id = best.template_id; p.fold = best.fold; p.bin = best.bin; p.power = best.power; p.sigma = best.sigma;
    p.n_det = (uint32_t)(j - i + 1); p.first = (uint32_t)i; p.pad = 0;
    peaks[id] = p;
    for (size_t q = i; q <= j; ++q) peak_of[q] = id;
}

// order-preserving map of a float to an unsigned integer
__device__ __forceinline__ uint32_t float_key(float f)
{
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// R2 keys: (sigma descending, template, fold, bin)
__global__ void __launch_bounds__(256) k_red_peak_keys(const Peak* __restrict__ p, size_t n, size_t npad, SortRec* __restrict__ r)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npad) return;
    SortRec o;
    if (i < n) { o.hi = ((uint64_t)(~float_key(p[i].sigma)) << 32) | p[i].template_id; o.lo = (p[i].fold << 28) | p[i].bin; o.val = (uint32_t)i; }
    else       { o.hi = ~0ull; o.lo = ~0u; o.val = ~0u; }
    r[i] = o;
}

// after the rank sort: F of every rank, state = undecided, inverse permutation
__global__ void __launch_bounds__(256)
k_red_rank_init(const Peak* __restrict__ p, const SortRec* __restrict__ rank, size_t n, uint32_t* __restrict__ F, int* __restrict__ state,
                uint32_t* __restrict__ rank_of_peak)
{
    const size_t r = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const uint32_t id = rank[r].val;
    F[r] = p[id].bin << (4u - p[id].fold);
    state[r] = -1;
    rank_of_peak[id] = (uint32_t)r;
}

// sort keys of the F-sorted view: (F, rank); padding sorts last
__global__ void __launch_bounds__(256) k_red_freq_keys(const uint32_t* __restrict__ F, size_t n, size_t npad, SortRec* __restrict__ r)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= npad) return;
    SortRec o;
    if (i < n) { o.hi = F[i]; o.lo = (uint32_t)i; o.val = (uint32_t)i; }
    else       { o.hi = ~0ull; o.lo = ~0u; o.val = ~0u; }
    r[i] = o;
}

// the F-sorted view as two plain arrays (4-byte strides for the binary searches)
__global__ void __launch_bounds__(256)
k_red_freq_split(const SortRec* __restrict__ fs, size_t n, uint32_t* __restrict__ Fs, uint32_t* __restrict__ rank_at)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    Fs[i] = (uint32_t)fs[i].hi;
    rank_at[i] = fs[i].val;
}

__device__ __forceinline__ bool red_coprime(int p, int q)
{
    while (q) { const int t = p % q; p = q; q = t; }
    return p == 1;
}

// R3, one round.  state[r]: -1 undecided, r = head, h != r = absorbed by head h.  Decisions are final
// and depend only on final decisions of stronger peaks, so concurrent rounds reach the greedy result.
// Peak r looks up, window by window, the strongest (lowest-rank) related peak that is not absorbed:
// none -> r is a head; a head -> it absorbs r; still undecided -> r waits for the next round.
__global__ void __launch_bounds__(256)
k_red_distill_round(const uint32_t* __restrict__ F, const uint32_t* __restrict__ Fs, const uint32_t* __restrict__ rank_at,
                    volatile int* state, size_t n, int64_t tol, unsigned int* __restrict__ undecided)
{
    const size_t r = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n || state[r] >= 0) return;
    const int64_t Fb = F[r];
    uint32_t best = 0xffffffffu;
    int best_state = 0;
    for (int q = 1; q <= 16; ++q) {
        const int64_t c = q * Fb;
        for (int p = 1; p <= 16; ++p) {
            if (!red_coprime(p, q)) continue;
            int64_t lo = c - tol;                                                    // p Fa in [c - tol, c + tol]
            lo = lo <= 0 ? 0 : (lo + p - 1) / p;
            const int64_t hi = (c + tol) / p;
            if (hi < lo) continue;
            size_t a0 = 0, a1 = n;                                                   // first i with Fs[i] >= lo
            while (a0 < a1) { const size_t m = (a0 + a1) >> 1; if ((int64_t)Fs[m] < lo) a0 = m + 1; else a1 = m; }
            for (size_t i = a0; i < n && (int64_t)Fs[i] <= hi; ++i) {
                const uint32_t a = rank_at[i];
                if (a >= r || a >= best) continue;                                   // weaker than r, or no better than what we have
                const int sa = state[a];
                if (sa >= 0 && (uint32_t)sa != a) continue;                          // absorbed peaks absorb nothing
                best = a; best_state = sa;
            }
        }
    }
    if (best == 0xffffffffu) { state[r] = (int)r; return; }
    if (best_state < 0) { if (undecided) atomicAdd(undecided, 1u); return; }         // a stronger related peak is still open
    state[r] = (int)best;
}

// R4a: heads numbered in rank order (single CTA, chunked scan)
__global__ void __launch_bounds__(1024) k_red_number_heads(const int* __restrict__ state, size_t n, uint32_t* __restrict__ gid, unsigned int* __restrict__ n_groups)
{
    __shared__ unsigned int s_w[32];
    __shared__ unsigned int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (size_t base = 0; base < n; base += 1024) {
        const size_t r = base + threadIdx.x;
        const unsigned head = (r < n && state[r] == (int)r) ? 1u : 0u;
        const unsigned bal = __ballot_sync(0xffffffffu, head);
        const unsigned lane = threadIdx.x & 31, w = threadIdx.x >> 5;
        if (lane == 0) s_w[w] = __popc(bal);
        __syncthreads();
        unsigned before = s_carry;
        for (unsigned i = 0; i < w; ++i) before += s_w[i];
        if (head) gid[r] = before + __popc(bal & ((1u << lane) - 1u));
        __syncthreads();
        if (threadIdx.x == 0) { unsigned t = 0; for (int i = 0; i < 32; ++i) t += s_w[i]; s_carry += t; }
        __syncthreads();
    }
    if (threadIdx.x == 0) *n_groups = s_carry;
}

struct Group {                   // == tb_group, 32 bytes
    uint32_t template_id, fold, bin;
    float    power, sigma;
    uint32_t n_peaks, n_detections, n_templates;
};

// R4b: group records and counts; also the (group, template) keys for the distinct-template count
__global__ void __launch_bounds__(256)
k_red_groups(const Peak* __restrict__ p, const SortRec* __restrict__ rank, const int* __restrict__ state, const uint32_t* __restrict__ gid,
             size_t n, size_t npad, Group* __restrict__ groups, SortRec* __restrict__ gt)
{
    const size_t r = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= npad) return;
    if (r >= n) { SortRec o; o.hi = ~0ull; o.lo = ~0u; o.val = ~0u; gt[r] = o; return; }
    const Peak pk = p[rank[r].val];
    const uint32_t g = gid[state[r]];
    if (state[r] == (int)r) {
        groups[g].template_id = pk.template_id; groups[g].fold = pk.fold; groups[g].bin = pk.bin;
        groups[g].power = pk.power; groups[g].sigma = pk.sigma;
    }
    atomicAdd(&groups[g].n_peaks, 1u);
    atomicAdd(&groups[g].n_detections, pk.n_det);
    SortRec o;
    o.hi = ((uint64_t)g << 32) | pk.template_id; o.lo = 0; o.val = (uint32_t)r;
    gt[r] = o;
}

// R4c: distinct templates per group from the (group, template)-sorted keys
__global__ void __launch_bounds__(256) k_red_count_templates(const SortRec* __restrict__ gt, size_t n, Group* __restrict__ groups)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (i == 0 || gt[i - 1].hi != gt[i].hi) atomicAdd(&groups[gt[i].hi >> 32].n_templates, 1u);
}

// group of every detection of the (template, fold, bin)-sorted list
__global__ void __launch_bounds__(256)
k_red_members(const uint32_t* __restrict__ peak_of, const uint32_t* __restrict__ rank_of_peak, const int* __restrict__ state,
              const uint32_t* __restrict__ gid, size_t n, uint32_t* __restrict__ member_of)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    member_of[i] = gid[state[rank_of_peak[peak_of[i]]]];
}

}  // namespace tb
