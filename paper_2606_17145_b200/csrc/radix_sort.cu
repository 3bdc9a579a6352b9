// radix_sort.cu -- row a2 of SURVEY.md Sec. 8(a): stable LSD radix sort of (u64 key, u32 val)
// pairs, 8 bits per pass (C2, R3).  Stability is what delivers the index tie-break: the
// values start as the identity, so equal keys stay in ascending original index.
//
// One-sweep passes (n < 2^30): ONE kernel reads the keys once up front and builds the global digit
// histograms of all passes (k_sort_ghist; k_sort_gscan turns them into digit bases).  A pass is then a
// single kernel, k_sort_onesweep: a block takes the next 2048-pair tile (dynamic ticket, so tiles start in
// order), ranks every key inside the tile in input order (nine ballots give the lanes with an equal digit,
// per-warp digit counters in shared memory), publishes the tile's digit counts and obtains the counts of all
// earlier tiles by a decoupled look-back (thread d follows digit d), reorders the tile by digit in shared
// memory and writes coalesced runs: 12 B read + 12 B written per pair per pass.  Larger inputs use the
// three-kernel pass (k_sort_hist / k_sort_scan / k_sort_scatter, 32 B/pair/pass).  A pass sorts on the bits
// [shift, shift + nbits) only (nbits < 8 in the last pass of a range that is not a multiple of 8).
#include "og_internal.cuh"

namespace {

constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_ITEMS = 8;                        // keys per thread
constexpr int SORT_WARP_TILE = 32 * SORT_ITEMS;      // 256 consecutive keys per warp
constexpr int SORT_TILE = SORT_THREADS * SORT_ITEMS; // 2048 keys per block

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
// Lanes of the warp whose 8-bit digit equals this lane's (and whose `ok` flag equals this lane's): nine
// ballots instead of __match_any_sync, which the hardware serialises over the distinct values.
__device__ __forceinline__ uint32_t digit_peers(uint32_t d, bool ok)
{
    uint32_t peers = __ballot_sync(0xffffffffu, ok);
    peers = ok ? peers : ~peers;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
        const bool bit = (d >> b) & 1u;
        const uint32_t bal = __ballot_sync(0xffffffffu, bit);
        peers &= bit ? bal : ~bal;
    }
    return peers;
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// hist[d * n_tiles + tile] = number of keys of the tile whose digit is d; ghist[d] += same.
__global__ void __launch_bounds__(SORT_THREADS)
k_sort_hist(const uint64_t *__restrict__ keys, uint64_t n, int shift, uint32_t dmask, uint32_t n_tiles,
            uint32_t *__restrict__ hist, uint32_t *__restrict__ ghist)
{
    __shared__ uint32_t h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * SORT_TILE + (threadIdx.x >> 5) * SORT_WARP_TILE + lane_id();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint64_t i = base + (uint64_t)r * 32;
        {
            const bool ok = i < n;
            const uint32_t d = ok ? ((uint32_t)(__ldg(keys + i) >> shift) & dmask) : 0u;
            // aggregate equal digits inside the warp before touching shared memory
            const uint32_t peers = digit_peers(d, ok);
            if (ok && (peers & lanemask_lt()) == 0) atomicAdd(&h[d], __popc(peers));
        }
    }
    __syncthreads();
    const uint32_t c = h[threadIdx.x];
    hist[(uint64_t)threadIdx.x * n_tiles + blockIdx.x] = c;
    if (c) atomicAdd(&ghist[threadIdx.x], c);
}

// One block per digit d: exclusive scan of hist[d][0..n_tiles) plus the number of keys with a
// smaller digit.
__global__ void __launch_bounds__(1024)
k_sort_scan(uint32_t *__restrict__ hist, const uint32_t *__restrict__ ghist, uint32_t n_tiles)
{
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t carry_s;
    const uint32_t d = blockIdx.x, tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    // digit base = sum of ghist[0..d)
    uint32_t v = (tid < d && tid < 256) ? ghist[tid] : 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) warp_sums[wid] = v;
    __syncthreads();
    if (tid == 0) {
        uint32_t s = 0;
        for (int w = 0; w < 32; ++w) s += warp_sums[w];
        carry_s = s;
    }
    __syncthreads();
    uint32_t *row = hist + (uint64_t)d * n_tiles;
    for (uint32_t b0 = 0; b0 < n_tiles; b0 += 1024) {
        const uint32_t b = b0 + tid;
        const uint32_t x = (b < n_tiles) ? row[b] : 0;
        uint32_t incl = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (uint32_t)o) incl += y;
        }
        const uint32_t carry = carry_s;
        __syncthreads();  // everyone has read carry_s / previous warp_sums
        if (lane == 31) warp_sums[wid] = incl;
        __syncthreads();
        uint32_t woff = 0;
        for (uint32_t w = 0; w < wid; ++w) woff += warp_sums[w];
        if (b < n_tiles) row[b] = carry + woff + incl - x;
        __syncthreads();
        if (tid == 1023) carry_s = carry + woff + incl;
        __syncthreads();
    }
}

// Stable scatter of one 2048-pair tile.  Every key is ranked inside the tile in input order (ballot
// ranking, per-warp digit counters, exclusive prefix over the warps and over the digits),
// the tile is reordered by digit in shared memory, and then written out: consecutive threads write
// consecutive elements of a digit's run, so the global stores are coalesced runs instead of 32
// scattered 8-byte writes per warp instruction.
struct ScatterSmem {
    uint64_t keys[SORT_TILE];
    uint32_t vals[SORT_TILE];
    uint32_t cnt[SORT_WARPS][256];
    uint32_t gbase[256];    // global offset of the tile's first key of digit d, minus its position in the tile
};

__global__ void __launch_bounds__(SORT_THREADS)
k_sort_scatter(const uint64_t *__restrict__ keys_in, const uint32_t *__restrict__ vals_in,
               uint64_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out, uint64_t n,
               int shift, uint32_t dmask, uint32_t n_tiles, const uint32_t *__restrict__ offs)
{
    extern __shared__ __align__(16) unsigned char sort_smem_raw[];
    ScatterSmem &sm = *reinterpret_cast<ScatterSmem *>(sort_smem_raw);
    __shared__ uint32_t wsum[SORT_WARPS];
    const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.cnt[w][tid] = 0;
    const uint32_t goff = offs[(uint64_t)tid * n_tiles + blockIdx.x];
    __syncthreads();

    const uint64_t tile0 = (uint64_t)blockIdx.x * SORT_TILE;
    const uint64_t base = tile0 + wid * SORT_WARP_TILE + lane;
    uint64_t key[SORT_ITEMS];
    uint32_t val[SORT_ITEMS];
    uint32_t rank[SORT_ITEMS];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint64_t i = base + (uint64_t)r * 32;
        const bool ok = i < n;
        key[r] = ok ? __ldg(keys_in + i) : ~0ull;
        val[r] = ok ? __ldg(vals_in + i) : 0u;
    }
    // rank inside the warp's 256-key chunk, in input order (round-major, lane-minor)
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const bool ok = (base + (uint64_t)r * 32) < n;
        const uint32_t d = ok ? ((uint32_t)(key[r] >> shift) & dmask) : 0u;
        const uint32_t peers = digit_peers(d, ok);
        const int leader = __ffs(peers) - 1;
        uint32_t b = 0;
        if ((int)lane == leader && ok) {
            b = sm.cnt[wid][d];
            sm.cnt[wid][d] = b + __popc(peers);
        }
        b = __shfl_sync(0xffffffffu, b, leader);
        rank[r] = b + __popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    // per digit (thread tid = digit): exclusive prefix over the warps, then over the digits of the tile
    uint32_t total = 0;
    {
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            const uint32_t c = sm.cnt[w][tid];
            sm.cnt[w][tid] = total;
            total += c;
        }
    }
    uint32_t incl = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    uint32_t dstart = incl - total;   // first position of digit tid inside the tile
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) dstart += (w < (int)wid) ? wsum[w] : 0u;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.cnt[w][tid] += dstart;
    sm.gbase[tid] = goff - dstart;
    __syncthreads();
    // reorder the tile by digit in shared memory
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        if ((base + (uint64_t)r * 32) < n) {
            const uint32_t d = (uint32_t)(key[r] >> shift) & dmask;
            const uint32_t p = sm.cnt[wid][d] + rank[r];
            sm.keys[p] = key[r];
            sm.vals[p] = val[r];
        }
    }
    __syncthreads();
    const uint32_t in_tile = (uint32_t)min((uint64_t)SORT_TILE, n - tile0);
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = tid + r * SORT_THREADS;
        if (i < in_tile) {
            const uint64_t k = sm.keys[i];
            const uint32_t p = sm.gbase[(uint32_t)(k >> shift) & dmask] + i;
            keys_out[p] = k;
            vals_out[p] = sm.vals[i];
        }
    }
}

// ---- one-sweep passes --------------------------------------------------------------------------------------------
constexpr int SORT_MAX_PASSES = 8;

// ghist[p][d] = number of keys whose digit of pass p is d (all passes from one read of the keys)
__global__ void __launch_bounds__(SORT_THREADS)
k_sort_ghist(const uint64_t *__restrict__ keys, uint64_t n, int begin_bit, int end_bit, int passes,
             uint32_t *__restrict__ ghist)
{
    __shared__ uint32_t h[SORT_MAX_PASSES][256];
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) (&h[0][0])[i] = 0;
    __syncthreads();
    const uint64_t stride = (uint64_t)gridDim.x * SORT_THREADS;
    for (uint64_t i = (uint64_t)blockIdx.x * SORT_THREADS + threadIdx.x; i < n; i += stride) {
        const uint64_t k = __ldg(keys + i);
        for (int p = 0; p < passes; ++p) {
            const int shift = begin_bit + 8 * p;
            const int nbits = (end_bit - shift) < 8 ? (end_bit - shift) : 8;
            atomicAdd(&h[p][(uint32_t)(k >> shift) & ((1u << nbits) - 1u)], 1u);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < passes * 256; i += SORT_THREADS) {
        const uint32_t c = (&h[0][0])[i];
        if (c) atomicAdd(ghist + i, c);
    }
}

// exclusive scan of every pass's 256 counts (one block per pass)
__global__ void __launch_bounds__(256) k_sort_gscan(uint32_t *__restrict__ ghist)
{
    __shared__ uint32_t wsum[8];
    uint32_t *g = ghist + 256 * blockIdx.x;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    const uint32_t x = g[tid];
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    uint32_t off = 0;
    for (uint32_t w = 0; w < wid; ++w) off += wsum[w];
    g[tid] = off + incl - x;
}

// tile status word: bits 0..29 a count, bits 30..31 the flag (1 = the tile's own count of digit d, 2 = inclusive
// count of digit d over tiles 0..t); 0 = not published (the array is zeroed before the pass)
#define SORT_FLAG_AGG 0x40000000u
#define SORT_FLAG_INCL 0x80000000u
#define SORT_VALUE_MASK 0x3fffffffu
#ifndef SORT_LOOK
#define SORT_LOOK 8
#endif
#ifndef SORT_OS_BLOCKS
#define SORT_OS_BLOCKS 4
#endif

__global__ void __launch_bounds__(SORT_THREADS, SORT_OS_BLOCKS)
k_sort_onesweep(const uint64_t *__restrict__ keys_in, const uint32_t *__restrict__ vals_in,
                uint64_t *__restrict__ keys_out, uint32_t *__restrict__ vals_out, uint64_t n,
                int shift, uint32_t dmask, uint32_t n_tiles, const uint32_t *__restrict__ gbase,
                uint32_t *__restrict__ status, uint32_t *__restrict__ ticket)
{
    extern __shared__ __align__(16) unsigned char sort_smem_raw[];
    ScatterSmem &sm = *reinterpret_cast<ScatterSmem *>(sort_smem_raw);
    __shared__ uint32_t wsum[SORT_WARPS];
    __shared__ uint32_t tile_s;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    if (tid == 0) tile_s = atomicAdd(ticket, 1u);
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.cnt[w][tid] = 0;
    __syncthreads();
    const uint32_t tile = tile_s;
    if (tile >= n_tiles) return;

    const uint64_t tile0 = (uint64_t)tile * SORT_TILE;
    const uint64_t base = tile0 + wid * SORT_WARP_TILE + lane;
    uint64_t key[SORT_ITEMS];
    uint32_t val[SORT_ITEMS];
    uint32_t rank[SORT_ITEMS];
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint64_t i = base + (uint64_t)r * 32;
        const bool ok = i < n;
        key[r] = ok ? __ldg(keys_in + i) : ~0ull;
        val[r] = ok ? __ldg(vals_in + i) : 0u;
    }
    const uint32_t lt = lanemask_lt();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const bool ok = (base + (uint64_t)r * 32) < n;
        const uint32_t d = ok ? ((uint32_t)(key[r] >> shift) & dmask) : 0u;
        const uint32_t peers = digit_peers(d, ok);
        const int leader = __ffs(peers) - 1;
        uint32_t b = 0;
        if ((int)lane == leader && ok) {
            b = sm.cnt[wid][d];
            sm.cnt[wid][d] = b + __popc(peers);
        }
        b = __shfl_sync(0xffffffffu, b, leader);
        rank[r] = b + __popc(peers & lt);
        __syncwarp();
    }
    __syncthreads();
    // per digit (thread tid = digit): the tile's count, exclusive prefix over the warps
    uint32_t total = 0;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) {
        const uint32_t c = sm.cnt[w][tid];
        sm.cnt[w][tid] = total;
        total += c;
    }
    // publish the tile's counts at once; the look-back over the earlier tiles comes last, after the tile has been
    // reordered in shared memory (which needs only the tile's own counts), so that the predecessors have had time
    // to publish their inclusive counts
    volatile uint32_t *st = status + tid;     // status[t * 256 + d]
    st[(size_t)tile * 256] = (tile == 0 ? SORT_FLAG_INCL : SORT_FLAG_AGG) | total;
    // first position of digit tid inside the tile: exclusive prefix of the tile's counts over the digits
    uint32_t incl = total;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    uint32_t dstart = incl - total;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) dstart += (w < (int)wid) ? wsum[w] : 0u;
#pragma unroll
    for (int w = 0; w < SORT_WARPS; ++w) sm.cnt[w][tid] += dstart;
    __syncthreads();
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        if ((base + (uint64_t)r * 32) < n) {
            const uint32_t d = (uint32_t)(key[r] >> shift) & dmask;
            const uint32_t p = sm.cnt[wid][d] + rank[r];
            sm.keys[p] = key[r];
            sm.vals[p] = val[r];
        }
    }
    __syncthreads();
    uint32_t excl = 0;
    if (tile > 0) {
        // SORT_LOOK predecessors per round trip (independent loads), consumed in order up to the first one that is not
        // published yet (re-read in the next round) or that carries an inclusive count (done)
        int64_t t = (int64_t)tile - 1;
        bool done = false;
        while (!done) {
            uint32_t v[SORT_LOOK];
#pragma unroll
            for (int j = 0; j < SORT_LOOK; ++j) v[j] = (t - j >= 0) ? st[(size_t)(t - j) * 256] : SORT_FLAG_INCL;
            int used = 0;
#pragma unroll
            for (int j = 0; j < SORT_LOOK; ++j) {
                if (!done && used == j && v[j] != 0u) {
                    excl += v[j] & SORT_VALUE_MASK;
                    done = (v[j] & SORT_FLAG_INCL) != 0u;
                    used = j + 1;
                }
            }
            t -= used;
        }
        st[(size_t)tile * 256] = SORT_FLAG_INCL | (excl + total);
    }
    sm.gbase[tid] = __ldg(gbase + tid) + excl - dstart;
    __syncthreads();
    const uint32_t in_tile = (uint32_t)min((uint64_t)SORT_TILE, n - tile0);
#pragma unroll
    for (int r = 0; r < SORT_ITEMS; ++r) {
        const uint32_t i = tid + r * SORT_THREADS;
        if (i < in_tile) {
            const uint64_t k = sm.keys[i];
            const uint32_t p = sm.gbase[(uint32_t)(k >> shift) & dmask] + i;
            keys_out[p] = k;
            vals_out[p] = sm.vals[i];
        }
    }
}

}  // namespace

static inline uint32_t sort_tiles(uint64_t n) { return (uint32_t)((n + SORT_TILE - 1) / SORT_TILE); }

// one-sweep scratch: [8][256] global histograms / digit bases, 8 tickets, then per pass a [n_tiles][256] status array
static inline bool sort_onesweep(uint64_t n) { return n < (1ull << 30); }

size_t ogk_sort_scratch_bytes(uint64_t n)
{
    const size_t tiles = sort_tiles(n);
    if (sort_onesweep(n)) return ((size_t)SORT_MAX_PASSES * 256 + 64 + (size_t)SORT_MAX_PASSES * tiles * 256) * sizeof(uint32_t) + 256;
    // per-tile histogram (digit-major) + 8 global histograms
    return (tiles * 256 + 8 * 256) * sizeof(uint32_t) + 256;
}

cudaError_t ogk_radix_sort(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt,
                           uint64_t n, int begin_bit, int end_bit, void *scratch, int *in_alt,
                           cudaStream_t st)
{
    const uint32_t n_tiles = sort_tiles(n);
    const int passes = (end_bit - begin_bit + 7) / 8;
    uint64_t *kin = keys, *kout = keys_alt;
    uint32_t *vin = vals, *vout = vals_alt;
    if (in_alt) *in_alt = (passes & 1);
    if (passes <= 0 || n == 0) return cudaSuccess;
    if (sort_onesweep(n) && passes <= SORT_MAX_PASSES) {
        uint32_t *ghist = reinterpret_cast<uint32_t *>(scratch);
        uint32_t *ticket = ghist + SORT_MAX_PASSES * 256;
        uint32_t *status = ticket + 64;
        cudaError_t e = cudaFuncSetAttribute(k_sort_onesweep, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ScatterSmem));
        if (e != cudaSuccess) return e;
        e = cudaMemsetAsync(scratch, 0, ((size_t)SORT_MAX_PASSES * 256 + 64 + (size_t)passes * n_tiles * 256) * sizeof(uint32_t), st);
        if (e != cudaSuccess) return e;
        const uint64_t hwant = (n + SORT_THREADS * 16 - 1) / (SORT_THREADS * 16);
        const uint64_t hmax = (uint64_t)ogk_sm_count() * 8;          // 8 resident blocks of 256 threads per SM
        const unsigned hgrid = (unsigned)(hwant < hmax ? hwant : hmax);
        k_sort_ghist<<<hgrid, SORT_THREADS, 0, st>>>(kin, n, begin_bit, end_bit, passes, ghist);
        k_sort_gscan<<<passes, 256, 0, st>>>(ghist);
        for (int p = 0; p < passes; ++p) {
            const int shift = begin_bit + 8 * p;
            const int nbits = (end_bit - shift) < 8 ? (end_bit - shift) : 8;     // the contract is [begin_bit, end_bit)
            const uint32_t dmask = (1u << nbits) - 1u;
            k_sort_onesweep<<<n_tiles, SORT_THREADS, sizeof(ScatterSmem), st>>>(kin, vin, kout, vout, n, shift, dmask, n_tiles,
                                                                                ghist + 256 * p, status + (size_t)p * n_tiles * 256,
                                                                                ticket + p);
            uint64_t *tk = kin; kin = kout; kout = tk;
            uint32_t *tv = vin; vin = vout; vout = tv;
        }
        return cudaGetLastError();
    }
    uint32_t *hist = reinterpret_cast<uint32_t *>(scratch);
    uint32_t *ghist = hist + (size_t)n_tiles * 256;
    cudaError_t e = cudaFuncSetAttribute(k_sort_scatter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(ScatterSmem));
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(ghist, 0, 8 * 256 * sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    for (int p = 0; p < passes; ++p) {
        const int shift = begin_bit + 8 * p;
        const int nbits = (end_bit - shift) < 8 ? (end_bit - shift) : 8;     // the contract is [begin_bit, end_bit)
        const uint32_t dmask = (1u << nbits) - 1u;
        k_sort_hist<<<n_tiles, SORT_THREADS, 0, st>>>(kin, n, shift, dmask, n_tiles, hist, ghist + 256 * p);
        k_sort_scan<<<256, 1024, 0, st>>>(hist, ghist + 256 * p, n_tiles);
        k_sort_scatter<<<n_tiles, SORT_THREADS, sizeof(ScatterSmem), st>>>(kin, vin, kout, vout, n, shift, dmask, n_tiles, hist);
        uint64_t *tk = kin; kin = kout; kout = tk;
        uint32_t *tv = vin; vin = vout; vout = tv;
    }
    return cudaGetLastError();
}

// ---- og_radix_sort_pairs_noalloc: the same sort with its scratch inside the library --------------------------------
// For callers that must not allocate device memory at the moment they need a sort: a host code whose device memory
// was handed out in full at start-up to its own arena, a step that runs while another thread holds the allocator,
// a plug-in that is only lent buffers.  They cannot supply og_radix_sort_pairs' scratch from a fresh cudaMalloc, so
// the scratch of this variant (digit histograms, tile tickets, look-back status words of the one-sweep passes) is a
// fixed array in the library image: OG_SORT_NOALLOC_MAX_N pairs at most, about 4 MiB, resident on every GPU that
// loads libogtree.so for as long as the process lives.
//
// The array is one object shared by every call on a device.  ogk_radix_sort zeroes the part a call uses (cudaMemsetAsync
// on the caller's stream) before its kernels run, so what the previous call left behind never matters; two calls
// that are in flight on the GPU at the same time (different streams, or different host threads) would overwrite
// each other's status words and must be ordered by the caller.
//
// g_sort_noalloc_scratch below is a DEVICE object.  In host code its name is only the host-side handle of the
// symbol, never an address a kernel may dereference; the device address is asked for once per device with
// cudaGetSymbolAddress (with that device current) and kept in g_noalloc_ptr[].  That first call per device may make
// the runtime load this module, which is why og.h asks for it to happen outside a stream capture.
#include <mutex>

namespace {
constexpr uint64_t NOALLOC_MAX_N = OG_SORT_NOALLOC_MAX_N;
constexpr size_t NOALLOC_TILES = (NOALLOC_MAX_N + SORT_TILE - 1) / SORT_TILE;
constexpr size_t NOALLOC_BYTES =
    ((size_t)SORT_MAX_PASSES * 256 + 64 + (size_t)SORT_MAX_PASSES * NOALLOC_TILES * 256) * sizeof(uint32_t) + 256;
constexpr int NOALLOC_MAX_DEVICES = 64;
void *g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of the array on device d, 0 until asked for
std::mutex g_noalloc_mu;
}  // namespace

static __device__ __align__(256) unsigned char g_sort_noalloc_scratch[NOALLOC_BYTES];

size_t ogk_sort_noalloc_max_n(void) { return (size_t)NOALLOC_MAX_N; }

// Resolves the array's address on the current device (first call per device only), then runs the unchanged sort on
// it.  Calls nothing that allocates: cudaGetDevice, cudaGetSymbolAddress, cudaFuncSetAttribute, cudaMemsetAsync and
// kernel launches.  n <= OG_SORT_NOALLOC_MAX_N is the caller's (api.cu's) check; it is repeated here because an
// overrun of a file-scope array would corrupt whatever the linker placed behind it.
cudaError_t ogk_radix_sort_noalloc(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt, uint64_t n,
                                   int begin_bit, int end_bit, int *in_alt, cudaStream_t st)
{
    if (n > NOALLOC_MAX_N || ogk_sort_scratch_bytes(n) > NOALLOC_BYTES) return cudaErrorInvalidValue;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    void *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mu);
        if (!g_noalloc_ptr[dev]) {
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_sort_noalloc_scratch);
            if (e != cudaSuccess) return e;
            if (!p) return cudaErrorInvalidSymbol;
            g_noalloc_ptr[dev] = p;
        }
        scratch = g_noalloc_ptr[dev];
    }
    return ogk_radix_sort(keys, vals, keys_alt, vals_alt, n, begin_bit, end_bit, scratch, in_alt, st);
}
