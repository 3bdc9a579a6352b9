// timestep.cu -- row f2 of SURVEY.md Sec. 8: the time-step shell around the force calls.
// PAPER.md:80 (time bins with few active particles), :82 ("we execute the particle drifting process at the onset of a
// GPU-ported timestep for all particles (i.e., active and non-active ones)"), :320 (find_sync_point_and_drift).
// Readings R37..R42 of DESIGN.md Sec. 11 (Gadget-2's individual power-of-two time steps, Springel 2005):
//
//   k_ts_drift      R39  x += v dt for EVERY particle, wrapped into [0, L)
//   k_ts_maxbin     R37  largest occupied bin -> the next synchronisation tick
//   k_ts_count / k_ts_scan / k_ts_fill   R37  ascending list of the particles whose step divides the tick
//   k_ts_kick       R38, R40, R41  wanted bin from sqrt(2 eta eps / |a|) (fp32, fixed operation order), one-level growth at
//                   aligned ticks only, v += a (dt_old + dt_new) / 2, a_old = |a|
//
// oracle/timestep.py restates the same rules in NumPy and shares nothing with this file.
#include "og_internal.cuh"

namespace {

constexpr int TS_THREADS = 256;
constexpr int TS_ITEMS = 8;
constexpr int TS_TILE = TS_THREADS * TS_ITEMS;

__global__ void __launch_bounds__(256)
k_ts_drift(float *__restrict__ pos, const float *__restrict__ vel, uint64_t n3, float dt, float L)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;   // one coordinate per thread
    if (i >= n3) return;
    float x = fmaf(__ldg(vel + i), dt, pos[i]);
    x = fmaf(-L, floorf(x / L), x);          // into [0, L) for any displacement
    if (!(x >= 0.0f) || !(x < L)) x = 0.0f;  // the subtraction may round up to L
    pos[i] = x;
}

__global__ void __launch_bounds__(256)
k_ts_maxbin(const uint8_t *__restrict__ bin, uint64_t n, uint32_t *out)
{
    uint32_t m = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        m = max(m, (uint32_t)__ldg(bin + i));
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31u) == 0) atomicMax(out, m);
}

__device__ __forceinline__ bool ts_active(uint32_t b, uint64_t tick, uint32_t bmax)
{
    const uint64_t step = 1ull << (bmax - min(b, bmax));
    return (tick & (step - 1)) == 0;
}

// counts[tile] = active particles of the tile
__global__ void __launch_bounds__(TS_THREADS)
k_ts_count(const uint8_t *__restrict__ bin, uint64_t n, uint64_t tick, uint32_t bmax, uint32_t *__restrict__ counts)
{
    __shared__ uint32_t wsum[TS_THREADS / 32];
    const uint64_t base = (uint64_t)blockIdx.x * TS_TILE + (uint64_t)threadIdx.x * TS_ITEMS;
    uint32_t c = 0;
#pragma unroll
    for (int k = 0; k < TS_ITEMS; ++k)
        if (base + k < n && ts_active(__ldg(bin + base + k), tick, bmax)) ++c;
    c = __reduce_add_sync(0xffffffffu, c);
    if ((threadIdx.x & 31u) == 0) wsum[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t s = 0;
        for (int w = 0; w < TS_THREADS / 32; ++w) s += wsum[w];
        counts[blockIdx.x] = s;
    }
}

// exclusive scan of counts[0..n_tiles) in place by ONE block; total -> *total
__global__ void __launch_bounds__(1024)
k_ts_scan(uint32_t *__restrict__ counts, uint32_t n_tiles, unsigned long long *__restrict__ total)
{
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t carry_s;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    for (uint32_t b0 = 0; b0 < n_tiles; b0 += 1024) {
        const uint32_t b = b0 + tid;
        const uint32_t x = (b < n_tiles) ? counts[b] : 0;
        uint32_t incl = x;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= (uint32_t)o) incl += y;
        }
        const uint32_t carry = carry_s;
        __syncthreads();
        if (lane == 31) warp_sums[wid] = incl;
        __syncthreads();
        uint32_t woff = 0;
        for (uint32_t w = 0; w < wid; ++w) woff += warp_sums[w];
        if (b < n_tiles) counts[b] = carry + woff + incl - x;
        __syncthreads();
        if (tid == 1023) carry_s = carry + woff + incl;
        __syncthreads();
    }
    if (tid == 0) *total = carry_s;
}

// active_idx[offset of the tile + rank inside the tile] = i, ascending
__global__ void __launch_bounds__(TS_THREADS)
k_ts_fill(const uint8_t *__restrict__ bin, uint64_t n, uint64_t tick, uint32_t bmax, const uint32_t *__restrict__ offs,
          uint32_t *__restrict__ active_idx)
{
    __shared__ uint32_t wsum[TS_THREADS / 32];
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const uint64_t base = (uint64_t)blockIdx.x * TS_TILE + (uint64_t)threadIdx.x * TS_ITEMS;
    uint32_t flags = 0, c = 0;
#pragma unroll
    for (int k = 0; k < TS_ITEMS; ++k)
        if (base + k < n && ts_active(__ldg(bin + base + k), tick, bmax)) { flags |= 1u << k; ++c; }
    uint32_t incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    uint32_t woff = 0;
    for (uint32_t w = 0; w < wid; ++w) woff += wsum[w];
    uint32_t p = offs[blockIdx.x] + woff + incl - c;
#pragma unroll
    for (int k = 0; k < TS_ITEMS; ++k)
        if (flags & (1u << k)) active_idx[p++] = (uint32_t)(base + k);
}

// R38 in fp32, operation order fixed (no contraction): ratio = ((dt_max dt_max) |a|) / ((2 eta) eps);
// wanted bin = smallest b in [0, bmax] with 4^b >= ratio.
__device__ __forceinline__ uint32_t ts_wanted_bin(float an, float eps, float eta, float dt_max, uint32_t bmax)
{
    const float ratio = __fdiv_rn(__fmul_rn(__fmul_rn(dt_max, dt_max), an), __fmul_rn(__fmul_rn(2.0f, eta), eps));
    uint32_t b = 0;
    float p = 1.0f;
    for (uint32_t k = 0; k < bmax; ++k) {
        b += (ratio > p) ? 1u : 0u;
        p = __fmul_rn(p, 4.0f);
    }
    return b;
}

__global__ void __launch_bounds__(256)
k_ts_kick(float *__restrict__ vel, uint8_t *__restrict__ bin, float *__restrict__ a_old,
          const uint32_t *__restrict__ active_idx, uint64_t n, uint64_t n_active, const float *__restrict__ acc,
          const float *__restrict__ soft, float eta, float dt_max, uint32_t bmax, uint64_t tick, int first,
          uint32_t *status)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_active) return;
    uint64_t i = t;
    if (active_idx) {
        i = __ldg(active_idx + t);
        if (i >= n) { if (status) atomicOr(status, OG_DEV_BAD_INDEX); return; }
    }
    const float ax = __ldg(acc + 3 * t), ay = __ldg(acc + 3 * t + 1), az = __ldg(acc + 3 * t + 2);
    // |a| in fp32, fixed order: ((ax ax + ay ay) + az az), IEEE sqrt
    const float an = __fsqrt_rn(__fadd_rn(__fadd_rn(__fmul_rn(ax, ax), __fmul_rn(ay, ay)), __fmul_rn(az, az)));
    const uint32_t want = ts_wanted_bin(an, __ldg(soft + i), eta, dt_max, bmax);
    uint32_t nb;
    float half_dt;
    if (first) {                      // start of the integration: everybody takes the wanted bin, opening half kick only
        nb = want;
        half_dt = 0.5f * ldexpf(dt_max, -(int)nb);
    } else {
        const uint32_t cur = min((uint32_t)bin[i], bmax);
        nb = (want >= cur) ? want : cur;                                    // shrink (or keep) freely
        if (want < cur && ts_active(cur - 1u, tick, bmax)) nb = cur - 1u;   // grow one level at an aligned tick only
        half_dt = 0.5f * (ldexpf(dt_max, -(int)cur) + ldexpf(dt_max, -(int)nb));   // closing + opening half kick (R40)
    }
    vel[3 * i] = fmaf(ax, half_dt, vel[3 * i]);
    vel[3 * i + 1] = fmaf(ay, half_dt, vel[3 * i + 1]);
    vel[3 * i + 2] = fmaf(az, half_dt, vel[3 * i + 2]);
    bin[i] = (uint8_t)nb;
    a_old[i] = an;                                                          // R41
}

static_assert(OG_TS_BAD_INDEX == OG_DEV_BAD_INDEX, "og.h's status bit of og_ts_kick is the bit k_ts_kick sets");

inline size_t ts_tiles(uint64_t n) { return (size_t)((n + TS_TILE - 1) / TS_TILE); }

}  // namespace

extern "C" size_t og_ts_scratch_bytes(uint64_t n)
{
    return (ts_tiles(n) + 8) * sizeof(uint32_t) + 64;
}

extern "C" int og_ts_drift(float *pos, const float *vel, uint64_t n, float dt, float box, og_stream stream)
{
    og_set_error("%s", "");
    if (!pos || !vel || n == 0 || !(box > 0.0f)) { og_set_error("og_ts_drift: bad argument"); return OG_ERR_INVALID_ARG; }
    const uint64_t n3 = 3 * n;
    k_ts_drift<<<(unsigned)((n3 + 255) / 256), 256, 0, (cudaStream_t)stream>>>(pos, vel, n3, dt, box);
    OG_CUDA_TRY(cudaGetLastError(), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_ts_next_tick(const uint8_t *bin, uint64_t n, uint64_t tick, uint32_t bmax, uint64_t *next_tick_host,
                               void *scratch, size_t scratch_bytes, og_stream stream)
{
    og_set_error("%s", "");
    if (!bin || !next_tick_host || !scratch || n == 0 || bmax > 40 || scratch_bytes < og_ts_scratch_bytes(n)) {
        og_set_error("og_ts_next_tick: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t *d_max = reinterpret_cast<uint32_t *>(scratch);
    OG_CUDA_TRY(cudaMemsetAsync(d_max, 0, sizeof(uint32_t), st), return OG_ERR_CUDA);
    const uint64_t want_blocks = (n + 255) / 256;
    const uint64_t max_blocks = (uint64_t)ogk_sm_count() * 16;
    const unsigned grid = (unsigned)(want_blocks < max_blocks ? want_blocks : max_blocks);
    k_ts_maxbin<<<grid, 256, 0, st>>>(bin, n, d_max);
    uint32_t mb = 0;
    OG_CUDA_TRY(cudaMemcpyAsync(&mb, d_max, sizeof(mb), cudaMemcpyDeviceToHost, st), return OG_ERR_CUDA);
    OG_CUDA_TRY(cudaStreamSynchronize(st), return OG_ERR_CUDA);
    if (mb > bmax) mb = bmax;
    const uint64_t step = 1ull << (bmax - mb);           // smallest occupied step; every larger step is a multiple of it
    *next_tick_host = (tick / step + 1) * step;
    return OG_OK;
}

extern "C" int og_ts_active_list(const uint8_t *bin, uint64_t n, uint64_t tick, uint32_t bmax, uint32_t *active_idx,
                                 uint64_t *n_active_host, void *scratch, size_t scratch_bytes, og_stream stream)
{
    og_set_error("%s", "");
    if (!bin || !active_idx || !n_active_host || !scratch || n == 0 || n >= (1ull << 31) || bmax > 40 ||
        scratch_bytes < og_ts_scratch_bytes(n)) {
        og_set_error("og_ts_active_list: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t nt = (uint32_t)ts_tiles(n);
    unsigned long long *d_total = reinterpret_cast<unsigned long long *>(scratch);
    uint32_t *counts = reinterpret_cast<uint32_t *>(d_total + 2);
    k_ts_count<<<nt, TS_THREADS, 0, st>>>(bin, n, tick, bmax, counts);
    k_ts_scan<<<1, 1024, 0, st>>>(counts, nt, d_total);
    k_ts_fill<<<nt, TS_THREADS, 0, st>>>(bin, n, tick, bmax, counts, active_idx);
    unsigned long long tot = 0;
    OG_CUDA_TRY(cudaMemcpyAsync(&tot, d_total, sizeof(tot), cudaMemcpyDeviceToHost, st), return OG_ERR_CUDA);
    OG_CUDA_TRY(cudaStreamSynchronize(st), return OG_ERR_CUDA);
    *n_active_host = tot;
    return OG_OK;
}

extern "C" int og_ts_kick(float *vel, uint8_t *bin, float *a_old, const uint32_t *active_idx, uint64_t n,
                          uint64_t n_active, const float *acc, const float *soft, float eta, float dt_max, uint32_t bmax,
                          uint64_t tick, int first, uint32_t *status, og_stream stream)
{
    og_set_error("%s", "");
    if (n_active == 0) return OG_OK;
    if (!vel || !bin || !a_old || !acc || !soft || n == 0 || bmax > 40 || !(eta > 0.0f) || !(dt_max > 0.0f) ||
        (!active_idx && n_active != n)) {
        og_set_error("og_ts_kick: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    k_ts_kick<<<(unsigned)((n_active + 255) / 256), 256, 0, (cudaStream_t)stream>>>(vel, bin, a_old, active_idx, n, n_active,
                                                                                   acc, soft, eta, dt_max, bmax, tick, first,
                                                                                   status);
    OG_CUDA_TRY(cudaGetLastError(), return OG_ERR_CUDA);
    return OG_OK;
}
