// let.cu -- row f4 of SURVEY.md Sec. 8: the pieces of a domain-decomposed short-range force around the walk.
// PAPER.md:59 ("primary" walk of the particles of the same rank, particles that need other ranks' trees are exported,
// "secondary" walk there, results sent back), :80 (export buffers).  Readings R49..R53, DESIGN.md Sec. 13.
//   k_cell_hist       particles per level-5 cell (top 15 key bits): the input of the splitter rule R49
//   k_owner           domain of every particle from the splitters
//   k_let_mark        R52: is a target within r_cut of one of a domain's top-cell boxes?
//   k_flag_count / k_flag_scan / k_flag_fill   ascending list of the flagged targets (what is exported)
//   k_let_accumulate  R51: partial results of another domain's walk added to the targets they belong to
//   k_ext_gather      imported targets put in their Morton order as (x, y, z, h) for the walk (walk.cu, a.ext)
// The exchange between the ranks is NCCL all-to-all in the host layer (paper_2606_17145_b200/let.py); nothing here
// communicates.
#include "og_internal.cuh"

namespace {

constexpr int LET_TILE = 2048;

__global__ void __launch_bounds__(256) k_cell_hist(const uint64_t *__restrict__ keys, uint64_t n, uint32_t *__restrict__ hist)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicAdd(hist + (uint32_t)(keys[i] >> 48), 1u);
}

// owner = the d with S[d] <= cell < S[d + 1] (S ascending, S[0] = 0, S[R] = 2^15)
__global__ void __launch_bounds__(256) k_owner(const uint64_t *__restrict__ keys, uint64_t n, const uint32_t *__restrict__ S,
                                               uint32_t R, uint32_t *__restrict__ owner)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t cell = (uint32_t)(keys[i] >> 48);
    uint32_t lo = 0u, hi = R;                    // invariant: S[lo] <= cell < S[hi]
    while (hi - lo > 1u) {
        const uint32_t mid = (lo + hi) >> 1;
        if (__ldg(S + mid) <= cell) lo = mid; else hi = mid;
    }
    owner[i] = lo;
}

// boxes: [nb][6] = (lo_x, lo_y, lo_z, hi_x, hi_y, hi_z).  The test is conservative by a relative 1e-5 (+ rounding of
// the box centre): a target marked without need is walked on the other domain and receives exactly nothing there.
__global__ void __launch_bounds__(256) k_let_mark(const float *__restrict__ tpos, uint64_t n_t, const float *__restrict__ boxes,
                                                  uint32_t nb, float r_cut, float L, uint8_t *__restrict__ flag)
{
    extern __shared__ float sb[];
    for (uint32_t i = threadIdx.x; i < nb * 6u; i += blockDim.x) sb[i] = boxes[i];
    __syncthreads();
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_t) return;
    const float x = tpos[3 * t], y = tpos[3 * t + 1], z = tpos[3 * t + 2];
    const float invL = 1.0f / L, pad = 4.0e-7f * L;
    const float rc = r_cut * (1.0f + 1.0e-5f) + pad;
    const float rc2 = rc * rc;
    bool hit = false;
    for (uint32_t b = 0; b < nb && !hit; ++b) {
        const float *q = sb + 6u * b;
        float dx = 0.5f * (q[0] + q[3]) - x, dy = 0.5f * (q[1] + q[4]) - y, dz = 0.5f * (q[2] + q[5]) - z;
        dx = fmaf(-L, rintf(dx * invL), dx); dy = fmaf(-L, rintf(dy * invL), dy); dz = fmaf(-L, rintf(dz * invL), dz);
        const float ex = fmaxf(fabsf(dx) - 0.5f * (q[3] - q[0]) - pad, 0.0f), ey = fmaxf(fabsf(dy) - 0.5f * (q[4] - q[1]) - pad, 0.0f),
                    ez = fmaxf(fabsf(dz) - 0.5f * (q[5] - q[2]) - pad, 0.0f);
        hit = fmaf(ez, ez, fmaf(ey, ey, ex * ex)) <= rc2;
    }
    flag[t] = hit ? 1 : 0;
}

__global__ void __launch_bounds__(256) k_flag_count(const uint8_t *__restrict__ flag, uint64_t n, uint32_t *__restrict__ tile_cnt)
{
    __shared__ uint32_t s;
    if (threadIdx.x == 0) s = 0u;
    __syncthreads();
    const uint64_t base = (uint64_t)blockIdx.x * LET_TILE;
    uint32_t c = 0u;
    for (uint32_t k = threadIdx.x; k < LET_TILE; k += 256u)
        if (base + k < n && flag[base + k]) ++c;
    atomicAdd(&s, c);
    __syncthreads();
    if (threadIdx.x == 0) tile_cnt[blockIdx.x] = s;
}

// exclusive scan of the tile counts by one block (tiles <= a few 10^4); total -> tile_cnt[n_tiles]
__global__ void __launch_bounds__(1024) k_flag_scan(uint32_t *__restrict__ tile_cnt, uint32_t n_tiles)
{
    __shared__ uint32_t part[1024];
    const uint32_t per = (n_tiles + 1023u) / 1024u;
    const uint32_t b = threadIdx.x * per, e = min(b + per, n_tiles);
    uint32_t s = 0u;
    for (uint32_t i = b; i < e; ++i) s += tile_cnt[i];
    part[threadIdx.x] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = 0u;
        for (int i = 0; i < 1024; ++i) { const uint32_t v = part[i]; part[i] = run; run += v; }
        tile_cnt[n_tiles] = run;
    }
    __syncthreads();
    uint32_t run = part[threadIdx.x];
    for (uint32_t i = b; i < e; ++i) { const uint32_t v = tile_cnt[i]; tile_cnt[i] = run; run += v; }
}

// one warp per 32-element chunk keeps the order: ballot ranks inside the chunk, chunk offsets by a block scan
__global__ void __launch_bounds__(256) k_flag_fill(const uint8_t *__restrict__ flag, uint64_t n, const uint32_t *__restrict__ tile_off,
                                                   uint32_t *__restrict__ out)
{
    __shared__ uint32_t wcnt[8];
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    const uint64_t base = (uint64_t)blockIdx.x * LET_TILE;
    uint32_t run = tile_off[blockIdx.x];
    for (uint32_t k0 = 0; k0 < LET_TILE; k0 += 256u) {
        const uint64_t i = base + k0 + threadIdx.x;
        const bool f = i < n && flag[i] != 0;
        const uint32_t b = __ballot_sync(0xffffffffu, f);
        if (lane == 0) wcnt[wid] = __popc(b);
        __syncthreads();
        uint32_t off = run, tot = 0u;
        for (uint32_t w = 0; w < 8u; ++w) { if (w < wid) off += wcnt[w]; tot += wcnt[w]; }
        if (f) out[off + __popc(b & ((1u << lane) - 1u))] = (uint32_t)i;
        run += tot;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(256) k_let_accumulate(float *__restrict__ acc, float *__restrict__ pot, const uint32_t *__restrict__ idx,
                                                        const float *__restrict__ pacc, const float *__restrict__ ppot, uint64_t m,
                                                        uint64_t n)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    const uint32_t i = idx[k];
    if (i >= n) return;      // (never written out of bounds; the host layer builds idx from its own lists)
    acc[3 * (uint64_t)i] += pacc[3 * k]; acc[3 * (uint64_t)i + 1] += pacc[3 * k + 1]; acc[3 * (uint64_t)i + 2] += pacc[3 * k + 2];
    if (pot && ppot) pot[i] += ppot[k];
}

__global__ void __launch_bounds__(256) k_ext_gather(const float *__restrict__ tpos, const float *__restrict__ tsoft,
                                                    const uint32_t *__restrict__ order, uint64_t n_t, float4 *__restrict__ ext)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_t) return;
    const uint32_t i = order[k];
    // R9: h = fl32(2.8 * eps), product formed in fp64 (as for the particles of the tree)
    ext[k] = make_float4(__ldg(tpos + 3 * (uint64_t)i), __ldg(tpos + 3 * (uint64_t)i + 1), __ldg(tpos + 3 * (uint64_t)i + 2),
                         __double2float_rn(__dmul_rn(2.8, (double)__ldg(tsoft + i))));
}

inline unsigned grid_for(uint64_t n, unsigned per) { return (unsigned)((n + per - 1) / per); }

}  // namespace

cudaError_t ogk_ext_gather(const float *tpos, const float *tsoft, const uint32_t *order, uint64_t n_t, float4 *ext,
                           cudaStream_t st)
{
    k_ext_gather<<<grid_for(n_t, 256), 256, 0, st>>>(tpos, tsoft, order, n_t, ext);
    return cudaGetLastError();
}

cudaError_t ogk_cell_hist(const uint64_t *keys, uint64_t n, uint32_t *hist, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(hist, 0, 32768 * sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    if (n) k_cell_hist<<<grid_for(n, 256), 256, 0, st>>>(keys, n, hist);
    return cudaGetLastError();
}

cudaError_t ogk_owner(const uint64_t *keys, uint64_t n, const uint32_t *S, uint32_t R, uint32_t *owner, cudaStream_t st)
{
    if (n) k_owner<<<grid_for(n, 256), 256, 0, st>>>(keys, n, S, R, owner);
    return cudaGetLastError();
}

cudaError_t ogk_let_mark(const float *tpos, uint64_t n_t, const float *boxes, uint32_t nb, float r_cut, float L,
                         uint8_t *flag, cudaStream_t st)
{
    if (n_t) k_let_mark<<<grid_for(n_t, 256), 256, nb * 6 * sizeof(float), st>>>(tpos, n_t, boxes, nb, r_cut, L, flag);
    return cudaGetLastError();
}

size_t ogk_flag_scratch_bytes(uint64_t n) { return ((n + LET_TILE - 1) / LET_TILE + 2) * sizeof(uint32_t); }

// ascending indices of the set flags -> out; the total is left at scratch[n_tiles] (DEVICE)
cudaError_t ogk_flag_compact(const uint8_t *flag, uint64_t n, uint32_t *out, uint32_t *scratch, uint32_t **total_dev,
                             cudaStream_t st)
{
    const uint32_t tiles = (uint32_t)((n + LET_TILE - 1) / LET_TILE);
    *total_dev = scratch + tiles;
    if (n == 0) return cudaMemsetAsync(scratch, 0, sizeof(uint32_t), st);
    k_flag_count<<<tiles, 256, 0, st>>>(flag, n, scratch);
    k_flag_scan<<<1, 1024, 0, st>>>(scratch, tiles);
    k_flag_fill<<<tiles, 256, 0, st>>>(flag, n, scratch, out);
    return cudaGetLastError();
}

cudaError_t ogk_let_accumulate(float *acc, float *pot, const uint32_t *idx, const float *pacc, const float *ppot, uint64_t m,
                               uint64_t n, cudaStream_t st)
{
    if (m) k_let_accumulate<<<grid_for(m, 256), 256, 0, st>>>(acc, pot, idx, pacc, ppot, m, n);
    return cudaGetLastError();
}
