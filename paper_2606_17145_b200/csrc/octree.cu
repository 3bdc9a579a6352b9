// octree.cu -- rows a4 (canonical octree from sorted keys) and a5 (upward pass) of
// SURVEY.md Sec. 8(a).
//
// a4 (C3, R5..R7): cell (l, p) = sorted slots whose key >> (63 - 3l) == p.  Root = node 0;
// a node is a leaf iff count <= leaf_max or l == 21; otherwise it gets one child per
// non-empty octant, ascending octant; numbering is breadth-first, so children are contiguous.
// Built level by level in ONE persistent cooperative kernel (no host round trip), one pass and one grid
// synchronisation per level: every node finds its non-empty octants by a 7-way lock-step binary search on
// the octant digit, a single-pass scan (decoupled look-back over chunk totals) gives the children's BFS
// indices, and the children records are written in the same pass.  Integer work only; the result is unique.
//
// a5 (C4, R8..R11): leaves sum over their slots in slot order, internal nodes over their
// children in order, all in fp64 with separately rounded products and sums (__dmul_rn /
// __dadd_rn: no FMA contraction, so the sums are reproducible bit for bit); the record the
// walk reads is the fp32 rounding of those results (R9).
#include <cooperative_groups.h>
#include "og_internal.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int OCT_THREADS = 256;

struct OctArgs {
    const uint64_t *keys;
    uint32_t n;
    uint32_t leaf_max;
    uint32_t max_nodes;
    uint8_t *level;
    uint32_t *first;
    uint32_t *count;
    uint32_t *first_child;
    uint8_t *nchild;
    uint32_t *level_start;  // [24]
    uint32_t *status;
    unsigned long long *chunk_status;   // [ceil(max_nodes / OCT_THREADS) + 1], zeroed before the launch
};

// lb[o] (o = 1..7) = number of slots of [f, f + c) whose octant digit is < o.
__device__ __forceinline__ void octant_bounds(const uint64_t *__restrict__ keys, uint32_t f, uint32_t c,
                                              int shift, uint32_t lb[9])
{
    uint32_t base[7];
#pragma unroll
    for (int o = 0; o < 7; ++o) base[o] = 0;
    uint32_t m = c;
    while (m > 1) {
        const uint32_t half = m >> 1;
#pragma unroll
        for (int o = 0; o < 7; ++o) {
            const uint32_t dg = (uint32_t)(__ldg(keys + f + base[o] + half - 1) >> shift) & 7u;
            base[o] = (dg < (uint32_t)(o + 1)) ? base[o] + half : base[o];
        }
        m -= half;
    }
#pragma unroll
    for (int o = 0; o < 7; ++o) {
        const uint32_t dg = (uint32_t)(__ldg(keys + f + base[o]) >> shift) & 7u;
        lb[o + 1] = base[o] + ((dg < (uint32_t)(o + 1)) ? 1u : 0u);
    }
    lb[0] = 0;
    lb[8] = c;
}

__device__ __forceinline__ uint32_t block_excl_scan(uint32_t x, uint32_t *warp_buf, uint32_t *total)
{
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    __syncthreads();
    if (lane == 31) warp_buf[wid] = incl;
    __syncthreads();
    uint32_t woff = 0, tot = 0;
#pragma unroll
    for (uint32_t w = 0; w < OCT_THREADS / 32; ++w) {
        const uint32_t s = warp_buf[w];
        if (w < wid) woff += s;
        tot += s;
    }
    *total = tot;
    return woff + incl - x;
}

// Chunk status word of the decoupled look-back scan over the children counts of a level: bits 0..31 the value,
// bits 32..33 the flag (1 = the chunk's own total, 2 = inclusive prefix up to and including the chunk), bits 34.. a
// tag = level + 1, so that the words left by earlier levels (and the zeroed initial state) read as "not published".
#define OCT_FLAG_AGG 1ull
#define OCT_FLAG_INCL 2ull

__device__ __forceinline__ unsigned long long oct_ld(const unsigned long long *p)
{
    return *reinterpret_cast<const volatile unsigned long long *>(p);
}
__device__ __forceinline__ void oct_st(unsigned long long *p, unsigned long long v)
{
    *reinterpret_cast<volatile unsigned long long *>(p) = v;
}

__global__ void __launch_bounds__(OCT_THREADS)
k_octree(OctArgs a)
{
    cg::grid_group grid = cg::this_grid();
    __shared__ uint32_t warp_buf[OCT_THREADS / 32];
    __shared__ uint32_t carry_s;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, wid = tid >> 5;
    if (blockIdx.x == 0 && tid == 0) {
        a.level[0] = 0; a.first[0] = 0; a.count[0] = a.n;
        a.level_start[0] = 0;
        for (int k = 1; k < 24; ++k) a.level_start[k] = 1;
    }
    grid.sync();
    uint32_t beg = 0, end = 1;
    for (int lv = 0; lv <= OG_MAX_LEVEL; ++lv) {
        const uint32_t nl = end - beg;
        if (nl == 0) break;
        if (lv == OG_MAX_LEVEL) {  // deepest level: everything is a leaf
            for (uint32_t j = beg + blockIdx.x * OCT_THREADS + tid; j < end; j += gridDim.x * OCT_THREADS) {
                a.nchild[j] = 0; a.first_child[j] = 0;
            }
            break;
        }
        const int shift = 60 - 3 * lv;
        const uint32_t nchunks = (nl + OCT_THREADS - 1) / OCT_THREADS;
        const unsigned long long tag = (unsigned long long)(lv + 1) << 34;
        // One pass per level: every chunk of 256 nodes finds its nodes' octant boundaries (kept in registers),
        // scans the children counts inside the chunk, obtains the number of children of all earlier chunks by a
        // decoupled look-back over the published chunk totals, and writes its children at once.  A block takes its
        // chunks in ascending order and all blocks are resident (cooperative launch), so the look-back always
        // finds its predecessors in progress or done.
        for (uint32_t ch = blockIdx.x; ch < nchunks; ch += gridDim.x) {
            const uint32_t node = beg + ch * OCT_THREADS + tid;
            uint32_t nc = 0, f = 0, c = 0;
            uint32_t lb[9];
            if (node < end) {
                c = a.count[node];
                f = a.first[node];
                if (c > a.leaf_max) {
                    octant_bounds(a.keys, f, c, shift, lb);
#pragma unroll
                    for (int o = 0; o < 8; ++o) nc += (lb[o + 1] > lb[o]) ? 1u : 0u;
                }
            }
            uint32_t tot;
            const uint32_t off = block_excl_scan(nc, warp_buf, &tot);
            if (wid == 0) {
                if (lane == 0) oct_st(a.chunk_status + ch, tag | ((ch == 0 ? OCT_FLAG_INCL : OCT_FLAG_AGG) << 32) | tot);
                uint32_t excl = 0;
                if (ch > 0) {
                    for (int64_t base = (int64_t)ch - 1;; base -= 32) {
                        const int64_t idx = base - (int64_t)lane;
                        unsigned long long sw;
                        do {
                            sw = (idx >= 0) ? oct_ld(a.chunk_status + idx) : (tag | (OCT_FLAG_INCL << 32));
                        } while (!__all_sync(0xffffffffu, (sw >> 34) == (tag >> 34)));
                        const uint32_t incl_lanes = __ballot_sync(0xffffffffu, ((sw >> 32) & 3ull) == OCT_FLAG_INCL);
                        const uint32_t upto = incl_lanes ? (uint32_t)(__ffs(incl_lanes) - 1) : 31u;   // nearest inclusive prefix
                        uint32_t v = (lane <= upto) ? (uint32_t)sw : 0u;
#pragma unroll
                        for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                        excl += v;
                        if (incl_lanes) break;
                    }
                    if (lane == 0) oct_st(a.chunk_status + ch, tag | (OCT_FLAG_INCL << 32) | (excl + tot));
                }
                if (lane == 0) {
                    carry_s = excl;
                    if (ch == nchunks - 1) {   // the level's total: where the next level ends
                        uint64_t new_end = (uint64_t)end + excl + tot;
                        if (new_end > a.max_nodes) {  // R6: latch the overflow, stop splitting
                            atomicOr(a.status, OG_DEV_NODE_OVERFLOW);
                            new_end = end;
                        }
                        for (int k = lv + 2; k < 24; ++k) a.level_start[k] = (uint32_t)new_end;
                    }
                }
            }
            __syncthreads();
            if (node < end) {
                uint32_t child = end + carry_s + off;
                const bool fits = (uint64_t)child + nc <= (uint64_t)a.max_nodes;   // (else the level is undone below)
                a.nchild[node] = (uint8_t)(fits ? nc : 0u);
                a.first_child[node] = (nc && fits) ? child : 0u;
                if (nc && fits) {
#pragma unroll
                    for (int o = 0; o < 8; ++o) {
                        const uint32_t cc = lb[o + 1] - lb[o];
                        if (cc) {
                            a.level[child] = (uint8_t)(lv + 1);
                            a.first[child] = f + lb[o];
                            a.count[child] = cc;
                            ++child;
                        }
                    }
                }
            }
            __syncthreads();   // carry_s, warp_buf are reused by the block's next chunk
        }
        grid.sync();
        const uint32_t new_end = *((volatile uint32_t *)&a.level_start[lv + 2]);
        if ((*((volatile uint32_t *)a.status) & OG_DEV_NODE_OVERFLOW) != 0) {
            // the node capacity is exceeded at this level: its nodes stay leaves (the status is latched)
            for (uint32_t j = beg + blockIdx.x * OCT_THREADS + tid; j < end; j += gridDim.x * OCT_THREADS) {
                a.nchild[j] = 0; a.first_child[j] = 0;
            }
            break;
        }
        beg = end;
        end = new_end;
    }
}

// ---- a5 upward pass ----------------------------------------------------------------------
struct UpArgs {
    const uint64_t *keys;
    const float4 *spos;
    const float *sh;
    float box;
    const uint8_t *level;
    const uint32_t *first;
    const uint32_t *count;
    const uint32_t *first_child;
    const uint8_t *nchild;
    const uint32_t *level_start;
    double4 *sums;      // (M, sum m x, sum m y, sum m z) per node, fp64
    float4 *com, *cell, *lo, *hi;
    uint2 *info;
    uint4 *rec;         // packed walk records, 3 x 16 B per node
    uint32_t *status;
};

__device__ __forceinline__ uint32_t og_compact3(uint64_t x)
{
    x &= 0x1249249249249249ull;
    x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
    x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
    x = (x ^ (x >> 8)) & 0x001f0000ff0000ffull;
    x = (x ^ (x >> 16)) & 0x001f00000000ffffull;
    x = (x ^ (x >> 32)) & 0x1fffffull;
    return (uint32_t)x;
}

// Writes every record of a finished node: the fp64 sums (read by the parent), the fp32 records (R9) and the packed
// walk record n0, n1, n2 (og_internal.cuh).  R and ng are bounds used only by conservative tests of the walk, so they
// are rounded up.
__device__ __forceinline__ void up_store(const UpArgs &a, uint32_t j, int lv, float4 cc, uint2 info, double M, double ax,
                                         double ay, double az, float3 lo, float3 hi, float hm)
{
    a.sums[j] = make_double4(M, ax, ay, az);
    const float4 s = make_float4(__double2float_rn(__ddiv_rn(ax, M)), __double2float_rn(__ddiv_rn(ay, M)),
                                 __double2float_rn(__ddiv_rn(az, M)), __double2float_rn(M));
    a.com[j] = s;
    a.cell[j] = cc;
    a.info[j] = info;
    a.lo[j] = make_float4(lo.x, lo.y, lo.z, hm);
    a.hi[j] = make_float4(hi.x, hi.y, hi.z, 0.0f);
    const double ex = fmax((double)s.x - (double)lo.x, (double)hi.x - (double)s.x),
                 ey = fmax((double)s.y - (double)lo.y, (double)hi.y - (double)s.y),
                 ez = fmax((double)s.z - (double)lo.z, (double)hi.z - (double)s.z);
    const float R = __double2float_ru(sqrt(ex * ex + ey * ey + ez * ez) * (1.0 + 1e-6));
    const double lim = 0.6 * (double)cc.w;
    const double gx = lim + fabs((double)s.x - (double)cc.x), gy = lim + fabs((double)s.y - (double)cc.y),
                 gz = lim + fabs((double)s.z - (double)cc.z);
    const float rg = __double2float_ru(sqrt(gx * gx + gy * gy + gz * gz) * (1.0 + 1e-6));
    const uint32_t leaf = (info.y & OG_LEAF_BIT) ? 1u : 0u;
    const uint32_t cnt = info.y & ~OG_LEAF_BIT;
    if (cnt >= (1u << 26)) atomicOr(a.status, OG_DEV_NODE_OVERFLOW);   // does not fit the packed record
    const uint32_t meta = ((uint32_t)lv << 27) | (leaf << 26) | (cnt & 0x03ffffffu);
    uint4 *r = a.rec + 3 * (size_t)j;
    r[0] = make_uint4(__float_as_uint(s.x), __float_as_uint(s.y), __float_as_uint(s.z), __float_as_uint(s.w));
    r[1] = make_uint4(__float_as_uint(R), __float_as_uint(fmaxf(rg, hm)), info.x, meta);
    r[2] = make_uint4(__float_as_uint(cc.x), __float_as_uint(cc.y), __float_as_uint(cc.z), __float_as_uint(hm));
}

// geometric centre and side of the cell of node (level lv, first slot f): (c_x, c_y, c_z, l)
__device__ __forceinline__ float4 up_cell(const UpArgs &a, int lv, uint32_t f)
{
    const uint64_t key = __ldg(a.keys + f);
    const double l = ldexp((double)a.box, -lv);
    const int sh = OG_MAX_LEVEL - lv;
    const uint32_t px = lv ? (og_compact3(key >> 2) >> sh) : 0u;
    const uint32_t py = lv ? (og_compact3(key >> 1) >> sh) : 0u;
    const uint32_t pz = lv ? (og_compact3(key) >> sh) : 0u;
    return make_float4(__double2float_rn(__dmul_rn((double)px + 0.5, l)), __double2float_rn(__dmul_rn((double)py + 0.5, l)),
                       __double2float_rn(__dmul_rn((double)pz + 0.5, l)), __double2float_rn(l));
}

__global__ void __launch_bounds__(OCT_THREADS)
k_upward(UpArgs a)
{
    cg::grid_group grid = cg::this_grid();
    const uint32_t n_nodes = a.level_start[22];
    const uint32_t stride = gridDim.x * OCT_THREADS;
    const uint32_t t0 = blockIdx.x * OCT_THREADS + threadIdx.x;
    // (A) leaves (every level at once): sums over their slots in slot order, all records
    for (uint32_t j = t0; j < n_nodes; j += stride) {
        if (a.nchild[j] != 0) continue;
        const int lv = a.level[j];
        const uint32_t f = a.first[j], c = a.count[j];
        double M = 0.0, ax = 0.0, ay = 0.0, az = 0.0;
        float4 p = __ldg(a.spos + f);
        float3 lo = make_float3(p.x, p.y, p.z), hi = lo;
        float hm = __ldg(a.sh + f);
        for (uint32_t s = f; s < f + c; ++s) {
            p = __ldg(a.spos + s);
            const double m = (double)p.w;
            M = __dadd_rn(M, m);
            ax = __dadd_rn(ax, __dmul_rn(m, (double)p.x));
            ay = __dadd_rn(ay, __dmul_rn(m, (double)p.y));
            az = __dadd_rn(az, __dmul_rn(m, (double)p.z));
            lo.x = fminf(lo.x, p.x); lo.y = fminf(lo.y, p.y); lo.z = fminf(lo.z, p.z);
            hi.x = fmaxf(hi.x, p.x); hi.y = fmaxf(hi.y, p.y); hi.z = fmaxf(hi.z, p.z);
            hm = fmaxf(hm, __ldg(a.sh + s));
        }
        up_store(a, j, lv, up_cell(a, lv, f), make_uint2(f, c | OG_LEAF_BIT), M, ax, ay, az, lo, hi, hm);
    }
    // (B) internal nodes, deepest level first: sums over the children in order, all records
    int max_lv = 0;
    for (int lv = 0; lv <= OG_MAX_LEVEL; ++lv)
        if (a.level_start[lv + 1] > a.level_start[lv]) max_lv = lv;
    for (int lv = max_lv - 1; lv >= 0; --lv) {
        grid.sync();
        const uint32_t beg = a.level_start[lv], end = a.level_start[lv + 1];
        for (uint32_t j = beg + t0; j < end; j += stride) {
            const uint32_t nc = a.nchild[j];
            if (nc == 0) continue;
            const uint32_t fc = a.first_child[j];
            double M = 0.0, ax = 0.0, ay = 0.0, az = 0.0;
            // children were written by other blocks in this launch: read them past L1
            float4 l4 = __ldcg(a.lo + fc), h4 = __ldcg(a.hi + fc);
            float3 lo = make_float3(l4.x, l4.y, l4.z), hi = make_float3(h4.x, h4.y, h4.z);
            float hm = l4.w;
            for (uint32_t ch = fc; ch < fc + nc; ++ch) {
                const double2 *sp = reinterpret_cast<const double2 *>(a.sums + ch);
                const double2 s0 = __ldcg(sp), s1 = __ldcg(sp + 1);
                M = __dadd_rn(M, s0.x);
                ax = __dadd_rn(ax, s0.y); ay = __dadd_rn(ay, s1.x); az = __dadd_rn(az, s1.y);
                l4 = __ldcg(a.lo + ch); h4 = __ldcg(a.hi + ch);
                lo.x = fminf(lo.x, l4.x); lo.y = fminf(lo.y, l4.y); lo.z = fminf(lo.z, l4.z);
                hi.x = fmaxf(hi.x, h4.x); hi.y = fmaxf(hi.y, h4.y); hi.z = fmaxf(hi.z, h4.z);
                hm = fmaxf(hm, l4.w);
            }
            up_store(a, j, lv, up_cell(a, lv, a.first[j]), make_uint2(fc, nc), M, ax, ay, az, lo, hi, hm);
        }
    }
}

// cover[off(l) + m] (l = 0..5, off(l) = (8^l - 1) / 7, m = Morton index of the cell at level l) = the node that covers
// that cell: the node of level l, or the leaf above it; 0xffffffff for a cell without particles.  One thread per node of
// the levels 0..5.  The neighbour walk of og_sph_density enters the tree at the level-5 cells around its target (sph.cu).
__global__ void __launch_bounds__(256)
k_cover(const uint64_t *__restrict__ keys, const uint8_t *__restrict__ level, const uint32_t *__restrict__ first,
        const uint8_t *__restrict__ nchild, const uint32_t *__restrict__ level_start, uint32_t *__restrict__ cover)
{
    const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= level_start[6]) return;
    const uint32_t lv = level[j];
    const uint32_t m5 = (uint32_t)(keys[first[j]] >> 48);
    const uint32_t off[6] = {0u, 1u, 9u, 73u, 585u, 4681u};
    cover[off[lv] + (m5 >> (3u * (5u - lv)))] = j;
    if (nchild[j] != 0u) return;
    for (uint32_t l = lv + 1u; l <= 5u; ++l) {      // a leaf covers every cell below it
        const uint32_t sh = 3u * (l - lv);
        const uint32_t m0 = (m5 >> (3u * (5u - lv))) << sh;
        for (uint32_t m = m0; m < m0 + (1u << sh); ++m) cover[off[l] + m] = j;
    }
}

int coop_grid(const void *kernel, int threads, int sm_count)
{
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, 0) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    if (per_sm > 8) per_sm = 8;
    return per_sm * sm_count;
}

}  // namespace

size_t ogk_octree_scratch_bytes(uint32_t max_nodes)
{
    const size_t chunks = ((size_t)max_nodes + OCT_THREADS - 1) / OCT_THREADS + 1;
    return ((chunks * sizeof(unsigned long long) + 255) & ~(size_t)255) + (size_t)max_nodes * sizeof(double4);
}

cudaError_t ogk_octree_upward(og_tree *t, void *scratch, cudaStream_t st)
{
    const size_t chunks = ((size_t)t->max_nodes + OCT_THREADS - 1) / OCT_THREADS + 1;
    unsigned long long *chunk_status = reinterpret_cast<unsigned long long *>(scratch);
    double4 *sums = reinterpret_cast<double4 *>(reinterpret_cast<char *>(scratch) +
                                                ((chunks * sizeof(unsigned long long) + 255) & ~(size_t)255));
    cudaError_t e = cudaMemsetAsync(chunk_status, 0, chunks * sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    OctArgs oa{t->keys, (uint32_t)t->n, t->prm.leaf_max, t->max_nodes, t->node_level, t->node_first,
               t->node_count, t->node_first_child, t->node_nchild, t->d_level_start, t->d_status,
               chunk_status};
    void *args1[] = {&oa};
    e = cudaLaunchCooperativeKernel((const void *)k_octree,
                                                dim3(coop_grid((const void *)k_octree, OCT_THREADS, t->sm_count)),
                                                dim3(OCT_THREADS), args1, 0, st);
    if (e != cudaSuccess) return e;
    UpArgs ua{t->keys, t->spos, t->sh, t->box, t->node_level, t->node_first, t->node_count,
              t->node_first_child, t->node_nchild, t->d_level_start, sums, t->node_com, t->node_cell,
              t->node_lo, t->node_hi, t->node_info, t->node_rec, t->d_status};
    void *args2[] = {&ua};
    e = cudaLaunchCooperativeKernel((const void *)k_upward,
                                    dim3(coop_grid((const void *)k_upward, OCT_THREADS, t->sm_count)),
                                    dim3(OCT_THREADS), args2, 0, st);
    return e;
}

// The cell table is written on first use (og_sph_density): a gravity-only step does not pay for it.
cudaError_t ogk_cover(const og_tree *t, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(t->cover, 0xff, 37449 * sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    k_cover<<<(37449 + 255) / 256, 256, 0, st>>>(t->keys, t->node_level, t->node_first, t->node_nchild, t->d_level_start, t->cover);
    return cudaGetLastError();
}
