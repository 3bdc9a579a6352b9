// sph.cu -- row f3 of SURVEY.md Sec. 8: SPH density / smoothing length on the gravity tree.
// PAPER.md:61 ("the SPH density module ... operates as an iterative process, aiming to determine a smoothing
// length containing a fixed number of neighbours"), :74 ("collects all neighbours within a sphere around the
// target particle and processes them in a separate evaluate function").  Readings R43..R47, DESIGN.md Sec. 12.
//
// k_sph_density: one warp per target.
//   1. radius H: 1.05 x the caller's h_guess, or from the deepest ancestor cell of the target that still holds n_des
//      particles (found by descending the target's own path from the root): the radius that would hold 1.5 n_des
//      at the cell's mean density;
//   2. COLLECT: the warp walks the tree (32 nodes per step from a warp-private stack in shared memory; a node is
//      opened when the nearest image of its tight AABB is within H of the target; children are contiguous) and
//      appends (r, m) of every particle with r < H to a candidate list in shared memory (ballot compaction);
//   3. N(H) < n_des: H *= 2^(1/3), back to 2.  The list does not fit: H *= 0.8, back to 2, from then on growing by
//      1.04 only (if the list overflows again before N(H) reaches n_des, OG_DEV_NGB_OVERFLOW is latched);
//   4. ROOT: N(h) = n_des on the list (every h <= H sees all its neighbours there): Newton steps kept inside a
//      bisection bracket, N and dN/dh summed by the lanes over their slices and reduced by shuffles (fixed order:
//      bit-reproducible); stops at |N - n_des| <= tol_n or when the bracket has collapsed to fp32 resolution;
//   5. rho = (8 / (pi h^3)) sum m w(r / h) with that h.
#include "og_internal.cuh"

namespace {

constexpr int SPH_WARPS = 4;
constexpr int SPH_CAP = 512;     // candidates per warp
constexpr int SPH_QCAP = 256;    // pending nodes per warp

struct __align__(16) SphSmem {
    float cr[SPH_CAP];           // distance to the target
    float cm[SPH_CAP];           // mass
    uint32_t q[SPH_QCAP];
};

struct SphArgs {
    const float4 *lo, *hi;
    const uint2 *info;
    const uint32_t *node_first, *node_count, *first_child;
    const uint8_t *nchild;
    const uint32_t *seed5;       // level-5 cell -> covering node (og_internal.cuh)
    const float4 *spos;
    const uint32_t *inv_perm, *perm;
    const uint32_t *active_idx;  // NULL: target k = sorted slot k, written at perm[k]
    const float *h_guess;        // NULL or [n_active] in the caller's order
    float *h_out, *rho_out, *nn_out;
    uint32_t n, n_active;
    float L, invL, n_des, tol_n;
    uint32_t *status;
    uint32_t *ticket;            // zeroed before the launch
};

__device__ __forceinline__ float sph_wrap(float d, float L, float invL) { return fmaf(-L, rintf(d * invL), d); }

// R43: w(u) and u w'(u) of the cubic spline with support u <= 1
__device__ __forceinline__ void sph_w(float u, float &w, float &uwp)
{
    if (u <= 0.5f) {
        w = fmaf(u * u, fmaf(6.0f, u, -6.0f), 1.0f);
        uwp = u * u * fmaf(18.0f, u, -12.0f);
    } else if (u <= 1.0f) {
        const float v = 1.0f - u;
        w = 2.0f * v * v * v;
        uwp = -6.0f * v * v * u;
    } else {
        w = 0.0f; uwp = 0.0f;
    }
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// N(h) and h dN/dh over the candidate list (R44): every lane returns the same bits
__device__ __forceinline__ void sph_number(const SphSmem &s, int cnt, float h, uint32_t lane, float &N, float &hdN)
{
    const float hinv = 1.0f / h;
    float a = 0.0f, b = 0.0f;
    for (int j = lane; j < cnt; j += 32) {
        float w, uwp;
        sph_w(s.cr[j] * hinv, w, uwp);
        a += w; b += uwp;
    }
    const float k = 32.0f / 3.0f;
    N = k * warp_sum(a);
    hdN = -k * warp_sum(b);    // dN/dh = -(32/3) sum w'(u) u / h
}

// No periodic image can matter if the sphere (padded) lies inside [0, L) on every axis: the scans then skip the wraps.
__device__ __forceinline__ bool sph_interior(const SphArgs &a, float px, float py, float pz, float H)
{
    const float e = H * (1.0f + 1.0e-5f) + 1.0e-6f * a.L;
    return px - e >= 0.0f && py - e >= 0.0f && pz - e >= 0.0f && px + e < a.L && py + e < a.L && pz + e < a.L;
}

// Step 2.  STORE: fills the candidate list with every particle closer than H to (px, py, pz) and returns their number,
// or -1 if the list or the node stack overflowed.  !STORE (the fallback of a target whose candidates do not fit the
// list): nothing is stored, the lanes add w, u w' and m w of the particles inside H = h to (sa, sb, sc) on the fly, and
// the node stack may use the whole per-warp area; -1 only if even that stack overflows.
template <bool STORE, bool WRAP>
__device__ int sph_scan(const SphArgs &a, SphSmem &s, float px, float py, float pz, float H, uint32_t lane, float &sa,
                        float &sb, float &sc)
{
    const float H2 = H * H;
    const float H2n = H2 * (1.0f + 1.0e-5f);      // nodes: conservative
    const float pad = 4.0e-7f * a.L;              // rounding of the box centre / half size
    const float hinv = 1.0f / H;
    const uint32_t lt = (1u << lane) - 1u;
    uint32_t *q = STORE ? s.q : reinterpret_cast<uint32_t *>(&s);
    const int qcap = STORE ? SPH_QCAP : (int)(sizeof(SphSmem) / sizeof(uint32_t));
    int qn = 1, cnt = 0;
    {
        // Entry points: the walk starts from the nodes that cover the level-5 cells the sphere's bounding box touches (at
        // most 3 x 3 x 3 of them when the sphere is smaller than a cell; found in the tree's cell table, each node once),
        // not from the root: the five upper levels of every walk are the same few nodes.
        const float e = H * (1.0f + 1.0e-5f) + 2.0e-6f * a.L;
        const float sc5 = 32.0f * a.invL;
        const int x0 = (int)floorf((px - e) * sc5), x1 = (int)floorf((px + e) * sc5);
        const int y0 = (int)floorf((py - e) * sc5), y1 = (int)floorf((py + e) * sc5);
        const int z0 = (int)floorf((pz - e) * sc5), z1 = (int)floorf((pz + e) * sc5);
        const int nx = x1 - x0 + 1, ny = y1 - y0 + 1, nz = z1 - z0 + 1;
        if (nx <= 3 && ny <= 3 && nz <= 3) {
            uint32_t node = 0xffffffffu;
            if ((int)lane < nx * ny * nz) {
                const int ix = (x0 + (int)lane % nx) & 31, iy = (y0 + ((int)lane / nx) % ny) & 31, iz = (z0 + (int)lane / (nx * ny)) & 31;
                uint32_t m = 0u;
#pragma unroll
                for (int b = 0; b < 5; ++b)
                    m |= (((uint32_t)ix >> b) & 1u) << (3 * b + 2) | (((uint32_t)iy >> b) & 1u) << (3 * b + 1) | (((uint32_t)iz >> b) & 1u) << (3 * b);
                node = __ldg(a.seed5 + m);
            }
            const bool have = node != 0xffffffffu;
            const uint32_t peers = __match_any_sync(0xffffffffu, node);
            const bool first = have && (peers & lt) == 0u;            // a leaf above level 5 covers several cells: once
            const uint32_t fb = __ballot_sync(0xffffffffu, first);
            if (first) q[__popc(fb & lt)] = node;
            qn = __popc(fb);
        } else if (lane == 0) {
            q[0] = 0u;
        }
    }
    __syncwarp();
    while (qn > 0) {
        const int take = min(qn, 32);
        qn -= take;
        bool hit = false;
        uint2 info = make_uint2(0u, 0u);
        if ((int)lane < take) {
            const uint32_t node = q[qn + lane];
            const float4 lo = __ldg(a.lo + node), hi = __ldg(a.hi + node);
            info = __ldg(a.info + node);
            float cx = 0.5f * (lo.x + hi.x) - px, cy = 0.5f * (lo.y + hi.y) - py, cz = 0.5f * (lo.z + hi.z) - pz;
            if (WRAP) { cx = sph_wrap(cx, a.L, a.invL); cy = sph_wrap(cy, a.L, a.invL); cz = sph_wrap(cz, a.L, a.invL); }
            const float dx = fmaxf(fabsf(cx) - (0.5f * (hi.x - lo.x) + pad), 0.0f);
            const float dy = fmaxf(fabsf(cy) - (0.5f * (hi.y - lo.y) + pad), 0.0f);
            const float dz = fmaxf(fabsf(cz) - (0.5f * (hi.z - lo.z) + pad), 0.0f);
            hit = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) <= H2n;
        }
        __syncwarp();
        const bool leaf = (info.y & OG_LEAF_BIT) != 0u;
        const uint32_t c = info.y & ~OG_LEAF_BIT;
        const uint32_t nch = (hit && !leaf) ? c : 0u;
        // Opened leaves.  Every lane takes ITS OWN leaf (<= 32 particles; the few larger ones below) and tests its particles
        // one after the other: the loads of all the leaves of the batch are in flight together (one L2 round trip per
        // batch instead of one per leaf).  The list keeps the order leaf by leaf (ascending lane), particle by particle.
        const bool small_leaf = hit && leaf && c <= 32u;
        uint32_t inmask = 0u;
        if (small_leaf) {
            for (uint32_t j = 0; j < c; ++j) {
                const float4 pq = __ldg(a.spos + info.x + j);
                float dx = pq.x - px, dy = pq.y - py, dz = pq.z - pz;
                if (WRAP) { dx = sph_wrap(dx, a.L, a.invL); dy = sph_wrap(dy, a.L, a.invL); dz = sph_wrap(dz, a.L, a.invL); }
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if (r2 < H2) {
                    if (STORE) {
                        inmask |= 1u << j;
                    } else {
                        float w, uwp;
                        sph_w(sqrtf(r2) * hinv, w, uwp);
                        sa += w; sb += uwp; sc = fmaf(pq.w, w, sc);
                        ++inmask;                    // (a count in this mode)
                    }
                }
            }
        }
        // one scan for both offsets: children pushed (high half, <= 8 x 32) and particles appended (low half, <= 32 x 32)
        const uint32_t mine = STORE ? (uint32_t)__popc(inmask) : inmask;
        const uint32_t both = (nch << 16) | mine;
        uint32_t run = both;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, run, o);
            if (lane >= (uint32_t)o) run += y;
        }
        const uint32_t tot2 = __shfl_sync(0xffffffffu, run, 31);
        const uint32_t total = tot2 >> 16, tot = tot2 & 0xffffu;
        if (qn + (int)total > qcap) return -1;
        {
            uint32_t *dst = q + qn + ((run - both) >> 16);
#pragma unroll
            for (uint32_t k = 0; k < 8u; ++k)
                if (k < nch) dst[k] = info.x + k;
        }
        qn += (int)total;
        if (STORE) {
            if (cnt + (int)tot > SPH_CAP) return -1;
            uint32_t at = (uint32_t)cnt + ((run - both) & 0xffffu);
            while (inmask) {
                const uint32_t j = (uint32_t)__ffs(inmask) - 1u;
                inmask &= inmask - 1u;
                const float4 pq = __ldg(a.spos + info.x + j);
                float dx = pq.x - px, dy = pq.y - py, dz = pq.z - pz;
                if (WRAP) { dx = sph_wrap(dx, a.L, a.invL); dy = sph_wrap(dy, a.L, a.invL); dz = sph_wrap(dz, a.L, a.invL); }
                s.cr[at] = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
                s.cm[at] = pq.w;
                ++at;
            }
        }
        cnt += (int)tot;
        // leaves with more than 32 particles (deepest level only): the warp takes them one by one, 32 particles at a time
        uint32_t lb = __ballot_sync(0xffffffffu, hit && leaf && c > 32u);
        while (lb) {
            const int src = __ffs(lb) - 1;
            lb &= lb - 1u;
            const uint32_t first = __shfl_sync(0xffffffffu, info.x, src);
            const uint32_t pc = __shfl_sync(0xffffffffu, c, src);
            for (uint32_t base = 0; base < pc; base += 32u) {
                bool in = false;
                float r2 = 0.0f, m = 0.0f;
                if (base + lane < pc) {
                    const float4 pq = __ldg(a.spos + first + base + lane);
                    const float dx = sph_wrap(pq.x - px, a.L, a.invL), dy = sph_wrap(pq.y - py, a.L, a.invL),
                                dz = sph_wrap(pq.z - pz, a.L, a.invL);
                    r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                    in = r2 < H2;
                    m = pq.w;
                }
                const uint32_t b = __ballot_sync(0xffffffffu, in);
                const int nb = __popc(b);
                if (STORE) {
                    if (cnt + nb > SPH_CAP) return -1;
                    if (in) {
                        const int p = cnt + __popc(b & lt);
                        s.cr[p] = sqrtf(r2);
                        s.cm[p] = m;
                    }
                } else if (in) {
                    float w, uwp;
                    sph_w(sqrtf(r2) * hinv, w, uwp);
                    sa += w; sb += uwp; sc = fmaf(m, w, sc);
                }
                cnt += nb;
            }
        }
        __syncwarp();
    }
    return cnt;
}

// The fallback evaluator: N(h), h dN/dh and sum m w by a walk of the tree with radius h.  false: stack overflow.
__device__ __forceinline__ bool sph_number_stream(const SphArgs &a, SphSmem &s, float px, float py, float pz, float h,
                                                  uint32_t lane, float &N, float &hdN, float &msum)
{
    float sa = 0.0f, sb = 0.0f, sc = 0.0f;
    const int cnt = sph_interior(a, px, py, pz, h) ? sph_scan<false, false>(a, s, px, py, pz, h, lane, sa, sb, sc)
                                                    : sph_scan<false, true>(a, s, px, py, pz, h, lane, sa, sb, sc);
    __syncwarp();
    const float k = 32.0f / 3.0f;
    N = k * warp_sum(sa); hdN = -k * warp_sum(sb); msum = warp_sum(sc);
    return cnt >= 0;
}

__global__ void __launch_bounds__(SPH_WARPS * 32) k_sph_density(const __grid_constant__ SphArgs a)
{
    __shared__ SphSmem sm[SPH_WARPS];
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    SphSmem &s = sm[wid];
    // targets are handed out four at a time by a ticket: a few targets cost a thousand times the typical one (their
    // kernel rim grazes a dense clump and every trial radius re-walks the tree), and with a fixed assignment the warps
    // that drew them finished long after the others
    uint32_t k = 0, kend = 0;
    for (;; ++k) {
        if (k >= kend) {
            if (lane == 0) k = atomicAdd(a.ticket, 4u);
            k = __shfl_sync(0xffffffffu, k, 0);
            kend = min(k + 4u, a.n_active);
            if (k >= a.n_active) break;
        }
        uint32_t slot, out;
        if (a.active_idx) {
            const uint32_t i = __ldg(a.active_idx + k);
            if (i >= a.n) { if (lane == 0) atomicOr(a.status, OG_DEV_BAD_INDEX); continue; }
            slot = __ldg(a.inv_perm + i); out = k;
        } else {
            slot = k; out = __ldg(a.perm + k);
        }
        const float4 p = __ldg(a.spos + slot);
        float H;
        if (a.h_guess) {
            H = 1.05f * __ldg(a.h_guess + out);     // (a previous h: N(H) >= n_des at the first try, almost always)
            if (!(H > 0.0f)) H = 1.0e-3f * a.L;
        } else {
            // deepest ancestor of the target with at least n_des particles (the root if there is none): its particle
            // count and side give the local density, hence the radius of a sphere that holds about 1.5 n_des
            uint32_t node = 0u, level = 0u, ncount = a.n;
            for (;;) {
                const uint32_t nc = __ldg(a.nchild + node);
                if (nc == 0u) break;
                const uint32_t fc = __ldg(a.first_child + node);
                uint32_t cf = 0xffffffffu, cc = 0u;
                if (lane < nc) { cf = __ldg(a.node_first + fc + lane); cc = __ldg(a.node_count + fc + lane); }
                const uint32_t mine = __ballot_sync(0xffffffffu, lane < nc && slot >= cf && slot < cf + cc);
                if (mine == 0u) break;
                const int src = __ffs(mine) - 1;
                const uint32_t ccnt = __shfl_sync(0xffffffffu, cc, src);
                if ((float)ccnt < a.n_des) break;
                node = fc + (uint32_t)src; ncount = ccnt; ++level;
            }
            const float l = a.L * __uint_as_float((127u - level) << 23);
            H = l * cbrtf(0.358f * a.n_des / (float)ncount);
        }
        const float hcap = 0.5f * a.L * (1.0f - 1.0e-6f);
        H = fminf(H, hcap);
        // steps 2, 3: a sphere that holds the root of N(h) = n_des and fits the list
        int cnt = 0;
        float NH = 0.0f, hdN = 0.0f;
        bool shrunk = false, regrown = false, fail = false;   // fail: pending nodes exceed even the fallback's stack
        float grow = 1.2599211f;
        for (int tries = 0; tries < 200; ++tries) {
            {
                float d0 = 0.f, d1 = 0.f, d2 = 0.f;
                cnt = sph_interior(a, p.x, p.y, p.z, H) ? sph_scan<true, false>(a, s, p.x, p.y, p.z, H, lane, d0, d1, d2)
                                                        : sph_scan<true, true>(a, s, p.x, p.y, p.z, H, lane, d0, d1, d2);
            }
            __syncwarp();
            if (cnt < 0) {
                if (regrown) break;            // no sphere both holds n_des and fits the list
                H *= 0.8f; shrunk = true; grow = 1.04f;
                continue;
            }
            sph_number(s, cnt, H, lane, NH, hdN);
            if (NH >= a.n_des || H >= hcap) break;
            regrown = shrunk;
            H = fminf(H * grow, hcap);
        }
        if (cnt < 0) {
            // the candidates of the sphere that holds the root do not fit the list (a target in a void next to a dense
            // clump: thousands of neighbours near the rim of its kernel): the same root search with every N(h) summed
            // by a walk of the tree
            float lo = 0.0f, hi = 0.0f, h = H, N = 0.0f, msum = 0.0f;      // hi = 0: no upper bound yet
            for (int it = 0; it < 400; ++it) {
                if (!sph_number_stream(a, s, p.x, p.y, p.z, h, lane, N, hdN, msum)) { fail = true; break; }
                if (fabsf(N - a.n_des) <= a.tol_n) break;
                if (N > a.n_des) hi = h; else lo = h;
                if (lo == 0.0f && hi != 0.0f && hi < 1.0e-12f * a.L) { fail = true; break; }   // no root: coincident pile
                float hn;
                if (hi == 0.0f) {
                    if (h >= hcap) break;
                    hn = fminf(h * 1.2599211f, hcap);
                } else {
                    if (hi - lo <= 2.4e-7f * hi) break;
                    hn = (hdN > 0.0f) ? h * (1.0f - (N - a.n_des) / hdN) : 0.0f;
                    if (!(hn > lo && hn < hi)) hn = 0.5f * (lo + hi);
                    if (hn == h) break;
                }
                h = hn;
            }
            if (lane == 0) {
                if (fail) { atomicOr(a.status, OG_DEV_NGB_OVERFLOW); h = 0.0f; N = 0.0f; msum = 0.0f; }
                const float hinv = fail ? 0.0f : 1.0f / h;
                a.h_out[out] = h;
                if (a.rho_out) a.rho_out[out] = 2.5464790894703255f * hinv * hinv * hinv * msum;
                if (a.nn_out) a.nn_out[out] = N;
            }
            __syncwarp();
            continue;
        }
        // step 4: root of N(h) = n_des in (0, H]; N is increasing in h
        float lo = 0.0f, hi = H, h = H, N = NH;
        bool noroot = false;       // more than 3 n_des / 32 particles coincide with the target: N(h) > n_des for every h
        if (NH >= a.n_des) {
            for (int it = 0; it < 100; ++it) {
                if (fabsf(N - a.n_des) <= a.tol_n) break;
                if (N > a.n_des) hi = h; else lo = h;
                if (lo == 0.0f && hi < 1.0e-12f * a.L) { noroot = true; break; }
                if (hi - lo <= 2.4e-7f * hi) break;
                float hn = (hdN > 0.0f) ? h * (1.0f - (N - a.n_des) / hdN) : 0.0f;     // Newton step
                if (!(hn > lo && hn < hi)) hn = 0.5f * (lo + hi);
                if (hn == h) break;
                h = hn;
                sph_number(s, cnt, h, lane, N, hdN);
            }
        }
        if (noroot) {
            if (lane == 0) {
                atomicOr(a.status, OG_DEV_NGB_OVERFLOW);
                a.h_out[out] = 0.0f;
                if (a.rho_out) a.rho_out[out] = 0.0f;
                if (a.nn_out) a.nn_out[out] = 0.0f;
            }
            __syncwarp();
            continue;
        }
        // step 5
        const float hinv = 1.0f / h;
        float sum = 0.0f;
        for (int j = lane; j < cnt; j += 32) {
            float w, uwp;
            sph_w(s.cr[j] * hinv, w, uwp);
            sum = fmaf(s.cm[j], w, sum);
        }
        sum = warp_sum(sum);
        if (lane == 0) {
            a.h_out[out] = h;
            if (a.rho_out) a.rho_out[out] = 2.5464790894703255f * hinv * hinv * hinv * sum;   // 8 / pi
            if (a.nn_out) a.nn_out[out] = N;
        }
        __syncwarp();
    }
}

}  // namespace

cudaError_t ogk_sph_density(const og_tree *t, const uint32_t *active_idx, uint64_t n_active, float n_des, float tol_n,
                            const float *h_guess, float *h_out, float *rho_out, float *nn_out, cudaStream_t st)
{
    SphArgs a;
    a.lo = t->node_lo; a.hi = t->node_hi; a.info = t->node_info;
    a.node_first = t->node_first; a.node_count = t->node_count; a.first_child = t->node_first_child;
    a.nchild = t->node_nchild;
    a.seed5 = t->cover + OG_COVER_L5;
    a.spos = t->spos; a.inv_perm = t->inv_perm; a.perm = t->perm;
    a.active_idx = active_idx; a.h_guess = h_guess;
    a.h_out = h_out; a.rho_out = rho_out; a.nn_out = nn_out;
    a.n = (uint32_t)t->n; a.n_active = (uint32_t)n_active;
    a.L = t->box; a.invL = 1.0f / t->box; a.n_des = n_des; a.tol_n = tol_n;
    a.status = t->d_status;
    a.ticket = t->d_status + 3;
    cudaError_t e0 = cudaMemsetAsync(a.ticket, 0, sizeof(uint32_t), st);
    if (e0 != cudaSuccess) return e0;
    int per_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sph_density, SPH_WARPS * 32, 0);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    const uint64_t want = (n_active + SPH_WARPS - 1) / SPH_WARPS;
    const uint64_t cap = (uint64_t)per_sm * (uint64_t)t->sm_count;
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    k_sph_density<<<grid, SPH_WARPS * 32, 0, st>>>(a);
    return cudaGetLastError();
}
