// walk.cu -- rows a6 (short-range tree walk) and a7 (scatter to the caller's order) of
// SURVEY.md Sec. 8(a).  PAPER.md:59 (a tree walk per active particle), :74 (per-node
// interaction and opening criterion).
//
// k_walk_group (the product path): one warp walks the tree for a group of 32 targets that are
// consecutive in Morton order.  The warp traverses the UNION of its lanes' walks, but every
// lane accepts / opens exactly the nodes its own serial walk would (C6): each pending entry
// carries a 32-bit lane mask = the lanes that opened the parent.  Per iteration the warp pops
// up to 32 child nodes from a shared-memory stack of (first, count, mask) ranges and lane k
// loads node k (3 x LDG.128 of the packed walk record, children are contiguous) and classifies
// it against the GROUP (bounding box of the 32 targets, range of a_old, largest h): dropped by
// the cutoff box, opened by every target, accepted by every target, or undecided.  Undecided
// nodes are staged in shared memory and tested by all lanes, two per loop iteration (broadcast
// LDS.128, branch-free; the rare lanes inside a guard region or within OG_BAND of a threshold take
// the exact path); a 32 x 32 bit transpose of the per-lane "open" words yields the masks of the
// children.  Accepted nodes and the particles of opened leaves (after a group-level cutoff test
// and an exact periodic shift to the group's image) are staged in a shared-memory ring of GW_NSEG
// segments of 32 sources; every lane walks the set bits of its OWN words W[seg][lane], two
// sources per iteration, and may lag up to a whole ring behind the producer, so a lane idles
// only when it has nothing left in the ring.  The split factors T, E are evaluated in registers
// (polynomial x ex2, walk_math.cuh).  Results are written straight to the caller's order (a7
// fused).  DESIGN.md Sec. 5 has the measured per-group counts and the instruction budget.
#include "walk_math.cuh"

namespace {

struct WalkArgs {
    const float4 *com, *cell, *lo, *hi;   // full node records (exact path, simple walk); com doubles as n0
    const uint2 *info;
    const uint4 *rec;          // packed walk records (n0, n1, n2), 48 contiguous bytes per node, og_internal.cuh
    const float4 *spos;
    const float *sh;
    const uint32_t *tgt_slot;  // NULL -> identity
    const float4 *ext;         // row f4: NULL, or EXTERNAL targets (x, y, z, h) in walk order (not particles of the tree:
                               // no slot, nothing excluded); tgt_slot is NULL then
    const uint32_t *tgt_out;   // position in the caller's order
    const float *a_old;
    float *acc_out;
    float *pot_out;
    uint32_t n_active;
    uint32_t n_groups;
    uint32_t *work;            // dynamic group counter
    uint32_t *status;
    unsigned long long *counters;
    uint32_t *spill;
    uint32_t spill_cap;        // entries per warp
    uint32_t stack_cap;        // ranges kept in shared memory before half of them are spilled (<= GW_STACK, even)
    const uint32_t *sel_flag;  // device flag: this launch runs iff *sel_flag == sel (NULL: always); see launch()
    uint32_t sel;
    uint32_t *cost;            // OG_COUNT: interactions evaluated per target (caller's order), or NULL
    WalkConst c;
};

__device__ __forceinline__ NodeRec load_node(const WalkArgs &a, uint32_t j)
{
    NodeRec n;
    n.com = __ldg(a.com + j);
    n.cell = __ldg(a.cell + j);
    n.lo = __ldg(a.lo + j);
    n.hi = __ldg(a.hi + j);
    return n;
}

__device__ __forceinline__ Target load_target(const WalkArgs &a, uint32_t k, uint32_t &out, bool geom)
{
    Target t;
    out = __ldg(a.tgt_out + k);
    if (a.ext != nullptr) {
        const float4 p = __ldg(a.ext + k);
        t.x = p.x; t.y = p.y; t.z = p.z; t.h = p.w;
        t.slot = 0xffffffffu;      // equals no particle's slot: the self exclusion never fires
    } else {
        const uint32_t slot = a.tgt_slot ? __ldg(a.tgt_slot + k) : k;
        const float4 p = __ldg(a.spos + slot);
        t.x = p.x; t.y = p.y; t.z = p.z;
        t.h = __ldg(a.sh + slot);
        t.slot = slot;
    }
    t.aold = geom ? 0.0f : __ldg(a.a_old + out);
    t.A = a.c.alpha * t.aold;
    return t;
}

// -------------------------------------------------------------------------------------------
#ifndef OG_GW_WARPS
#define OG_GW_WARPS 8
#endif
#ifndef OG_GW_MINBLOCKS
#define OG_GW_MINBLOCKS 2
#endif
#ifndef OG_GW_NSEG
#define OG_GW_NSEG 8
#endif
#ifndef OG_GW_SPARSE_G
#define OG_GW_SPARSE_G 8   // targets per warp for sparse active subsets (4, 8 or 16; zoom: 31.9 / 31.3 / 36.7 ms)
#endif
#ifndef OG_GW_STACK
#define OG_GW_STACK 256
#endif
#ifndef OG_CONSUME_FOUR
#define OG_CONSUME_FOUR 1   // two takes (4 sources) per consume iteration: nfw256 49.2 -> 48.2 ms
#endif
constexpr int GW_WARPS = OG_GW_WARPS;           // warps per block
constexpr int GW_THREADS = GW_WARPS * 32;
constexpr int GW_STACK = OG_GW_STACK;         // node-range stack entries per warp in shared memory
constexpr int GW_PLIST = 64;          // particle-range list entries per warp
constexpr int GW_NSEG = OG_GW_NSEG;            // 32-source segments in the per-warp source ring (power of two)

constexpr uint32_t GW_DUMMY = GW_NSEG * 32;   // ring slot of a source at (1e18, 1e18, 1e18) with mass 0

#define SEG_PART 2u      // particle segment (else node segment); only the counters care

// Per-warp working set.  Sources (accepted nodes and particles of opened leaves) are
// buffered in `ring_*` in segments of 32 slots; W[seg][lane] has bit j set iff lane's target interacts
// with slot j of the segment.  Each lane later walks its OWN set bits (per-lane compaction), so a lane
// is idle only when its list is shorter than the longest one of the buffered window.
struct __align__(16) WarpSmem {
    float4 ring_pos[GW_NSEG * 32 + 1];  // (x', y', z', G m): pre-shifted to the group's periodic image; + the dummy slot
    float ring_h[GW_NSEG * 32 + 4];     // softening length of the source (0 for nodes)
    uint32_t W[GW_NSEG][32];
    // undecided nodes of a batch, in pairs (for the packed test loop): pair p = nodes 2p, 2p + 1 of the batch's
    // undecided nodes in lane order; xq[p] = (x0, x1, y0, y1), (z0, z1, cull2_0, cull2_1),
    // (lhs_0 (1 - band), lhs_1 (1 - band), lhs_0 (1 + band), lhs_1 (1 + band)), (near2_0, near2_1, mask_0, mask_1)
    float4 xq[16][4];
    float4 xn_cel[32];                  // (c', l) per undecided node (guards, exact path)
    float xn_hm2[32];                   // h_max^2
    uint32_t xn_u[32];                  // undecided node: node index; node accepted by all: its target mask
    uint32_t seg_flags[GW_NSEG];
    uint32_t st_start[GW_STACK], st_cnt[GW_STACK], st_mask[GW_STACK];
    uint32_t pl_start[GW_PLIST], pl_cnt[GW_PLIST], pl_mask[GW_PLIST];
};

// w |= bit if p, as one predicated instruction (the compiler's select + or costs two)
__device__ __forceinline__ void or_if(uint32_t &w, const uint32_t bit, const bool p)
{
    asm("{\n\t.reg .pred q;\n\tsetp.ne.u32 q, %2, 0;\n\t@q or.b32 %0, %0, %1;\n\t}" : "+r"(w) : "r"(bit), "r"((uint32_t)p));
}

// index of the most significant set bit, 0xffffffff if x == 0 (one FLO; __ffs costs BREV + FLO)
__device__ __forceinline__ uint32_t og_bfind(uint32_t x)
{
    uint32_t r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}
// x << n with n >= 32 giving 0 (PTX shl clamps; the C++ operator is undefined there)
__device__ __forceinline__ uint32_t og_shl(uint32_t x, uint32_t n)
{
    uint32_t r;
    asm("shl.b32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(n));
    return r;
}

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// 32 x 32 bit-matrix transpose across the warp: lane j passes row j (bit t = element (j, t)); lane t
// receives column t (bit j = element (j, t)).  Five butterfly stages.
__device__ __forceinline__ uint32_t transpose32(uint32_t x, uint32_t lane)
{
#pragma unroll
    for (int k = 16; k >= 1; k >>= 1) {
        const uint32_t m = (k == 16) ? 0x0000ffffu : (k == 8) ? 0x00ff00ffu : (k == 4) ? 0x0f0f0f0fu
                         : (k == 2) ? 0x33333333u : 0x55555555u;
        const uint32_t y = __shfl_xor_sync(0xffffffffu, x, k);
        x = (lane & k) ? (((y >> k) & m) | (x & ~m)) : ((x & m) | ((y << k) & ~m));
    }
    return x;
}

// Pops up to 32 items from the top of a range list.  Lane j < total receives item index and
// mask.  Fully consumed entries are removed; a partially consumed one is shortened in place.
__device__ __forceinline__ uint32_t pop_items(uint32_t *s_start, uint32_t *s_cnt, uint32_t *s_mask, int &top,
                                              uint32_t lane, uint32_t &item, uint32_t &imask)
{
    const int e = top - 1 - (int)lane;
    uint32_t c = 0, st = 0, mk = 0;
    if (e >= 0) { c = s_cnt[e]; st = s_start[e]; mk = s_mask[e]; }
    const uint32_t cc = min(c, 32u);
    uint32_t incl = cc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= (uint32_t)o) incl += y;
    }
    const uint32_t excl = incl - cc;
    const uint32_t take = (excl < 32u) ? min(c, 32u - excl) : 0u;
    const bool full = (e >= 0) && (take == c);
    if (e >= 0 && take > 0 && take < c) { s_start[e] = st + take; s_cnt[e] = c - take; }
    top -= __popc(__ballot_sync(0xffffffffu, full));
    const uint32_t total = min(__shfl_sync(0xffffffffu, incl, 31), 32u);
    const uint32_t S = __reduce_or_sync(0xffffffffu, take > 0 ? (1u << excl) : 0u);
    const int src = __popc(S & (0xffffffffu >> (31 - lane))) - 1;
    const uint32_t sst = __shfl_sync(0xffffffffu, st, src & 31);
    const uint32_t sex = __shfl_sync(0xffffffffu, excl, src & 31);
    imask = __shfl_sync(0xffffffffu, mk, src & 31);
    item = sst + (lane - sex);
    __syncwarp();
    return total;
}

// Warp-uniform description of the 32 targets of a group: bounding box (centre, half size), range
// of a_old, largest softening length.
struct GroupInfo {
    float gcx, gcy, gcz, ghx, ghy, ghz;
    float amin, amax, hmax2;
};

enum { CL_DROP = 0, CL_OPEN = 1, CL_ACCEPT = 2, CL_GENERIC = 3 };

#define OG_GM 1.0e-4f   // relative safety margin of the group-level (conservative) classifications

// Group-level classification of one node by the lane that loaded it, from the packed
// walk record n0 = (s, M), n1 = (R, ng, first, meta): R = largest distance from s to a corner of the
// node's AABB, ng = max(h_max, largest |x - s| of a point inside the 0.6 l guard box).  Every outcome
// other than CL_GENERIC is one that EVERY target of the group would reach on its own:
//   CL_DROP    no target is within r_cut + R of s (then no particle of the node is within r_cut of any
//              target and r_COM > r_cut: the node contributes nothing whether accepted or opened, R17),
//              or all accept it but none is within r_cut of s;
//   CL_OPEN    every target opens it by the relative / geometric criterion (largest possible r, a_old);
//   CL_ACCEPT  every target accepts it (criterion at the smallest possible r and a_old, and no target
//              is within ng or its own h of s, so no guard can fire).
// `sc` = (s - k L, G M): one exact periodic shift serves all targets if `shifted` (k = 0, or k = +1 with
// s >= L/2), else sc holds s itself and the lanes wrap.
template <bool GEOM>
__device__ __forceinline__ int classify_node(const float4 n0, float R, float ng, float l, const GroupInfo &g,
                                             const WalkConst &c, float4 &sc, float &lhs, float &near2, float &cull2,
                                             bool &shifted, float &kx, float &ky, float &kz)
{
    kx = rintf((n0.x - g.gcx) * c.invL); ky = rintf((n0.y - g.gcy) * c.invL); kz = rintf((n0.z - g.gcz) * c.invL);
    const float adx = fabsf(fmaf(-c.L, kx, n0.x - g.gcx)), ady = fabsf(fmaf(-c.L, ky, n0.y - g.gcy)),
                adz = fabsf(fmaf(-c.L, kz, n0.z - g.gcz));
    const float nx = fmaxf(adx - g.ghx, 0.f), ny = fmaxf(ady - g.ghy, 0.f), nz = fmaxf(adz - g.ghz, 0.f);
    const float fx = adx + g.ghx, fy = ady + g.ghy, fz = adz + g.ghz;
    const float rmin2 = fmaf(nz, nz, fmaf(ny, ny, nx * nx));
    const float rmax2 = fmaf(fz, fz, fmaf(fy, fy, fx * fx));
    const float rc = c.cull_r + R;
    cull2 = rc * rc;
    if (rmin2 > cull2) return CL_DROP;
    const float l2 = l * l;
    const float GM = c.G * n0.w;
    float rhs_max, rhs_min;
    if (GEOM) {
        lhs = l2; rhs_max = c.theta2 * rmax2; rhs_min = c.theta2 * rmin2;
    } else {
        lhs = GM * l2;
        rhs_max = c.alpha * g.amax * rmax2 * rmax2;
        rhs_min = c.alpha * g.amin * rmin2 * rmin2;
    }
    if (lhs > rhs_max * (1.0f + OG_GM)) return CL_OPEN;
    // x - k L is exact for k = 0 and, by Sterbenz, for k = 1 with x >= L/2
    const float hL = 0.5f * c.L;
    shifted = fmaxf(fx, fmaxf(fy, fz)) < hL * (1.0f - OG_GM) && (kx == 0.0f || (kx == 1.0f && n0.x >= hL)) &&
              (ky == 0.0f || (ky == 1.0f && n0.y >= hL)) && (kz == 0.0f || (kz == 1.0f && n0.z >= hL));
    if (shifted) sc = make_float4(fmaf(-c.L, kx, n0.x), fmaf(-c.L, ky, n0.y), fmaf(-c.L, kz, n0.z), GM);
    else sc = make_float4(n0.x, n0.y, n0.z, GM);
    // no guard (R15 / R16) can fire for a target farther than this from s: ng covers the guard box and the
    // node's h_max, the group's largest own h covers every target's softening length
    near2 = fmaxf(ng * ng, g.hmax2) * (1.0f + OG_GM);
    if (lhs < rhs_min * (1.0f - OG_GM) && rmin2 > near2) {
        if (rmin2 > c.rcut2 * (1.0f + OG_GM)) return CL_DROP;
        return CL_ACCEPT;
    }
    return CL_GENERIC;
}

// Exact per-lane decision for one node from its full record (AABB cull, opening test with fp64 band):
// 0 = culled, 1 = open, 2 = accept.  Out of line: taken only when an fp32 test is within its band.
template <bool GEOM>
__device__ __noinline__ int slow_decide(const WalkArgs &a, uint32_t node, const Target &t, unsigned long long *cnt)
{
    const NodeRec m = load_node(a, node);
    if (og_cull(m, t, a.c)) return 0;
    float dx, dy, dz, r2;
    return og_open<GEOM>(m, t, a.c, dx, dy, dz, r2, cnt) ? 1 : 2;
}

// Group-level treatment of one particle by the lane that loaded it: 0 = no target within r_cut
// (dropped), 1 = staged with one exact periodic shift for all targets, 2 = staged as is (per-lane wrap).
__device__ __forceinline__ int classify_particle(float4 &p, const GroupInfo &g, const WalkConst &c)
{
    const float kx = rintf((p.x - g.gcx) * c.invL), ky = rintf((p.y - g.gcy) * c.invL), kz = rintf((p.z - g.gcz) * c.invL);
    const float adx = fabsf(fmaf(-c.L, kx, p.x - g.gcx)), ady = fabsf(fmaf(-c.L, ky, p.y - g.gcy)),
                adz = fabsf(fmaf(-c.L, kz, p.z - g.gcz));
    const float nx = fmaxf(adx - g.ghx, 0.f), ny = fmaxf(ady - g.ghy, 0.f), nz = fmaxf(adz - g.ghz, 0.f);
    if (fmaf(nz, nz, fmaf(ny, ny, nx * nx)) > c.rcut2 * (1.0f + OG_GM)) return 0;
    const float halfL = 0.5f * c.L * (1.0f - OG_GM);
    const float hL = 0.5f * c.L;
    if (fmaxf(adx + g.ghx, fmaxf(ady + g.ghy, adz + g.ghz)) < halfL && (kx == 0.0f || (kx == 1.0f && p.x >= hL)) &&
        (ky == 0.0f || (ky == 1.0f && p.y >= hL)) && (kz == 0.0f || (kz == 1.0f && p.z >= hL))) {
        p.x = fmaf(-c.L, kx, p.x); p.y = fmaf(-c.L, ky, p.y); p.z = fmaf(-c.L, kz, p.z);
        return 1;
    }
    return 2;
}

__device__ __forceinline__ float warp_min_pos(float v)   // v >= 0: integer order == float order
{
    return __uint_as_float(__reduce_min_sync(0xffffffffu, __float_as_uint(v)));
}
__device__ __forceinline__ float warp_max_pos(float v)
{
    return __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(v)));
}

// Per-lane interaction counters (OG_COUNT builds only).
struct LaneCount {
    uint32_t full, cull, ain, pin, psoft, pout;
};

// One source q = (x', y', z', G m) against the lane's target, exact in every respect: nearest-image wrap,
// cutoff decision with fp64 band, softened kernel.  Returns (dax, day, daz, dpot); kind = 0 outside r_cut,
// 1 inside with r >= h, 2 inside with r < h.  Out of line: the fast path below handles everything that is
// neither within OG_BAND of r_cut nor possibly softened.
template <bool POT>
__device__ __noinline__ float4 pair_exact(const float4 q, const float hj, const Target &t, const WalkConst &c,
                                          unsigned long long *cnt, int &kind)
{
    const float dx = og_wrap(q.x - t.x, c), dy = og_wrap(q.y - t.y, c), dz = og_wrap(q.z - t.z, c);
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    Accum d = {0.f, 0.f, 0.f, 0.f};
    kind = 0;
    if (og_inside_rcut(r2, q.x, q.y, q.z, t, c, cnt)) kind = og_pair_core<POT>(dx, dy, dz, r2, q.w, hj, t, c, d);
    return make_float4(d.ax, d.ay, d.az, d.pot);
}

// Position of a lane in the source ring: `nxt` = next segment (monotone counter) whose word the lane will
// take, `cur` = bits of segment nxt - 1 it has not evaluated yet, `base` = ring slot of that segment's
// first source, `nw` = the word of segment nxt, loaded ahead (valid while nxt < head).
struct LanePos {
    uint32_t nxt, cur, base, nw;
};

// Per-target accumulators of the group walk: two partial sums per component (the two source chains of the
// consume loop accumulate side by side in one register pair); pot holds +sum(G m E / r), negated at the end.
struct Accum2 {
    f32x2 ax, ay, az, pot;
};

__device__ __forceinline__ void acc2_add(f32x2 &v, float d)
{
    float a, b;
    upk2(v, a, b);
    v = pk2(a + d, b);
}

// Takes the next two sources of the lane's own list: moves on to the next produced segment if the current
// word is used up (its word was loaded ahead; the one after it is requested now), then extracts the lowest
// and the highest set bit of the word (two independent FLO; the order within a segment is free).  A lane
// without a (second) source gets the far-away dummy slot: beyond r_cut, nothing happens.
__device__ __forceinline__ void take_two(WarpSmem &w, LanePos &lp, const uint32_t head, const uint32_t lane,
                                         uint32_t &e0, uint32_t &e1)
{
    if (lp.cur == 0u && lp.nxt < head) {
        lp.cur = lp.nw;
        lp.base = (lp.nxt & (GW_NSEG - 1)) * 32u;
        ++lp.nxt;
        lp.nw = w.W[lp.nxt & (GW_NSEG - 1)][lane];   // (a stale word if nxt == head: reloaded at the next call)
    }
    const uint32_t cur = lp.cur;
    const uint32_t low = cur & (0u - cur);
    const uint32_t ilo = og_bfind(low), ihi = og_bfind(cur);     // 0xffffffff if there is none
    e0 = (cur != 0u) ? lp.base + ilo : GW_DUMMY;
    e1 = (ihi != ilo) ? lp.base + ihi : GW_DUMMY;
    lp.cur = (cur ^ low) & ~og_shl(1u, ihi);
}

// Two sources q0, q1 (ring slots e0, e1) against the lane's target, evaluated as ONE chain of packed fp32
// pairs (FFMA2 / FMUL2, walk_math.cuh).  Newtonian monopole x split factor (R21); a source that is within
// OG_BAND of r_cut or closer than the largest softening length of the whole particle set goes to pair_exact.
template <bool POT, bool COUNT, bool WRAP, bool HLOOK>
__device__ __forceinline__ uint32_t eval_two_fast(WarpSmem &w, const float4 q0, const float4 q1, const uint32_t e0,
                                                  const uint32_t e1, const Target &t, const float hmax2g,
                                                  const WalkConst &c, Accum2 &acc)
{
    const bool v0 = e0 != GW_DUMMY, v1 = e1 != GW_DUMMY;
    float dx0 = q0.x - t.x, dy0 = q0.y - t.y, dz0 = q0.z - t.z;
    float dx1 = q1.x - t.x, dy1 = q1.y - t.y, dz1 = q1.z - t.z;
    if (WRAP) {
        dx0 = og_wrap(dx0, c); dy0 = og_wrap(dy0, c); dz0 = og_wrap(dz0, c);
        dx1 = og_wrap(dx1, c); dy1 = og_wrap(dy1, c); dz1 = og_wrap(dz1, c);
    }
    const f32x2 dx = pk2(dx0, dx1), dy = pk2(dy0, dy1), dz = pk2(dz0, dz1);
    const f32x2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
    float r20, r21;
    upk2(r2, r20, r21);
    if (HLOOK) {
        // The 8-targets-per-warp kernel (sparse active subsets; a multi-species zoom has h comparable to r_cut and
        // most of its pairs softened: config 4 has 578 of 860 pairs per target inside h): the source's own h is
        // looked up below the largest h of the particle set (nodes carry h = 0: R16 keeps accepted nodes outside
        // the target's own h), and the spline-softened kernel (C5) is evaluated HERE, both polynomial pieces as
        // packed pairs and selected by u = r / h; g and p are continuous at u = 1/2 and u = 1, so only the cutoff
        // band (and r = 0) needs the exact path.
        const bool near0 = r20 < hmax2g, near1 = r21 < hmax2g;
        float hj0 = 0.0f, hj1 = 0.0f;
        if ((!WRAP || v0) && near0) hj0 = w.ring_h[e0];
        if ((!WRAP || v1) && near1) hj1 = w.ring_h[e1];
        const float hh0 = fmaxf(t.h, hj0), hh1 = fmaxf(t.h, hj1);
        const bool fast0 = (!WRAP || v0) && r20 < c.rcut2_lo && r20 > 1.0e-30f;
        const bool fast1 = (!WRAP || v1) && r21 < c.rcut2_lo && r21 > 1.0e-30f;
        const bool soft0 = fast0 && near0 && r20 < hh0 * hh0, soft1 = fast1 && near1 && r21 < hh1 * hh1;
        const bool slow0 = (!WRAP || v0) && !fast0 && r20 < c.rcut2_hi;
        const bool slow1 = (!WRAP || v1) && !fast1 && r21 < c.rcut2_hi;
        const f32x2 ri = pk2(fast0 ? og_rsqrt(r20) : 0.0f, fast1 ? og_rsqrt(r21) : 0.0f);
        const f32x2 r = mul2(r2, ri);
        f32x2 T, E;
        og_split2(r, r2, c, T, E);
        const f32x2 gm = pk2(fast0 ? q0.w : 0.0f, fast1 ? q1.w : 0.0f);
        f32x2 gfac = mul2(mul2(ri, ri), ri), pfac = ri;          // Newtonian: 1 / r^3, 1 / r (pot holds +sum)
        if (__any_sync(0xffffffffu, soft0 || soft1)) {
            const f32x2 hh = pk2(hh0, hh1);
            const f32x2 hinv = pk2(soft0 ? __frcp_rn(hh0) : 0.0f, soft1 ? __frcp_rn(hh1) : 0.0f);
            const f32x2 u = mul2(r, hinv), u2 = mul2(u, u);
            const f32x2 ui = mul2(hh, ri), ui3 = mul2(mul2(ui, ui), ui);            // 1 / u, 1 / u^3
            // u < 1/2:  g h^3 = 32/3 + u^2 (32 u - 192/5),  p h = -14/5 + u^2 (16/3 + u^2 (32/5 u - 48/5))
            f32x2 gi = fma2(u, bc2(32.0f), bc2(-38.4f));
            gi = fma2(u2, gi, bc2(10.666666666666666f));
            f32x2 pi = fma2(u, bc2(6.4f), bc2(-9.6f));
            pi = fma2(u2, pi, bc2(5.333333333333333f));
            pi = fma2(u2, pi, bc2(-2.8f));
            // 1/2 <= u < 1:  g h^3 = 64/3 - 48 u + 192/5 u^2 - 32/3 u^3 - 1 / (15 u^3),
            //                p h = -16/5 + 1 / (15 u) + u^2 (32/3 + u (-16 + u (48/5 - 32/15 u)))
            f32x2 go = fma2(u, bc2(-10.666666666666666f), bc2(38.4f));
            go = fma2(u, go, bc2(-48.0f));
            go = fma2(u, go, bc2(21.333333333333332f));
            go = fma2(ui3, bc2(-0.06666666666666667f), go);
            f32x2 po = fma2(u, bc2(-2.1333333333333333f), bc2(9.6f));
            po = fma2(u, po, bc2(-16.0f));
            po = fma2(u, po, bc2(10.666666666666666f));
            po = fma2(u2, po, bc2(-3.2f));
            po = fma2(ui, bc2(0.06666666666666667f), po);
            float u0, u1, gi0, gi1, go0, go1, pi0, pi1, po0, po1;
            upk2(u, u0, u1); upk2(gi, gi0, gi1); upk2(go, go0, go1); upk2(pi, pi0, pi1); upk2(po, po0, po1);
            const f32x2 gsel = pk2(u0 < 0.5f ? gi0 : go0, u1 < 0.5f ? gi1 : go1);
            const f32x2 psel = pk2(u0 < 0.5f ? pi0 : po0, u1 < 0.5f ? pi1 : po1);
            const f32x2 gs = mul2(mul2(mul2(hinv, hinv), hinv), gsel);
            const f32x2 ps = mul2(mul2(hinv, bc2(-1.0f)), psel);                    // -p > 0
            float gn0, gn1, pn0, pn1, gs0, gs1, ps0, ps1;
            upk2(gfac, gn0, gn1); upk2(pfac, pn0, pn1); upk2(gs, gs0, gs1); upk2(ps, ps0, ps1);
            gfac = pk2(soft0 ? gs0 : gn0, soft1 ? gs1 : gn1);
            pfac = pk2(soft0 ? ps0 : pn0, soft1 ? ps1 : pn1);
        }
        const f32x2 f = mul2(mul2(gm, T), gfac);
        acc.ax = fma2(f, dx, acc.ax); acc.ay = fma2(f, dy, acc.ay); acc.az = fma2(f, dz, acc.az);
        if (POT) acc.pot = fma2(mul2(gm, E), pfac, acc.pot);
        return (slow0 ? 1u : 0u) | (slow1 ? 2u : 0u) |
               (COUNT ? ((fast0 ? 4u : 0u) | (fast1 ? 8u : 0u) | (soft0 ? 16u : 0u) | (soft1 ? 32u : 0u)) : 0u);
    }
    // G = 32: fast = strictly inside the cutoff band and not softened: anything closer than the largest h of the
    // whole particle set (h_max of the root) takes the exact path.
    // (the wrapped distance of the dummy slot is arbitrary: WRAP keeps the validity predicates)
    const bool fast0 = (!WRAP || v0) && r20 < c.rcut2_lo && r20 >= hmax2g;
    const bool fast1 = (!WRAP || v1) && r21 < c.rcut2_lo && r21 >= hmax2g;
    const bool slow0 = (!WRAP || v0) && !fast0 && r20 < c.rcut2_hi;
    const bool slow1 = (!WRAP || v1) && !fast1 && r21 < c.rcut2_hi;
    {
        // 1 / r is replaced by 0 for a source that is not "fast" (masked, beyond r_cut, softened or exact path):
        // then r = w = 0, T = E = exp(..) <= 1 and the force and potential terms vanish, all finite (ring slots
        // hold finite values only); fast sources have hmax2g <= r^2 < r_cut^2, inside the range of og_split2
        const f32x2 ri = pk2(fast0 ? og_rsqrt(r20) : 0.0f, fast1 ? og_rsqrt(r21) : 0.0f);
        float ri0, ri1;
        upk2(ri, ri0, ri1);
        f32x2 T, E;
        og_split2(mul2(r2, ri), r2, c, T, E);
        const f32x2 gr = pk2(q0.w * ri0, q1.w * ri1);
        const f32x2 f = mul2(mul2(gr, T), mul2(ri, ri));
        acc.ax = fma2(f, dx, acc.ax); acc.ay = fma2(f, dy, acc.ay); acc.az = fma2(f, dz, acc.az);
        if (POT) acc.pot = fma2(gr, E, acc.pot);
    }
    // bits 0, 1: the source needs the exact path; bits 2, 3: it was evaluated here, bits 4, 5: softened (counters)
    return (slow0 ? 1u : 0u) | (slow1 ? 2u : 0u) | (COUNT ? ((fast0 ? 4u : 0u) | (fast1 ? 8u : 0u)) : 0u);
}

// The exact path of the sources flagged by eval_two_fast, and the counters.
template <bool POT, bool COUNT>
__device__ __forceinline__ void eval_two_slow(WarpSmem &w, const uint32_t flags, const float4 q0, const float4 q1,
                                              const uint32_t e0, const uint32_t e1, const Target &t, const WalkConst &c,
                                              Accum2 &acc, unsigned long long *cnt, LaneCount &lc)
{
    int k0 = (flags & 4u) ? ((flags & 16u) ? 2 : 1) : 0, k1 = (flags & 8u) ? ((flags & 32u) ? 2 : 1) : 0;
    if (flags & 3u) {
        if (flags & 1u) {
            const float4 d = pair_exact<POT>(q0, w.ring_h[e0], t, c, cnt, k0);
            acc2_add(acc.ax, d.x); acc2_add(acc.ay, d.y); acc2_add(acc.az, d.z); acc2_add(acc.pot, -d.w);
        }
        if (flags & 2u) {
            const float4 d = pair_exact<POT>(q1, w.ring_h[e1], t, c, cnt, k1);
            acc2_add(acc.ax, d.x); acc2_add(acc.ay, d.y); acc2_add(acc.az, d.z); acc2_add(acc.pot, -d.w);
        }
    }
    if (COUNT) {
        const bool v0 = e0 != GW_DUMMY, v1 = e1 != GW_DUMMY;
        const bool part0 = (w.seg_flags[(e0 >> 5) & (GW_NSEG - 1)] & SEG_PART) != 0u;
        const bool part1 = (w.seg_flags[(e1 >> 5) & (GW_NSEG - 1)] & SEG_PART) != 0u;
        if (v0) { if (part0) { lc.pin += (k0 != 0); lc.psoft += (k0 == 2); lc.pout += (k0 == 0); } else lc.ain += (k0 != 0); }
        if (v1) { if (part1) { lc.pin += (k1 != 0); lc.psoft += (k1 == 2); lc.pout += (k1 == 0); } else lc.ain += (k1 != 0); }
    }
}

template <bool POT, bool COUNT, bool WRAP, bool HLOOK>
__device__ __forceinline__ void eval_two(WarpSmem &w, const float4 q0, const float4 q1, const uint32_t e0, const uint32_t e1,
                                         const Target &t, const float hmax2g, const WalkConst &c, Accum2 &acc,
                                         unsigned long long *cnt, LaneCount &lc)
{
    const uint32_t fl = eval_two_fast<POT, COUNT, WRAP, HLOOK>(w, q0, q1, e0, e1, t, hmax2g, c, acc);
    eval_two_slow<POT, COUNT>(w, fl, q0, q1, e0, e1, t, c, acc, cnt, lc);
}

// Evaluates ring sources until every lane has finished all segments < target (tail <= target <= head; head =
// segments produced so far, tail = segments every lane had finished before).  Every lane walks the set bits
// of its own words, two sources per step; lanes with shorter lists run ahead into the segments >= target.
// The number of steps is known in advance (a word of k bits takes max(1, ceil(k / 2)) steps), so the loop has
// no exit test, and the sources of the next step are taken and loaded while the current pair is evaluated
// (unrolled by two so that the two pairs alternate between two register sets).  Returns the number of
// segments all lanes have finished.
template <bool POT, bool COUNT, bool WRAP, bool HLOOK>
__device__ __forceinline__ uint32_t consume(WarpSmem &w, const uint32_t head, const uint32_t tail, const uint32_t target,
                                            LanePos &lp, const Target &t, const float hmax2g, const WalkConst &c,
                                            Accum2 &acc, const uint32_t lane, unsigned long long *cnt, LaneCount &lc)
{
    // the word in progress is segment nxt - 1: it counts only if the lane is not already past the target
    uint32_t need = (lp.nxt <= target) ? (uint32_t)(__popc(lp.cur) + 1) >> 1 : 0u;
    for (uint32_t sg = tail; sg < target; ++sg) {
        const uint32_t ww = w.W[sg & (GW_NSEG - 1)][lane];
        const uint32_t k = max((uint32_t)(__popc(ww) + 1) >> 1, 1u);
        if (sg >= lp.nxt) need += k;
    }
    const uint32_t steps = __reduce_max_sync(0xffffffffu, need);
    lp.nw = w.W[lp.nxt & (GW_NSEG - 1)][lane];
#if OG_CONSUME_FOUR
    // two takes per iteration: two independent packed chains for the scheduler to interleave
    for (uint32_t it = 0u; it < steps; it += 2u) {
        uint32_t e0, e1, f0, f1;
        take_two(w, lp, head, lane, e0, e1);
        take_two(w, lp, head, lane, f0, f1);
        const float4 q0 = w.ring_pos[e0], q1 = w.ring_pos[e1], p0 = w.ring_pos[f0], p1 = w.ring_pos[f1];
        const uint32_t fa = eval_two_fast<POT, COUNT, WRAP, HLOOK>(w, q0, q1, e0, e1, t, hmax2g, c, acc);
        const uint32_t fb = eval_two_fast<POT, COUNT, WRAP, HLOOK>(w, p0, p1, f0, f1, t, hmax2g, c, acc);
        if (COUNT || ((fa | fb) & 3u)) {
            eval_two_slow<POT, COUNT>(w, fa, q0, q1, e0, e1, t, c, acc, cnt, lc);
            eval_two_slow<POT, COUNT>(w, fb, p0, p1, f0, f1, t, c, acc, cnt, lc);
        }
    }
#else
    for (uint32_t it = 0u; it < steps; ++it) {
        uint32_t e0, e1;
        take_two(w, lp, head, lane, e0, e1);
        const float4 q0 = w.ring_pos[e0], q1 = w.ring_pos[e1];
        eval_two<POT, COUNT, WRAP, HLOOK>(w, q0, q1, e0, e1, t, hmax2g, c, acc, cnt, lc);
    }
#endif
    return __reduce_min_sync(0xffffffffu, (lp.cur == 0u) ? lp.nxt : lp.nxt - 1u);
}

// G = targets per warp (32, or 8 for sparse active subsets), K = 32 / G lanes per target: lane = s * G + t
// serves target t and the staged sources / undecided nodes whose slot index is = s (mod K); all lane masks
// (imask, children masks) are G-bit TARGET masks; the K partial sums of a target are added at the end.
template <bool GEOM, bool POT, bool COUNT, int G>
__global__ void __launch_bounds__(GW_THREADS, OG_GW_MINBLOCKS)
k_walk_group(const __grid_constant__ WalkArgs a)
{
    constexpr int K = 32 / G;
    constexpr uint32_t TMASK = (G == 32) ? 0xffffffffu : ((1u << (G & 31)) - 1u);           // the G targets
    constexpr uint32_t REP = (G == 32) ? 1u : (G == 16) ? 0x00010001u : (G == 8) ? 0x01010101u : 0x11111111u;       // replicate a target mask to all slices
    constexpr uint32_t SLICE0 = (G == 32) ? 0xffffffffu : (G == 16) ? 0x55555555u : (G == 8) ? 0x11111111u : 0x01010101u;  // slots = 0 (mod K)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    WarpSmem *wsm = reinterpret_cast<WarpSmem *>(smem_raw);
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    WarpSmem &w = wsm[wid];
    const uint32_t lt = lanemask_lt();
    const uint32_t tl = lane & (G - 1), sl = lane / G;        // target and slice of this lane
    const uint32_t mybit = 1u << tl;                          // in target masks
    const uint32_t myslots = SLICE0 << sl;                    // the slots this lane evaluates
    const WalkConst &c = a.c;
    if (a.sel_flag != nullptr && __ldg(a.sel_flag) != a.sel) return;   // the other instantiation was chosen
    unsigned long long *cnt = COUNT ? a.counters : nullptr;
    uint32_t *sp_start = a.spill + (size_t)(blockIdx.x * GW_WARPS + wid) * 3 * a.spill_cap;
    uint32_t *sp_cnt = sp_start + a.spill_cap, *sp_mask = sp_cnt + a.spill_cap;
    const uint32_t half = a.stack_cap >> 1;   // ranges moved to / from the global slab at a time
    // largest softening length of the whole particle set = h_max of the root (R16 / R19 can only matter below it)
    const float hroot = __ldg(a.lo).w;
    // (> 0 even if no particle is softened: a coincident source, r = 0, must take the exact path)
    const float hmax2g = fmaxf(hroot * hroot * (1.0f + OG_BAND), 1.0e-30f);
    // stale ring slots are read (and masked out) by lanes that have nothing to do: keep them finite
    for (int i = lane; i < GW_NSEG * 32; i += 32) { w.ring_pos[i] = make_float4(0.f, 0.f, 0.f, 0.f); w.ring_h[i] = 0.f; }
    if (lane == 0) { w.ring_pos[GW_DUMMY] = make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f); w.ring_h[GW_DUMMY] = 0.f; }
    __syncwarp();

    for (;;) {
        uint32_t gi = 0;
        if (lane == 0) gi = atomicAdd(a.work, 1u);
        gi = __shfl_sync(0xffffffffu, gi, 0);
        if (gi >= a.n_groups) break;
        const uint32_t k = gi * (uint32_t)G + tl;
        const bool valid = k < a.n_active;
        const uint32_t klast = min(gi * (uint32_t)G + (uint32_t)(G - 1), a.n_active - 1u);
        uint32_t out = 0;
        // lanes past the end mirror the last target (keeps the group's bounds tight); they never
        // appear in a mask and write nothing
        Target t = load_target(a, valid ? k : klast, out, GEOM);
        t.x = fabsf(t.x); t.y = fabsf(t.y); t.z = fabsf(t.z);   // -0.0 -> +0.0 (integer-ordered reductions below)
        GroupInfo g;
        {
            // positions are >= 0 (0 <= x < L), a_old >= 0, h >= 0
            const float lox = warp_min_pos(t.x), loy = warp_min_pos(t.y), loz = warp_min_pos(t.z);
            const float hix = warp_max_pos(t.x), hiy = warp_max_pos(t.y), hiz = warp_max_pos(t.z);
            g.gcx = 0.5f * (lox + hix); g.gcy = 0.5f * (loy + hiy); g.gcz = 0.5f * (loz + hiz);
            // half sizes padded by 2 ulp(L) for the rounding of the centre
            const float pad = 2.4e-7f * c.L;
            g.ghx = 0.5f * (hix - lox) + pad; g.ghy = 0.5f * (hiy - loy) + pad; g.ghz = 0.5f * (hiz - loz) + pad;
            g.amin = warp_min_pos(fabsf(t.aold)); g.amax = warp_max_pos(fabsf(t.aold));
            const float hm = warp_max_pos(t.h);
            g.hmax2 = hm * hm;
            // A group that lies entirely in the upper quarter of the box along an axis is moved to the image
            // x - L (exact: L/2 <= x < L): its sources across the upper face then need no shift and the
            // others a shift by -L, which is exact for a source in the upper half (classify_node), so groups
            // next to the upper faces pre-shift their sources like all others.
            const float halfL = 0.75f * c.L;
            if (lox >= halfL) { t.x -= c.L; g.gcx = 0.5f * ((lox - c.L) + (hix - c.L)); }
            if (loy >= halfL) { t.y -= c.L; g.gcy = 0.5f * ((loy - c.L) + (hiy - c.L)); }
            if (loz >= halfL) { t.z -= c.L; g.gcz = 0.5f * ((loz - c.L) + (hiz - c.L)); }
        }
        // lanes whose target is the same sorted slot (duplicates in active_idx; the mirrored tail lanes)
        // (as a target mask; with the identity list every valid lane has its own slot, and the mirrored tail lanes
        // never appear in a mask)
        const uint32_t peers = a.tgt_slot ? (__match_any_sync(0xffffffffu, t.slot) & TMASK) : mybit;
        const float hi2 = t.h * t.h;
        Accum2 acc2 = {0ull, 0ull, 0ull, 0ull};
        LaneCount lc = {0, 0, 0, 0, 0, 0};
        int top = 0, pl_top = 0;
        uint32_t pl_items = 0, spill_n = 0;
        uint32_t head = 0, tail = 0;          // ring: segments produced / finished by all lanes
        bool anywrap = false;                 // some staged source of this group is not pre-shifted
        LanePos lp = {0u, 0u, 0u, 0u};
        {
            const uint32_t vm = __ballot_sync(0xffffffffu, valid) & TMASK;
            if (lane == 0) { w.st_start[0] = 0; w.st_cnt[0] = 1; w.st_mask[0] = vm; }
            top = 1;
            __syncwarp();
        }
        for (;;) {
            if (top == 0 && spill_n > 0) {  // reload spilled entries
                const uint32_t m = min(spill_n, half);
                for (uint32_t i = lane; i < m; i += 32) {
                    w.st_start[i] = sp_start[spill_n - m + i];
                    w.st_cnt[i] = sp_cnt[spill_n - m + i];
                    w.st_mask[i] = sp_mask[spill_n - m + i];
                }
                spill_n -= m;
                top = (int)m;
                __syncwarp();
            }
            // next action: a segment of particles of opened leaves, else a batch of nodes, else finish
            const bool parts = pl_items >= 32u || (top == 0 && pl_items > 0u);
            const bool fin = top == 0 && pl_items == 0u;
            if (head - tail == (uint32_t)GW_NSEG || (fin && head != tail)) {
                // ring full: free at least half of it; finishing: drain it
                __syncwarp();
                const uint32_t target = fin ? head : tail + GW_NSEG / 2;
                tail = anywrap ? consume<POT, COUNT, true, (G < 32)>(w, head, tail, target, lp, t, hmax2g, c, acc2, lane, cnt, lc)
                               : consume<POT, COUNT, false, (G < 32)>(w, head, tail, target, lp, t, hmax2g, c, acc2, lane, cnt, lc);
                __syncwarp();
            }
            if (fin) break;
            if (!parts) {
                const uint32_t slot0 = (head & (GW_NSEG - 1)) * 32u;
                uint32_t item, imask;
                const uint32_t total = pop_items(w.st_start, w.st_cnt, w.st_mask, top, lane, item, imask);
                uint32_t first = 0, meta = 0;
                int cls = CL_DROP;
                bool shifted = true;
                float4 sc = make_float4(0.f, 0.f, 0.f, 0.f), cel = sc;
                float lhs = 0.f, near2 = 0.f, cull2 = 0.f, hm2 = 0.f;
                if (lane < total) {
                    const uint4 *rp = a.rec + 3 * (size_t)item;
                    const uint4 r0 = __ldg(rp), n1 = __ldg(rp + 1), r2 = __ldg(rp + 2);
                    const float4 n0 = make_float4(__uint_as_float(r0.x), __uint_as_float(r0.y), __uint_as_float(r0.z), __uint_as_float(r0.w));
                    const float4 n2 = make_float4(__uint_as_float(r2.x), __uint_as_float(r2.y), __uint_as_float(r2.z), __uint_as_float(r2.w));
                    first = n1.z; meta = n1.w;
                    const float l = c.L * __uint_as_float((127u - (meta >> 27)) << 23);   // L / 2^level, exact
                    float kx, ky, kz;
                    cls = classify_node<GEOM>(n0, __uint_as_float(n1.x), __uint_as_float(n1.y), l, g, c, sc, lhs, near2,
                                              cull2, shifted, kx, ky, kz);
                    if (cls == CL_GENERIC) {
                        // cell centre in the same periodic image as sc (exact for k in {0, 1}, see classify_node)
                        cel = shifted ? make_float4(fmaf(-c.L, kx, n2.x), fmaf(-c.L, ky, n2.y), fmaf(-c.L, kz, n2.z), l)
                                      : make_float4(n2.x, n2.y, n2.z, l);
                        hm2 = n2.w * n2.w;
                    }
                }
                const uint32_t bA = __ballot_sync(0xffffffffu, cls == CL_ACCEPT);
                const uint32_t bX = __ballot_sync(0xffffffffu, cls == CL_GENERIC);
                const uint32_t bW = __ballot_sync(0xffffffffu, cls >= CL_ACCEPT && !shifted);
                anywrap |= bW != 0u;
                // ring slots of the segment: the undecided nodes first (in lane order), then the nodes every
                // target accepts; rX also numbers the undecided nodes in the staging arrays
                const uint32_t nX = __popc(bX), nA = __popc(bA);
                const uint32_t rX = __popc(bX & lt), rA = nX + __popc(bA & lt);
                if (cls == CL_GENERIC) {
                    w.ring_pos[slot0 + rX] = sc;
                    w.ring_h[slot0 + rX] = 0.0f;
                    float *f = &w.xq[rX >> 1][0].x + (rX & 1u);
                    f[0] = sc.x; f[2] = sc.y; f[4] = sc.z; f[6] = cull2;
                    f[8] = lhs * (1.0f - OG_BAND); f[10] = lhs * (1.0f + OG_BAND);
                    f[12] = near2; f[14] = __uint_as_float(imask);
                    if ((rX & 1u) == 0u && rX + 1u == nX) {   // odd count: the other half of the last pair tests nothing
                        f[1] = 0.f; f[3] = 0.f; f[5] = 0.f; f[7] = -1.0f; f[9] = 0.f; f[11] = 0.f; f[13] = 0.f; f[15] = 0.f;
                    }
                    w.xn_cel[rX] = cel; w.xn_hm2[rX] = hm2; w.xn_u[rX] = item;
                }
                if (cls == CL_ACCEPT) {
                    w.ring_pos[slot0 + rA] = sc;
                    w.ring_h[slot0 + rA] = 0.0f;
                    w.xn_u[rA] = imask;
                }
                __syncwarp();
                // MtA: bit j = my target is in the mask of the all-accepted node in ring slot j
                uint32_t MtA = 0u;
                if (bA != 0u) MtA = transpose32((lane >= nX && lane < nX + nA) ? w.xn_u[lane] * REP : 0u, lane);
                if (COUNT) {   // group-level outcomes counted as the per-target visits they stand for
                    const uint32_t bO = __ballot_sync(0xffffffffu, cls == CL_OPEN);
                    if (lane == 0) {
                        atomicAdd(&a.counters[OGC_CL_OPEN], (unsigned long long)__popc(bO));
                        atomicAdd(&a.counters[OGC_CL_ACCEPT], (unsigned long long)__popc(bA));
                        atomicAdd(&a.counters[OGC_CL_GENERIC], (unsigned long long)__popc(bX));
                        atomicAdd(&a.counters[OGC_CL_DROP], (unsigned long long)(total - __popc(bA | bX | bO)));
                        atomicAdd(&a.counters[OGC_BATCHES], 1ull);
                    }
                    for (uint32_t j = 0; j < total; ++j) {
                        const uint32_t mj = __shfl_sync(0xffffffffu, imask, j);
                        const int cj = __shfl_sync(0xffffffffu, cls, j);
                        if (sl == 0u && (mj & mybit) && (cj == CL_OPEN || cj == CL_ACCEPT)) ++lc.full;
                        if (sl == 0u && (mj & mybit) && cj == CL_DROP) ++lc.cull;
                    }
                }
                // Undecided nodes: every lane (G = 32; for G < 32 slice s of a target takes the pairs = s mod K)
                // tests the staged nodes two at a time as packed fp32 pairs (broadcast LDS.128), branch-free:
                // not in the mask or beyond r_cut + R of the node / opens / accepts / needs the guards.  The few
                // lanes of the last kind then evaluate the guards R15 / R16 from the staged cell, and anything
                // within the band of a threshold takes the exact out-of-line decision.
                uint32_t accw = 0u, myopen = 0u;
                if (bX != 0u) {
                    const bool xwrap = (bX & bW) != 0u;
                    uint32_t openw = 0u, sloww = 0u;
                    const uint32_t np = (nX + 1u) >> 1;
                    const f32x2 tx2 = bc2(t.x), ty2 = bc2(t.y), tz2 = bc2(t.z), A2 = bc2(GEOM ? c.theta2 : t.A);
                    uint32_t bit0 = 1u << (2u * sl);   // bit of the pair's first node (the second one is the next bit)
#pragma unroll 2
                    for (uint32_t p = sl; p < np; p += (uint32_t)K, bit0 <<= 2 * K) {
                        const float4 a0 = w.xq[p][0], a1 = w.xq[p][1], a2 = w.xq[p][2], a3 = w.xq[p][3];
                        f32x2 dx = sub2(pk2(a0.x, a0.y), tx2), dy = sub2(pk2(a0.z, a0.w), ty2), dz = sub2(pk2(a1.x, a1.y), tz2);
                        if (xwrap) {
                            float u0, u1;
                            upk2(dx, u0, u1); dx = pk2(og_wrap(u0, c), og_wrap(u1, c));
                            upk2(dy, u0, u1); dy = pk2(og_wrap(u0, c), og_wrap(u1, c));
                            upk2(dz, u0, u1); dz = pk2(og_wrap(u0, c), og_wrap(u1, c));
                        }
                        const f32x2 r2 = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
                        const f32x2 rhs = GEOM ? mul2(r2, A2) : mul2(mul2(r2, A2), r2);   // theta^2 r^2 / (A r^2) r^2
                        float r20, r21, rh0, rh1;
                        upk2(r2, r20, r21);
                        upk2(rhs, rh0, rh1);
                        const uint32_t bit1 = bit0 + bit0;
                        const bool in0 = (__float_as_uint(a3.z) & mybit) != 0u, in1 = (__float_as_uint(a3.w) & mybit) != 0u;
                        const bool cand0 = in0 && !(r20 > a1.z), cand1 = in1 && !(r21 > a1.w);
                        const bool fopen0 = rh0 < a2.x, fopen1 = rh1 < a2.y;
                        const bool facc0 = rh0 > a2.z && r20 > a3.x, facc1 = rh1 > a2.w && r21 > a3.y;
                        or_if(openw, bit0, cand0 && fopen0);
                        or_if(openw, bit1, cand1 && fopen1);
                        or_if(accw, bit0, cand0 && !fopen0 && facc0 && r20 < c.rcut2_hi);
                        or_if(accw, bit1, cand1 && !fopen1 && facc1 && r21 < c.rcut2_hi);
                        or_if(sloww, bit0, cand0 && !fopen0 && !facc0);
                        or_if(sloww, bit1, cand1 && !fopen1 && !facc1);
                        if (COUNT) {
                            if (in0 && !cand0) ++lc.cull;
                            if (in1 && !cand1) ++lc.cull;
                            if (cand0 && (fopen0 || facc0)) ++lc.full;
                            if (cand1 && (fopen1 || facc1)) ++lc.full;
                        }
                    }
                    while (sloww) {   // per lane, rare
                        const int j = __ffs(sloww) - 1;
                        sloww &= sloww - 1u;
                        const float *f = &w.xq[j >> 1][0].x + (j & 1);
                        const float4 cc = w.xn_cel[j];
                        float dx = f[0] - t.x, dy = f[2] - t.y, dz = f[4] - t.z;
                        float ex = cc.x - t.x, ey = cc.y - t.y, ez = cc.z - t.z;
                        if (xwrap) {
                            dx = og_wrap(dx, c); dy = og_wrap(dy, c); dz = og_wrap(dz, c);
                            ex = og_wrap(ex, c); ey = og_wrap(ey, c); ez = og_wrap(ez, c);
                        }
                        const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                        const float rhs = GEOM ? c.theta2 * r2 : t.A * r2 * r2;
                        const bool crit_open = rhs < f[8];
                        const float cmax = fmaxf(fabsf(ex), fmaxf(fabsf(ey), fabsf(ez)));
                        const float lim = 0.6f * cc.w;
                        const float hh2 = fmaxf(hi2, w.xn_hm2[j]);
                        const bool amb = (!crit_open && !(rhs > f[10])) || fabsf(cmax - lim) <= OG_BAND * cc.w ||
                                         fabsf(r2 - hh2) <= OG_BAND * hh2;
                        bool open, accept;
                        if (amb) {
                            const int d = slow_decide<GEOM>(a, w.xn_u[j], t, cnt);
                            open = d == 1; accept = d == 2;
                            if (COUNT) { if (d == 0) ++lc.cull; else ++lc.full; }
                        } else {
                            open = crit_open || cmax < lim || r2 < hh2;
                            accept = !open;
                            if (COUNT) ++lc.full;
                        }
                        const uint32_t bit = 1u << j;
                        if (open) openw |= bit;
                        if (accept && r2 < c.rcut2_hi) accw |= bit;
                    }
                    __syncwarp();
                    uint32_t ot = transpose32(openw, lane);   // lane j: the lanes that open undecided node j
                    if (G == 16) ot = (ot | (ot >> 16)) & TMASK;            // -> target mask
                    if (G == 8) { ot |= ot >> 16; ot = (ot | (ot >> 8)) & TMASK; }
                    if (G == 4) { ot |= ot >> 16; ot |= ot >> 8; ot = (ot | (ot >> 4)) & TMASK; }
                    myopen = __shfl_sync(0xffffffffu, ot, rX);   // back to the lane that holds the node
                }
                if ((bA | bX) != 0u) {
                    w.W[head & (GW_NSEG - 1)][lane] = (MtA & myslots) | accw;
                    if (COUNT && lane == 0) w.seg_flags[head & (GW_NSEG - 1)] = 0u;
                    ++head;
                }
                __syncwarp();
                // push opened internal nodes (children ranges) and opened leaves (particle ranges)
                const uint32_t cmask = (cls == CL_OPEN) ? imask : ((cls == CL_GENERIC) ? myopen : 0u);
                const bool is_leaf = (meta >> 26) & 1u;
                const uint32_t ccount = meta & 0x03ffffffu;
                const bool push_n = cmask != 0 && !is_leaf;
                const bool push_p = cmask != 0 && is_leaf;
                const uint32_t bn = __ballot_sync(0xffffffffu, push_n);
                const uint32_t bp = __ballot_sync(0xffffffffu, push_p);
                const int nn = __popc(bn);
                if ((uint32_t)(top + nn) > a.stack_cap) {  // spill the older half of the stack to global memory
                    if (spill_n + half > a.spill_cap) {
                        if (lane == 0) atomicOr(a.status, OG_DEV_STACK_OVERFLOW);
                        top = 0;  // give up on this group (result invalid, status latched)
                    } else {
                        for (uint32_t i = lane; i < half; i += 32) {
                            sp_start[spill_n + i] = w.st_start[i];
                            sp_cnt[spill_n + i] = w.st_cnt[i];
                            sp_mask[spill_n + i] = w.st_mask[i];
                        }
                        __syncwarp();
                        const uint32_t rest = (uint32_t)top - half;
                        for (uint32_t i0 = 0; i0 < rest; i0 += 32) {
                            const uint32_t i = i0 + lane;
                            uint32_t s0 = 0, s1 = 0, s2 = 0;
                            if (i < rest) { s0 = w.st_start[i + half]; s1 = w.st_cnt[i + half]; s2 = w.st_mask[i + half]; }
                            __syncwarp();
                            if (i < rest) { w.st_start[i] = s0; w.st_cnt[i] = s1; w.st_mask[i] = s2; }
                        }
                        spill_n += half;
                        top -= (int)half;
                        if (COUNT && lane == 0) atomicAdd(&a.counters[OGC_SPILLS], 1ull);
                        __syncwarp();
                    }
                }
                if (push_n) {
                    const int p = top + __popc(bn & lt);
                    w.st_start[p] = first; w.st_cnt[p] = ccount; w.st_mask[p] = cmask;
                }
                top += nn;
                if (push_p) {
                    const int p = pl_top + __popc(bp & lt);
                    w.pl_start[p] = first; w.pl_cnt[p] = ccount; w.pl_mask[p] = cmask;
                }
                pl_top += __popc(bp);
                pl_items += __reduce_add_sync(0xffffffffu, push_p ? ccount : 0u);
                __syncwarp();
            } else {
                // move 32 particles of opened leaves into a segment
                const uint32_t slot0 = (head & (GW_NSEG - 1)) * 32u;
                uint32_t item, imask;
                const uint32_t total = pop_items(w.pl_start, w.pl_cnt, w.pl_mask, pl_top, lane, item, imask);
                pl_items -= total;
                int pc = 0;
                if (lane < total) {
                    float4 p = __ldg(a.spos + item);
                    const float ph = __ldg(a.sh + item);
                    pc = classify_particle(p, g, c);
                    if (pc != 0) {
                        p.w *= c.G;
                        w.ring_pos[slot0 + lane] = p;
                        w.ring_h[slot0 + lane] = ph;
                    }
                }
                // self exclusion: the lanes whose target IS this particle (target slots ascend with the lane)
                uint32_t selfm = 0u;
                {
                    int lo = 0;
#pragma unroll
                    for (int step = G / 2; step >= 1; step >>= 1) {   // lanes 0 .. G-1 hold the G targets
                        const uint32_t v = __shfl_sync(0xffffffffu, t.slot, lo + step - 1);
                        if (v < item) lo += step;
                    }
                    const uint32_t v = __shfl_sync(0xffffffffu, t.slot, lo);
                    const uint32_t pm = __shfl_sync(0xffffffffu, peers, lo);
                    if (v == item) selfm = pm;
                }
                const uint32_t b2 = __ballot_sync(0xffffffffu, pc == 2);
                anywrap |= b2 != 0u;
                const uint32_t Mt = transpose32((lane < total && pc != 0) ? (imask & ~selfm) * REP : 0u, lane);
                w.W[head & (GW_NSEG - 1)][lane] = Mt & myslots;
                if (COUNT && lane == 0) w.seg_flags[head & (GW_NSEG - 1)] = SEG_PART;
                ++head;
                if (COUNT) {
                    const uint32_t b1 = __ballot_sync(0xffffffffu, pc == 1);
                    if (lane == 0) {
                        atomicAdd(&a.counters[OGC_PT_SHIFT], (unsigned long long)__popc(b1));
                        atomicAdd(&a.counters[OGC_PT_WRAP], (unsigned long long)__popc(b2));
                        atomicAdd(&a.counters[OGC_PT_DROP], (unsigned long long)(total - __popc(b1 | b2)));
                    }
                    for (uint32_t j = 0; j < total; ++j) {
                        const uint32_t mj = __shfl_sync(0xffffffffu, imask & ~selfm, j);
                        const int cj = __shfl_sync(0xffffffffu, pc, j);
                        if (sl == 0u && (mj & mybit) && cj == 0) ++lc.pout;
                    }
                }
                __syncwarp();
            }
        }
        Accum acc;
        {
            float a, b;
            upk2(acc2.ax, a, b); acc.ax = a + b;
            upk2(acc2.ay, a, b); acc.ay = a + b;
            upk2(acc2.az, a, b); acc.az = a + b;
            upk2(acc2.pot, a, b); acc.pot = -(a + b);
        }
        if (G < 32) {   // add the K partial sums of every target
#pragma unroll
            for (int o = G; o < 32; o <<= 1) {
                acc.ax += __shfl_xor_sync(0xffffffffu, acc.ax, o); acc.ay += __shfl_xor_sync(0xffffffffu, acc.ay, o);
                acc.az += __shfl_xor_sync(0xffffffffu, acc.az, o); acc.pot += __shfl_xor_sync(0xffffffffu, acc.pot, o);
            }
        }
        if (valid && sl == 0u) {
            a.acc_out[3 * (size_t)out] = acc.ax;
            a.acc_out[3 * (size_t)out + 1] = acc.ay;
            a.acc_out[3 * (size_t)out + 2] = acc.az;
            if (POT) a.pot_out[out] = acc.pot;
        }
        if (COUNT && a.cost != nullptr) {   // per-target work figure (OG_F_WALK_COST): interactions evaluated
            uint32_t wk = lc.ain + lc.pin + lc.pout;
            if (G < 32) {
#pragma unroll
                for (int o = G; o < 32; o <<= 1) wk += __shfl_xor_sync(0xffffffffu, wk, o);
            }
            if (valid && sl == 0u) a.cost[out] = wk;
        }
        if (COUNT) {
            const uint32_t v[6] = {lc.full, lc.cull, lc.ain, lc.pin, lc.psoft, lc.pout};
            const int slot[6] = {OGC_V_FULL, OGC_V_CULL, OGC_A_IN, OGC_P_IN, OGC_P_SOFT, OGC_P_OUT};
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                const uint32_t s = __reduce_add_sync(0xffffffffu, valid ? v[q] : 0u);
                if (lane == 0) atomicAdd(&a.counters[slot[q]], (unsigned long long)s);
            }
        }
    }
}

template <bool GEOM, bool POT, bool COUNT, int G>
cudaError_t launch_g(const og_tree *t, WalkArgs a, cudaStream_t st)
{
    a.n_groups = (uint32_t)(((uint64_t)a.n_active + G - 1) / G);
    const size_t smem = GW_WARPS * sizeof(WarpSmem);
    auto kern = k_walk_group<GEOM, POT, COUNT, G>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, GW_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    if (per_sm > OG_GW_MINBLOCKS) per_sm = OG_GW_MINBLOCKS;   // the spill slabs are sized for this many blocks per SM
    const unsigned grid = (unsigned)(per_sm * t->sm_count);
    kern<<<grid, GW_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

// Targets per warp: 32 when the active targets are dense in Morton order; 8 (4 lanes per target) for a sparse active
// list, whose 32 consecutive targets would span many cells (zoom: 52 -> 21 ms).  For the spread-out groups of a DENSE
// target set (uniform background of nfw256) 8 per warp is slower (measured).  With an explicit active list the choice
// is made on the device from the density of the list in the Morton range it covers (k_unpack_slots): both
// instantiations are launched and the one that was not chosen returns at once (no host round trip).
template <bool GEOM, bool POT, bool COUNT>
cudaError_t launch(const og_tree *t, WalkArgs &a, cudaStream_t st)
{
    if (a.sel_flag == nullptr) {       // identity list: always dense
        a.sel = 0u;
        return launch_g<GEOM, POT, COUNT, 32>(t, a, st);
    }
    a.sel = 0u;
    cudaError_t e = launch_g<GEOM, POT, COUNT, 32>(t, a, st);
    if (e != cudaSuccess) return e;
    a.sel = 1u;
    return launch_g<GEOM, POT, COUNT, OG_GW_SPARSE_G>(t, a, st);
}

}  // namespace

uint32_t ogk_walk_spill_entries(const og_params *p)
{
    return p->walk_spill_entries ? p->walk_spill_entries : 3072u;   // ranges per warp (x 12 B)
}

size_t ogk_walk_spill_bytes(int sm_count, uint32_t spill_entries)
{
    return (size_t)sm_count * OG_GW_MINBLOCKS * GW_WARPS * 3 * spill_entries * sizeof(uint32_t);
}

cudaError_t ogk_walk(const og_tree *t, const uint32_t *tgt_slot, const uint32_t *tgt_out, uint64_t n_active,
                     const float *a_old, float *acc_out, float *pot_out, cudaStream_t st, const float4 *ext,
                     const uint32_t *ext_sparse)
{
    WalkArgs a;
    a.ext = ext;
    // the device flag that picks 32 or 8 targets per warp: written by k_unpack_slots for an explicit active list, by
    // k_ext_sparse for external targets (the caller passes where); none for the identity list
    a.sel_flag = tgt_slot ? t->d_status + 2 : ext_sparse;
    a.com = t->node_com; a.cell = t->node_cell; a.lo = t->node_lo; a.hi = t->node_hi;
    a.info = t->node_info; a.rec = t->node_rec; a.spos = t->spos; a.sh = t->sh;
    a.tgt_slot = tgt_slot; a.tgt_out = tgt_out; a.a_old = a_old; a.acc_out = acc_out; a.pot_out = pot_out;
    a.n_active = (uint32_t)n_active;
    a.n_groups = (uint32_t)((n_active + 31) / 32);
    a.work = t->d_status + 1;
    a.status = t->d_status;
    a.counters = t->d_counters;
    a.spill = reinterpret_cast<uint32_t *>(t->walk_spill);
    // the per-target work array has one entry per particle of the tree: not written for external targets, nor for a
    // list longer than that (duplicates)
    a.cost = (ext == nullptr && n_active <= t->n) ? t->walk_cost : nullptr;
    a.spill_cap = t->walk_spill_cap;
    a.stack_cap = t->prm.walk_stack_entries ? min(t->prm.walk_stack_entries, (uint32_t)GW_STACK) : (uint32_t)GW_STACK;
    const og_params &p = t->prm;
    WalkConst &c = a.c;
    c.dL = (double)t->box;
    c.drcut = (double)p.rcut_over_rs * (double)p.r_s;
    c.dG = (double)p.G; c.dalpha = (double)p.alpha; c.dtheta2 = (double)p.theta * (double)p.theta;
    c.L = t->box; c.invL = 1.0f / t->box;
    c.rcut = (float)c.drcut; c.rcut2 = (float)(c.drcut * c.drcut);
    c.rcut2_lo = c.rcut2 * (1.0f - OG_BAND); c.rcut2_hi = c.rcut2 * (1.0f + OG_BAND);
    c.cull_r = (float)(c.drcut * (1.0 + 1e-5) + 1e-6 * c.dL);
    c.G = p.G; c.alpha = p.alpha; c.theta2 = (float)c.dtheta2;
    c.k_w = (float)(0.5 / (double)p.r_s);
    c.k_e = (float)(-1.4426950408889634 / (4.0 * (double)p.r_s * (double)p.r_s));
    c.hmax2g = 0.0f;   // read from the root record by the kernels
    cudaError_t e = cudaMemsetAsync(t->d_status + 1, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    const bool count = (p.flags & OG_COUNT) != 0;
    if (count) {
        e = cudaMemsetAsync(t->d_counters, 0, OGC_N * sizeof(unsigned long long), st);
        if (e != cudaSuccess) return e;
    }
    const bool geom = (a_old == nullptr), pot = (pot_out != nullptr);
#define OG_DISPATCH(G_, P_, C_) if (geom == G_ && pot == P_ && count == C_) return launch<G_, P_, C_>(t, a, st);
    OG_DISPATCH(false, false, false) OG_DISPATCH(false, false, true)
    OG_DISPATCH(false, true, false)  OG_DISPATCH(false, true, true)
    OG_DISPATCH(true, false, false)  OG_DISPATCH(true, false, true)
    OG_DISPATCH(true, true, false)   OG_DISPATCH(true, true, true)
#undef OG_DISPATCH
    return cudaErrorUnknown;
}
