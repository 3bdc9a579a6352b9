// walk.cu -- rows a6 (short-range tree walk) and a7 (scatter to the caller's order) of
// SURVEY.md Sec. 8(a).  PAPER.md:59 (a tree walk per active particle), :74 (per-node
// interaction and opening criterion).
//
// k_walk_group (the product path): one warp walks the tree for a group of 32 targets that are
// consecutive in Morton order.  The warp traverses the UNION of its lanes' walks, but every
// lane accepts / opens exactly the nodes its own serial walk would (C6): each pending entry
// carries a 32-bit lane mask = the lanes that opened the parent.  Per iteration the warp pops
// up to 32 child nodes from a shared-memory stack of (first, count, mask) ranges, lane k
// loads node k (4 x LDG.128, children are contiguous), the records are staged in shared
// memory, every lane scans the staged batch (broadcast LDS.128) doing cull / opening test /
// monopole for the entries whose mask holds its bit, and a ballot per entry yields the mask
// of the children.  Opened leaves go to a second range list whose particles are staged and
// evaluated the same way in batches of 32.  The split table (T, dT, E, dE) lives in shared
// memory.  Results are written straight to the caller's order (a7 fused).
//
// k_walk_simple: one thread per target with a private stack; debugging / comparison only.
#include "walk_math.cuh"

namespace {

struct WalkArgs {
    const float4 *com, *cell, *lo, *hi;
    const uint2 *info;
    const float4 *spos;
    const float *sh;
    const float4 *tab;
    const uint32_t *tgt_slot;  // NULL -> identity
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
    const uint32_t slot = a.tgt_slot ? __ldg(a.tgt_slot + k) : k;
    out = __ldg(a.tgt_out + k);
    const float4 p = __ldg(a.spos + slot);
    t.x = p.x; t.y = p.y; t.z = p.z;
    t.h = __ldg(a.sh + slot);
    t.slot = slot;
    t.aold = geom ? 0.0f : __ldg(a.a_old + out);
    t.A = a.c.alpha * t.aold;
    return t;
}

__device__ __forceinline__ void copy_table(float4 *s_tab, const float4 *g_tab)
{
    for (int i = threadIdx.x; i < OG_NTAB; i += blockDim.x) s_tab[i] = g_tab[i];
}

// -------------------------------------------------------------------------------------------
template <bool GEOM, bool POT, bool COUNT>
__global__ void __launch_bounds__(128)
k_walk_simple(WalkArgs a)
{
    __shared__ float4 s_tab[OG_NTAB];
    copy_table(s_tab, a.tab);
    __syncthreads();
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.n_active) return;
    uint32_t out;
    const Target t = load_target(a, k, out, GEOM);
    unsigned long long *cnt = COUNT ? a.counters : nullptr;
    unsigned long long c_full = 0, c_cull = 0, c_ain = 0, c_pin = 0, c_psoft = 0, c_pout = 0;
    Accum acc = {0.f, 0.f, 0.f, 0.f};
    uint32_t stack[176];
    int sp = 0;
    stack[sp++] = 0;
    while (sp) {
        const uint32_t j = stack[--sp];
        const NodeRec n = load_node(a, j);
        if (og_cull(n, t, a.c)) { ++c_cull; continue; }
        ++c_full;
        float dx, dy, dz, r2;
        if (!og_open<GEOM>(n, t, a.c, dx, dy, dz, r2, cnt)) {
            c_ain += og_monopole<POT>(n, t, a.c, s_tab, dx, dy, dz, r2, acc, cnt);
            continue;
        }
        const uint2 info = __ldg(a.info + j);
        if (info.y & OG_LEAF_BIT) {
            const uint32_t f = info.x, c = info.y & ~OG_LEAF_BIT;
            for (uint32_t s = f; s < f + c; ++s) {
                if (s == t.slot) continue;
                const int kind = og_pair<POT>(__ldg(a.spos + s), __ldg(a.sh + s), t, a.c, s_tab, acc, cnt);
                if (kind == 0) ++c_pout; else { ++c_pin; if (kind == 2) ++c_psoft; }
            }
        } else {
            for (uint32_t ch = 0; ch < info.y; ++ch) {
                if (sp >= 176) { atomicOr(a.status, OG_DEV_STACK_OVERFLOW); break; }
                stack[sp++] = info.x + info.y - 1 - ch;
            }
        }
    }
    a.acc_out[3 * (size_t)out] = acc.ax;
    a.acc_out[3 * (size_t)out + 1] = acc.ay;
    a.acc_out[3 * (size_t)out + 2] = acc.az;
    if (POT) a.pot_out[out] = acc.pot;
    if (COUNT) {
        atomicAdd(&a.counters[OGC_V_FULL], c_full);
        atomicAdd(&a.counters[OGC_V_CULL], c_cull);
        atomicAdd(&a.counters[OGC_A_IN], c_ain);
        atomicAdd(&a.counters[OGC_P_IN], c_pin);
        atomicAdd(&a.counters[OGC_P_SOFT], c_psoft);
        atomicAdd(&a.counters[OGC_P_OUT], c_pout);
    }
}

// -------------------------------------------------------------------------------------------
constexpr int GW_WARPS = 8;           // warps per block
constexpr int GW_THREADS = GW_WARPS * 32;
constexpr int GW_STACK = 384;         // node-range stack entries per warp in shared memory
constexpr int GW_SPILL = 192;         // entries moved to / from global memory at a time
constexpr int GW_PLIST = 64;          // particle-range list entries per warp

struct __align__(16) WarpSmem {
    float4 nd_com[32], nd_cell[32], nd_lo[32], nd_hi[32];
    float4 pt_pos[32];
    float pt_h[32];
    uint32_t pt_slot[32];
    uint32_t bt_mask[32];             // masks of the staged batch (nodes or particles)
    uint32_t st_start[GW_STACK], st_cnt[GW_STACK], st_mask[GW_STACK];
    uint32_t pl_start[GW_PLIST], pl_cnt[GW_PLIST], pl_mask[GW_PLIST];
};

__device__ __forceinline__ uint32_t lanemask_lt()
{
    uint32_t m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
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

template <bool GEOM, bool POT, bool COUNT>
__global__ void __launch_bounds__(GW_THREADS, 2)
k_walk_group(WalkArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *s_tab = reinterpret_cast<float4 *>(smem_raw);
    WarpSmem *wsm = reinterpret_cast<WarpSmem *>(smem_raw + OG_NTAB * sizeof(float4));
    copy_table(s_tab, a.tab);
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
    WarpSmem &w = wsm[wid];
    const uint32_t lt = lanemask_lt();
    const uint32_t mybit = 1u << lane;
    unsigned long long *cnt = COUNT ? a.counters : nullptr;
    uint32_t *sp_start = a.spill + (size_t)(blockIdx.x * GW_WARPS + wid) * 3 * a.spill_cap;
    uint32_t *sp_cnt = sp_start + a.spill_cap, *sp_mask = sp_cnt + a.spill_cap;

    for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(a.work, 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g >= a.n_groups) break;
        const uint32_t k = g * 32u + lane;
        const bool valid = k < a.n_active;
        uint32_t out = 0;
        Target t = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0xffffffffu};
        if (valid) t = load_target(a, k, out, GEOM);
        Accum acc = {0.f, 0.f, 0.f, 0.f};
        uint32_t c_full = 0, c_cull = 0, c_ain = 0, c_pin = 0, c_psoft = 0, c_pout = 0;
        int top = 0, pl_top = 0;
        uint32_t pl_items = 0, spill_n = 0;
        {
            const uint32_t vm = __ballot_sync(0xffffffffu, valid);
            if (lane == 0) { w.st_start[0] = 0; w.st_cnt[0] = 1; w.st_mask[0] = vm; }
            top = 1;
            __syncwarp();
        }
        for (;;) {
            if (top == 0 && spill_n > 0) {  // reload spilled entries
                const uint32_t m = min(spill_n, (uint32_t)GW_SPILL);
                for (uint32_t i = lane; i < m; i += 32) {
                    w.st_start[i] = sp_start[spill_n - m + i];
                    w.st_cnt[i] = sp_cnt[spill_n - m + i];
                    w.st_mask[i] = sp_mask[spill_n - m + i];
                }
                spill_n -= m;
                top = (int)m;
                __syncwarp();
            }
            if (top > 0) {
                uint32_t item, imask;
                const uint32_t total = pop_items(w.st_start, w.st_cnt, w.st_mask, top, lane, item, imask);
                uint2 info = make_uint2(0u, 0u);
                if (lane < total) {
                    const NodeRec n = load_node(a, item);
                    info = __ldg(a.info + item);
                    w.nd_com[lane] = n.com; w.nd_cell[lane] = n.cell;
                    w.nd_lo[lane] = n.lo; w.nd_hi[lane] = n.hi;
                    w.bt_mask[lane] = imask;
                }
                __syncwarp();
                uint32_t myopen = 0;
                for (uint32_t j = 0; j < total; ++j) {
                    bool open = false;
                    if (w.bt_mask[j] & mybit) {
                        NodeRec n;
                        n.com = w.nd_com[j]; n.cell = w.nd_cell[j]; n.lo = w.nd_lo[j]; n.hi = w.nd_hi[j];
                        if (og_cull(n, t, a.c)) {
                            if (COUNT) ++c_cull;
                        } else {
                            if (COUNT) ++c_full;
                            float dx, dy, dz, r2;
                            open = og_open<GEOM>(n, t, a.c, dx, dy, dz, r2, cnt);
                            if (!open) {
                                const int in = og_monopole<POT>(n, t, a.c, s_tab, dx, dy, dz, r2, acc, cnt);
                                if (COUNT) c_ain += in;
                            }
                        }
                    }
                    const uint32_t b = __ballot_sync(0xffffffffu, open);
                    if (lane == j) myopen = b;
                }
                __syncwarp();
                // push opened internal nodes (children ranges) and opened leaves (particle ranges)
                const bool is_leaf = (info.y & OG_LEAF_BIT) != 0;
                const bool push_n = myopen != 0 && !is_leaf;
                const bool push_p = myopen != 0 && is_leaf;
                const uint32_t bn = __ballot_sync(0xffffffffu, push_n);
                const uint32_t bp = __ballot_sync(0xffffffffu, push_p);
                const int nn = __popc(bn);
                if (top + nn > GW_STACK) {  // spill the bottom of the stack to global memory
                    if (spill_n + GW_SPILL > a.spill_cap) {
                        if (lane == 0) atomicOr(a.status, OG_DEV_STACK_OVERFLOW);
                        top = 0;  // give up on this group (result invalid, status latched)
                    } else {
                        for (uint32_t i = lane; i < (uint32_t)GW_SPILL; i += 32) {
                            sp_start[spill_n + i] = w.st_start[i];
                            sp_cnt[spill_n + i] = w.st_cnt[i];
                            sp_mask[spill_n + i] = w.st_mask[i];
                        }
                        __syncwarp();
                        const uint32_t rest = (uint32_t)top - GW_SPILL;
                        for (uint32_t i0 = 0; i0 < rest; i0 += 32) {
                            const uint32_t i = i0 + lane;
                            uint32_t s0 = 0, s1 = 0, s2 = 0;
                            if (i < rest) { s0 = w.st_start[i + GW_SPILL]; s1 = w.st_cnt[i + GW_SPILL]; s2 = w.st_mask[i + GW_SPILL]; }
                            __syncwarp();
                            if (i < rest) { w.st_start[i] = s0; w.st_cnt[i] = s1; w.st_mask[i] = s2; }
                        }
                        spill_n += GW_SPILL;
                        top -= GW_SPILL;
                        __syncwarp();
                    }
                }
                if (push_n) {
                    const int p = top + __popc(bn & lt);
                    w.st_start[p] = info.x; w.st_cnt[p] = info.y; w.st_mask[p] = myopen;
                }
                top += nn;
                if (push_p) {
                    const int p = pl_top + __popc(bp & lt);
                    w.pl_start[p] = info.x; w.pl_cnt[p] = info.y & ~OG_LEAF_BIT; w.pl_mask[p] = myopen;
                }
                pl_top += __popc(bp);
                pl_items += __reduce_add_sync(0xffffffffu, push_p ? (info.y & ~OG_LEAF_BIT) : 0u);
                __syncwarp();
            }
            // drain the particle list in batches of 32
            while (pl_items >= 32u || (top == 0 && spill_n == 0 && pl_items > 0u)) {
                uint32_t item, imask;
                const uint32_t total = pop_items(w.pl_start, w.pl_cnt, w.pl_mask, pl_top, lane, item, imask);
                pl_items -= total;
                if (lane < total) {
                    w.pt_pos[lane] = __ldg(a.spos + item);
                    w.pt_h[lane] = __ldg(a.sh + item);
                    w.pt_slot[lane] = item;
                    w.bt_mask[lane] = imask;
                }
                __syncwarp();
                for (uint32_t j = 0; j < total; ++j) {
                    if ((w.bt_mask[j] & mybit) && w.pt_slot[j] != t.slot) {
                        const int kind = og_pair<POT>(w.pt_pos[j], w.pt_h[j], t, a.c, s_tab, acc, cnt);
                        if (COUNT) { if (kind == 0) ++c_pout; else { ++c_pin; if (kind == 2) ++c_psoft; } }
                    }
                }
                __syncwarp();
            }
            if (top == 0 && spill_n == 0 && pl_items == 0u) break;
        }
        if (valid) {
            a.acc_out[3 * (size_t)out] = acc.ax;
            a.acc_out[3 * (size_t)out + 1] = acc.ay;
            a.acc_out[3 * (size_t)out + 2] = acc.az;
            if (POT) a.pot_out[out] = acc.pot;
        }
        if (COUNT) {
            const uint32_t v[6] = {c_full, c_cull, c_ain, c_pin, c_psoft, c_pout};
            const int slot[6] = {OGC_V_FULL, OGC_V_CULL, OGC_A_IN, OGC_P_IN, OGC_P_SOFT, OGC_P_OUT};
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                const uint32_t s = __reduce_add_sync(0xffffffffu, v[q]);
                if (lane == 0) atomicAdd(&a.counters[slot[q]], (unsigned long long)s);
            }
        }
    }
}

// split table rows (T, dT, E, dE) in fp64, stored fp32 (R18)
__global__ void k_split_table(float4 *tab, double rcut, double r_s)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= OG_NTAB) return;
    const double two_over_sqrt_pi = 1.1283791670955125738961589031215;
    const double w0 = (double)i * rcut / OG_NTAB / (2.0 * r_s);
    const double w1 = (double)(i + 1) * rcut / OG_NTAB / (2.0 * r_s);
    const double T0 = erfc(w0) + two_over_sqrt_pi * w0 * exp(-w0 * w0);
    const double T1 = erfc(w1) + two_over_sqrt_pi * w1 * exp(-w1 * w1);
    const double E0 = erfc(w0), E1 = erfc(w1);
    tab[i] = make_float4((float)T0, (float)(T1 - T0), (float)E0, (float)(E1 - E0));
}

template <bool GEOM, bool POT, bool COUNT>
cudaError_t launch(const og_tree *t, WalkArgs &a, cudaStream_t st)
{
    if (t->prm.walk_variant == OG_WALK_SIMPLE) {
        const unsigned grid = (a.n_active + 127) / 128;
        k_walk_simple<GEOM, POT, COUNT><<<grid, 128, 0, st>>>(a);
        return cudaGetLastError();
    }
    const size_t smem = OG_NTAB * sizeof(float4) + GW_WARPS * sizeof(WarpSmem);
    auto kern = k_walk_group<GEOM, POT, COUNT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, GW_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;   // spill slabs are sized for <= 4 blocks per SM
    const unsigned grid = (unsigned)(per_sm * t->sm_count);
    kern<<<grid, GW_THREADS, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace

static constexpr uint32_t SPILL_CAP = 3072;  // entries per warp (x 12 B)

size_t ogk_walk_spill_bytes(int sm_count)
{
    return (size_t)sm_count * 4 * GW_WARPS * 3 * SPILL_CAP * sizeof(uint32_t);
}

cudaError_t ogk_split_table(float4 *tab, double rcut, double r_s, cudaStream_t st)
{
    k_split_table<<<(OG_NTAB + 255) / 256, 256, 0, st>>>(tab, rcut, r_s);
    return cudaGetLastError();
}

cudaError_t ogk_walk(const og_tree *t, const uint32_t *tgt_slot, const uint32_t *tgt_out, uint64_t n_active,
                     const float *a_old, float *acc_out, float *pot_out, cudaStream_t st)
{
    WalkArgs a;
    a.com = t->node_com; a.cell = t->node_cell; a.lo = t->node_lo; a.hi = t->node_hi;
    a.info = t->node_info; a.spos = t->spos; a.sh = t->sh; a.tab = t->split_tab;
    a.tgt_slot = tgt_slot; a.tgt_out = tgt_out; a.a_old = a_old; a.acc_out = acc_out; a.pot_out = pot_out;
    a.n_active = (uint32_t)n_active;
    a.n_groups = (uint32_t)((n_active + 31) / 32);
    a.work = t->d_status + 1;
    a.status = t->d_status;
    a.counters = t->d_counters;
    a.spill = reinterpret_cast<uint32_t *>(t->walk_spill);
    a.spill_cap = SPILL_CAP;
    const og_params &p = t->prm;
    WalkConst &c = a.c;
    c.dL = (double)t->box;
    c.drcut = (double)p.rcut_over_rs * (double)p.r_s;
    c.dG = (double)p.G; c.dalpha = (double)p.alpha; c.dtheta2 = (double)p.theta * (double)p.theta;
    c.L = t->box; c.invL = 1.0f / t->box;
    c.rcut = (float)c.drcut; c.rcut2 = (float)(c.drcut * c.drcut);
    c.cull_r = (float)(c.drcut * (1.0 + 1e-5) + 1e-6 * c.dL);
    c.G = p.G; c.alpha = p.alpha; c.theta2 = (float)c.dtheta2;
    c.tab_scale = (float)((double)OG_NTAB / c.drcut);
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
