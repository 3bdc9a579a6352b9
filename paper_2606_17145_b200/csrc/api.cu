// api.cu -- the C ABI of include/og.h: argument checks, device arena layout, stream-ordered
// launch sequences.  Every step of the path runs in the kernels of this directory; there is no
// CPU fallback.
#include <atomic>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include "og_internal.cuh"

static thread_local char g_err[512] = "";

void og_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

extern "C" const char *og_last_error(void) { return g_err; }

namespace {

inline size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

struct Layout {
    size_t keysA, keysB, idxA, idxB, sort_scratch, spos, sh, inv_perm;
    size_t level, first, count, first_child, nchild, com, cell, lo, hi, info, rec;
    size_t oct_scratch, level_start, status, counters, small_end, spill, cost, cover, total;
};

Layout make_layout(uint64_t n, uint32_t max_nodes, int sm_count, uint32_t spill_entries, bool count)
{
    Layout L;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
    L.keysA = take(n * 8); L.keysB = take(n * 8);
    L.idxA = take(n * 4);  L.idxB = take(n * 4);
    L.sort_scratch = take(ogk_sort_scratch_bytes(n));
    L.spos = take(n * 16); L.sh = take(n * 4); L.inv_perm = take(n * 4);
    const size_t M = max_nodes;
    L.level = take(M); L.first = take(M * 4); L.count = take(M * 4); L.first_child = take(M * 4);
    L.nchild = take(M);
    L.com = take(M * 16); L.cell = take(M * 16); L.lo = take(M * 16); L.hi = take(M * 16);
    L.info = take(M * 8);
    L.rec = take(M * 48);
    L.oct_scratch = take(ogk_octree_scratch_bytes(max_nodes));
    L.level_start = take(24 * 4);
    L.status = take(16 * 4);
    L.counters = take(OGC_N * 8);
    L.small_end = o;
    L.spill = take(ogk_walk_spill_bytes(sm_count, spill_entries));
    L.cost = take(count ? n * 4 : 0);
    L.cover = take(37449 * 4);
    L.total = o;
    return L;
}

uint32_t default_max_nodes(uint64_t n, const og_params *p)
{
    if (p->max_nodes) return p->max_nodes;
    // R6: observed nodes/N is 0.14..0.49 at leaf_max = 8 and 1.49 at leaf_max = 1
    uint64_t m = (p->leaf_max >= 4) ? n : 3 * n;
    if (m < 4096) m = 4096;
    if (m > 0x7fffffffull) m = 0x7fffffffull;
    return (uint32_t)m;
}

bool check_params(const og_params *p, uint64_t n, float box)
{
    if (!p) { og_set_error("params is NULL"); return false; }
    if (p->struct_size != sizeof(og_params)) {
        og_set_error("og_params.struct_size = %u, expected %zu", p->struct_size, sizeof(og_params));
        return false;
    }
    if (n == 0 || n >= (1ull << 31)) { og_set_error("n = %llu out of range [1, 2^31)", (unsigned long long)n); return false; }
    if (!(box > 0.0f)) { og_set_error("box must be > 0"); return false; }
    if (!(p->flags & OG_PERIODIC)) { og_set_error("OG_PERIODIC is required in this build"); return false; }
    if ((p->flags & OG_WALK_G32) && (p->flags & OG_WALK_G8)) {
        og_set_error("OG_WALK_G32 and OG_WALK_G8 exclude each other");
        return false;
    }
    if (p->leaf_max == 0) { og_set_error("leaf_max must be >= 1"); return false; }
    if (!(p->r_s > 0.0f) || !(p->rcut_over_rs > 0.0f)) { og_set_error("r_s and rcut_over_rs must be > 0"); return false; }
    if (p->rcut_over_rs > 5.0f) {
        og_set_error("rcut_over_rs = %g > 5: the split-factor polynomial is fitted on r / (2 r_s) <= 2.5", (double)p->rcut_over_rs);
        return false;
    }
    if (!((double)p->rcut_over_rs * (double)p->r_s < 0.5 * (double)box)) {
        og_set_error("r_cut = %g must be < box/2 = %g (nearest-image convention, R13)",
                     (double)p->rcut_over_rs * (double)p->r_s, 0.5 * (double)box);
        return false;
    }
    if (p->walk_stack_entries != 0 && (p->walk_stack_entries < 64 || p->walk_stack_entries > 256 || (p->walk_stack_entries & 1u))) {
        og_set_error("walk_stack_entries = %u: must be 0 (default) or an even number in [64, 256]", p->walk_stack_entries);
        return false;
    }
    if (p->walk_spill_entries > (1u << 20)) { og_set_error("walk_spill_entries = %u: at most 2^20", p->walk_spill_entries); return false; }
    return true;
}

int device_sm_count(int *device_out)
{
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -1;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    if (device_out) *device_out = dev;
    return sms;
}

}  // namespace

// SMs of the current device, for the grid-stride kernels that size their grid as a multiple of it (the sort's histogram
// pass, the time-step reductions): asked once per device, 148 (a B200) when no device is visible.
int ogk_sm_count(void)
{
    static std::atomic<int> cache[64];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return 148; }
    if (dev >= 0 && dev < 64) {
        const int c = cache[dev].load(std::memory_order_relaxed);
        if (c > 0) return c;
    }
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) {
        (void)cudaGetLastError();
        return 148;
    }
    if (dev >= 0 && dev < 64) cache[dev].store(sms, std::memory_order_relaxed);
    return sms;
}

namespace {

// Stream-ordered allocations come from a pool owned by the library whose release threshold is
// unlimited: a tree arena (GBs) freed by og_tree_free is reused by the next og_tree_build instead
// of going back to the driver at every synchronisation (the default pool's behaviour, ~16 ms per
// 3 GB arena on B200).
std::mutex g_pool_mu;
cudaMemPool_t g_pools[64] = {};

cudaError_t og_malloc_async(void **ptr, size_t bytes, cudaStream_t st)
{
    std::mutex &mu = g_pool_mu;
    cudaMemPool_t *pools = g_pools;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64) return cudaMallocAsync(ptr, bytes, st);
    cudaMemPool_t pool;
    {
        std::lock_guard<std::mutex> lk(mu);
        if (!pools[dev]) {
            cudaMemPoolProps props = {};
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = dev;
            e = cudaMemPoolCreate(&pools[dev], &props);
            if (e != cudaSuccess) { pools[dev] = nullptr; return e; }
            unsigned long long keep = ~0ull;
            (void)cudaMemPoolSetAttribute(pools[dev], cudaMemPoolAttrReleaseThreshold, &keep);
        }
        pool = pools[dev];
    }
    return cudaMallocFromPoolAsync(ptr, bytes, pool, st);
}

int status_from_bits(uint32_t bits)
{
    if (bits & OG_DEV_NODE_OVERFLOW) return OG_ERR_NODE_OVERFLOW;
    if (bits & OG_DEV_BAD_POSITION) return OG_ERR_BAD_POSITION;
    if (bits & OG_DEV_STACK_OVERFLOW) return OG_ERR_STACK_OVERFLOW;
    if (bits & OG_DEV_BAD_INDEX) return OG_ERR_INVALID_ARG;
    if (bits & OG_DEV_NGB_OVERFLOW) return OG_ERR_NGB_OVERFLOW;
    return OG_OK;
}

// Synchronises the streams the tree has been used on and refreshes the host copies.
int tree_sync(const og_tree *t, uint32_t *bits_out)
{
    OG_CUDA_TRY(cudaEventSynchronize(t->ev_built), return OG_ERR_CUDA);
    if (t->walked) OG_CUDA_TRY(cudaEventSynchronize(t->ev_walked), return OG_ERR_CUDA);
    uint32_t ls[24];
    OG_CUDA_TRY(cudaMemcpy(ls, t->d_level_start, sizeof(ls), cudaMemcpyDeviceToHost), return OG_ERR_CUDA);
    t->n_nodes_host = ls[22];
    uint32_t ml = 0;
    for (uint32_t lv = 0; lv <= OG_MAX_LEVEL; ++lv)
        if (ls[lv + 1] > ls[lv]) ml = lv;
    t->max_level_host = ml;
    uint32_t bits = 0;
    OG_CUDA_TRY(cudaMemcpy(&bits, t->d_status, sizeof(bits), cudaMemcpyDeviceToHost), return OG_ERR_CUDA);
    if (bits_out) *bits_out = bits;
    return OG_OK;
}

void tree_delete(og_tree *t)
{
    if (t->ev_built) cudaEventDestroy(t->ev_built);
    if (t->ev_walked) cudaEventDestroy(t->ev_walked);
    delete t;
}

}  // namespace

extern "C" size_t og_tree_workspace_bytes(uint64_t n, const og_params *params)
{
    if (!params || params->struct_size != sizeof(og_params) || n == 0 || n >= (1ull << 31)) return 0;
    int sms = device_sm_count(nullptr);
    if (sms <= 0) sms = 148;  // no device visible: size for a B200
    return make_layout(n, default_max_nodes(n, params), sms, ogk_walk_spill_entries(params), (params->flags & OG_COUNT) != 0).total;
}

// og_tree_build; `before_gather` (may be NULL) is awaited on the stream before mass / soft are first read
// (the HOST entry point copies them on a second stream while the keys are generated and sorted).
static og_tree *tree_build_impl(const float *pos, const float *mass, const float *soft, uint64_t n,
                                float box, const og_params *params, og_stream stream, cudaEvent_t before_gather)
{
    g_err[0] = 0;
    if (!check_params(params, n, box)) return nullptr;
    if (!pos || !mass || !soft) { og_set_error("pos / mass / soft must be non-NULL device pointers"); return nullptr; }
    int dev = 0;
    const int sms = device_sm_count(&dev);
    if (sms <= 0) { og_set_error("no CUDA device available (there is no CPU fallback)"); return nullptr; }
    cudaStream_t st = (cudaStream_t)stream;
    og_tree *t = new (std::nothrow) og_tree();
    if (!t) { og_set_error("host allocation failed"); return nullptr; }
    memset(t, 0, sizeof(*t));
    t->n = n; t->box = box; t->prm = *params; t->device = dev; t->sm_count = sms;
    t->max_nodes = default_max_nodes(n, params);
    t->build_stream = st; t->n_nodes_host = -1;
    t->walk_spill_cap = ogk_walk_spill_entries(params);
    if (cudaEventCreateWithFlags(&t->ev_built, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&t->ev_walked, cudaEventDisableTiming) != cudaSuccess) {
        og_set_error("cudaEventCreate failed");
        (void)cudaGetLastError();
        if (t->ev_built) cudaEventDestroy(t->ev_built);
        delete t;
        return nullptr;
    }
    const Layout L = make_layout(n, t->max_nodes, sms, t->walk_spill_cap, (params->flags & OG_COUNT) != 0);
    if (params->workspace) {
        if (params->workspace_bytes < L.total || ((uintptr_t)params->workspace & 255u)) {
            og_set_error("workspace too small or not 256-byte aligned: %zu bytes given, %zu needed",
                         params->workspace_bytes, L.total);
            tree_delete(t);
            return nullptr;
        }
        t->arena = params->workspace; t->owns_arena = 0;
    } else {
        cudaError_t e = og_malloc_async(&t->arena, L.total, st);
        if (e != cudaSuccess) {
            og_set_error("cudaMallocAsync(%zu bytes) failed: %s", L.total, cudaGetErrorString(e));
            (void)cudaGetLastError();
            tree_delete(t);
            return nullptr;
        }
        t->owns_arena = 1;
    }
    t->arena_bytes = L.total;
    char *b = reinterpret_cast<char *>(t->arena);
    uint64_t *keysA = (uint64_t *)(b + L.keysA), *keysB = (uint64_t *)(b + L.keysB);
    uint32_t *idxA = (uint32_t *)(b + L.idxA), *idxB = (uint32_t *)(b + L.idxB);
    t->spos = (float4 *)(b + L.spos); t->sh = (float *)(b + L.sh); t->inv_perm = (uint32_t *)(b + L.inv_perm);
    t->node_level = (uint8_t *)(b + L.level); t->node_first = (uint32_t *)(b + L.first);
    t->node_count = (uint32_t *)(b + L.count); t->node_first_child = (uint32_t *)(b + L.first_child);
    t->node_nchild = (uint8_t *)(b + L.nchild);
    t->node_com = (float4 *)(b + L.com); t->node_cell = (float4 *)(b + L.cell);
    t->node_lo = (float4 *)(b + L.lo); t->node_hi = (float4 *)(b + L.hi); t->node_info = (uint2 *)(b + L.info);
    t->node_rec = (uint4 *)(b + L.rec);
    t->d_level_start = (uint32_t *)(b + L.level_start); t->d_status = (uint32_t *)(b + L.status);
    t->d_counters = (unsigned long long *)(b + L.counters);
    t->walk_cost = (params->flags & OG_COUNT) ? (uint32_t *)(b + L.cost) : nullptr;
    t->cover = (uint32_t *)(b + L.cover);
    t->walk_spill = b + L.spill; t->walk_spill_bytes = ogk_walk_spill_bytes(sms, t->walk_spill_cap);

#define OG_BUILD_TRY(expr)                                                    \
    OG_CUDA_TRY(expr, {                                                       \
        if (t->owns_arena) cudaFreeAsync(t->arena, st);                       \
        tree_delete(t);                                                       \
        return nullptr;                                                       \
    })
    // level_start, status, counters are adjacent: clear them in one memset
    OG_BUILD_TRY(cudaMemsetAsync(b + L.level_start, 0, L.small_end - L.level_start, st));
    OG_BUILD_TRY(ogk_keys(pos, n, box, keysA, idxA, t->d_status, (params->flags & OG_VALIDATE_POS) != 0, st));
    int in_alt = 0;
    OG_BUILD_TRY(ogk_radix_sort(keysA, idxA, keysB, idxB, n, 0, 64, b + L.sort_scratch, &in_alt, st));
    t->keys = in_alt ? keysB : keysA;
    t->perm = in_alt ? idxB : idxA;
    if (before_gather) OG_BUILD_TRY(cudaStreamWaitEvent(st, before_gather, 0));
    OG_BUILD_TRY(ogk_gather(pos, mass, soft, t->perm, n, t->spos, t->sh, t->inv_perm, st));
    OG_BUILD_TRY(ogk_octree_upward(t, b + L.oct_scratch, st));
    OG_BUILD_TRY(cudaEventRecord(t->ev_built, st));
#undef OG_BUILD_TRY
    return t;
}

extern "C" og_tree *og_tree_build(const float *pos, const float *mass, const float *soft, uint64_t n,
                                  float box, const og_params *params, og_stream stream)
{
    return tree_build_impl(pos, mass, soft, n, box, params, stream, nullptr);
}

extern "C" int og_shortrange_accel(const og_tree *t, const uint32_t *active_idx, uint64_t n_active,
                                   const float *a_old, float *acc_out, float *pot_out, og_stream stream)
{
    g_err[0] = 0;
    if (!t) { og_set_error("tree is NULL"); return OG_ERR_INVALID_ARG; }
    if (n_active == 0) return OG_OK;   // empty active list: nothing to do (pointers of empty buffers may be NULL)
    if (!acc_out) { og_set_error("acc_out is NULL"); return OG_ERR_INVALID_ARG; }
    if (!active_idx && n_active != t->n) {
        og_set_error("active_idx == NULL requires n_active == n (%llu != %llu)", (unsigned long long)n_active,
                     (unsigned long long)t->n);
        return OG_ERR_INVALID_ARG;
    }
    if (n_active >= (1ull << 31)) { og_set_error("n_active out of range"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    // after the build, and after the previous walk on this tree (its scratch state is shared): og.h
    if (st != t->build_stream) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_built, 0), return OG_ERR_CUDA);
    if (t->walked) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_walked, 0), return OG_ERR_CUDA);
    if (!active_idx) {
        OG_CUDA_TRY(ogk_walk(t, nullptr, t->perm, n_active, a_old, acc_out, pot_out, st), return OG_ERR_CUDA);
        OG_CUDA_TRY(cudaEventRecord(t->ev_walked, st), return OG_ERR_CUDA);
        t->walked = true;
        t->walk_kind = 1;
        return OG_OK;
    }
    // active subset: order the targets by sorted slot so that a warp's 32 targets are neighbours
    const size_t na = (size_t)n_active;
    const size_t o_k0 = 0, o_k1 = align_up(na * 8), o_v0 = o_k1 + align_up(na * 8), o_v1 = o_v0 + align_up(na * 4),
                 o_sl = o_v1 + align_up(na * 4), o_sc = o_sl + align_up(na * 4),
                 total = o_sc + align_up(ogk_sort_scratch_bytes(n_active));
    char *tmp = nullptr;
    cudaError_t e = og_malloc_async((void **)&tmp, total, st);
    if (e != cudaSuccess) {
        og_set_error("cudaMallocAsync(%zu bytes) failed: %s", total, cudaGetErrorString(e));
        (void)cudaGetLastError();
        return OG_ERR_OUT_OF_MEMORY;
    }
    uint64_t *k0 = (uint64_t *)(tmp + o_k0), *k1 = (uint64_t *)(tmp + o_k1);
    uint32_t *v0 = (uint32_t *)(tmp + o_v0), *v1 = (uint32_t *)(tmp + o_v1), *slots = (uint32_t *)(tmp + o_sl);
    int bits = 1;
    while (bits < 32 && (1ull << bits) < t->n) ++bits;
    int in_alt = 0;
#define OG_ACC_TRY(expr) OG_CUDA_TRY(expr, { cudaFreeAsync(tmp, st); return OG_ERR_CUDA; })
    OG_ACC_TRY(ogk_active_slots(active_idx, t->inv_perm, t->n, n_active, k0, v0, t->d_status, st));
    OG_ACC_TRY(ogk_radix_sort(k0, v0, k1, v1, n_active, 0, bits, tmp + o_sc, &in_alt, st));
    // grouping (og.h): n_active * div < span of the list in sorted slots -> 8 targets per warp.  The flags fix it through
    // the divisor: 0 makes the test true for every list, 2^32 - 1 false (n_active >= 1, span <= n < 2^31)
    const uint32_t sparse_div = (t->prm.flags & OG_WALK_G8) ? 0u : (t->prm.flags & OG_WALK_G32) ? 0xffffffffu : OG_SPARSE_DIV;
    OG_ACC_TRY(ogk_unpack_slots(in_alt ? k1 : k0, n_active, slots, sparse_div, t->d_status + 2, st));
    OG_ACC_TRY(ogk_walk(t, slots, in_alt ? v1 : v0, n_active, a_old, acc_out, pot_out, st));
    OG_ACC_TRY(cudaEventRecord(t->ev_walked, st));
    t->walked = true;
    t->walk_kind = 2;
    OG_ACC_TRY(cudaFreeAsync(tmp, st));
#undef OG_ACC_TRY
    return OG_OK;
}

extern "C" int og_sph_density(const og_tree *t, const uint32_t *active_idx, uint64_t n_active, float n_des, float tol_n,
                              const float *h_guess, float *h_out, float *rho_out, float *nn_out, og_stream stream)
{
    g_err[0] = 0;
    if (!t) { og_set_error("tree is NULL"); return OG_ERR_INVALID_ARG; }
    if (n_active == 0) return OG_OK;
    if (!h_out) { og_set_error("h_out is NULL"); return OG_ERR_INVALID_ARG; }
    if (!active_idx && n_active != t->n) {
        og_set_error("active_idx == NULL requires n_active == n (%llu != %llu)", (unsigned long long)n_active,
                     (unsigned long long)t->n);
        return OG_ERR_INVALID_ARG;
    }
    if (n_active >= (1ull << 31)) { og_set_error("n_active out of range"); return OG_ERR_INVALID_ARG; }
    if (!(n_des > 32.0f / 3.0f) || !(n_des <= 256.0f) || !(tol_n >= 0.0f)) {
        og_set_error("og_sph_density needs 32/3 < n_des <= 256 and tol_n >= 0 (n_des = %g, tol_n = %g)", n_des, tol_n);
        return OG_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (st != t->build_stream) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_built, 0), return OG_ERR_CUDA);
    // the cell table of the tree is written by the first call (calls on one tree from several host threads at once are not
    // supported, og.h; a later call on another stream is ordered after this one by the tree's event below)
    if (t->walked) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_walked, 0), return OG_ERR_CUDA);
    if (!t->cover_built) {
        OG_CUDA_TRY(ogk_cover(t, st), return OG_ERR_CUDA);
        t->cover_built = true;
    }
    OG_CUDA_TRY(ogk_sph_density(t, active_idx, n_active, n_des, tol_n, h_guess, h_out, rho_out, nn_out, st),
                return OG_ERR_CUDA);
    // og_tree_free and og_tree_status wait for this call like for a walk
    OG_CUDA_TRY(cudaEventRecord(t->ev_walked, st), return OG_ERR_CUDA);
    t->walked = true;
    return OG_OK;
}

// ---- row f4 ------------------------------------------------------------------------------------------------------
extern "C" int og_shortrange_accel_ext(const og_tree *t, const float *tpos, const float *tsoft, uint64_t n_t,
                                       const float *a_old, float *acc_out, float *pot_out, og_stream stream)
{
    g_err[0] = 0;
    if (!t) { og_set_error("tree is NULL"); return OG_ERR_INVALID_ARG; }
    if (n_t == 0) return OG_OK;
    if (!tpos || !tsoft || !acc_out) { og_set_error("tpos / tsoft / acc_out must be non-NULL device pointers"); return OG_ERR_INVALID_ARG; }
    if (n_t >= (1ull << 31)) { og_set_error("n_t out of range"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    if (st != t->build_stream) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_built, 0), return OG_ERR_CUDA);
    if (t->walked) OG_CUDA_TRY(cudaStreamWaitEvent(st, t->ev_walked, 0), return OG_ERR_CUDA);
    // Morton order of the imported targets, so that a warp's 32 targets are neighbours (as for the tree's own particles)
    const size_t nt = (size_t)n_t;
    const size_t o_k0 = 0, o_k1 = align_up(nt * 8), o_v0 = o_k1 + align_up(nt * 8), o_v1 = o_v0 + align_up(nt * 4),
                 o_ext = o_v1 + align_up(nt * 4), o_sc = o_ext + align_up(nt * 16),
                 total = o_sc + align_up(ogk_sort_scratch_bytes(n_t));
    char *tmp = nullptr;
    cudaError_t e = og_malloc_async((void **)&tmp, total, st);
    if (e != cudaSuccess) {
        og_set_error("cudaMallocAsync(%zu bytes) failed: %s", total, cudaGetErrorString(e));
        (void)cudaGetLastError();
        return OG_ERR_OUT_OF_MEMORY;
    }
    uint64_t *k0 = (uint64_t *)(tmp + o_k0), *k1 = (uint64_t *)(tmp + o_k1);
    uint32_t *v0 = (uint32_t *)(tmp + o_v0), *v1 = (uint32_t *)(tmp + o_v1);
    float4 *ext = (float4 *)(tmp + o_ext);
    int in_alt = 0;
#define OG_EXT_TRY(expr) OG_CUDA_TRY(expr, { cudaFreeAsync(tmp, st); return OG_ERR_CUDA; })
    OG_EXT_TRY(ogk_keys(tpos, n_t, t->box, k0, v0, t->d_status, (t->prm.flags & OG_VALIDATE_POS) != 0, st));
    OG_EXT_TRY(ogk_radix_sort(k0, v0, k1, v1, n_t, 0, 64, tmp + o_sc, &in_alt, st));
    const uint32_t *order = in_alt ? v1 : v0;
    OG_EXT_TRY(ogk_ext_gather(tpos, tsoft, order, n_t, ext, st));
    // grouping as for an active list (og.h), the targets' density taken against the tree's particles in their key range
    const uint32_t sparse_div = (t->prm.flags & OG_WALK_G8) ? 0u : (t->prm.flags & OG_WALK_G32) ? 0xffffffffu : OG_SPARSE_DIV;
    OG_EXT_TRY(ogk_ext_sparse(in_alt ? k1 : k0, n_t, t->keys, t->n, sparse_div, t->d_status + 2, st));
    OG_EXT_TRY(ogk_walk(t, nullptr, order, n_t, a_old, acc_out, pot_out, st, ext, t->d_status + 2));
    OG_EXT_TRY(cudaEventRecord(t->ev_walked, st));
    t->walked = true;
    t->walk_kind = 2;
    OG_EXT_TRY(cudaFreeAsync(tmp, st));
#undef OG_EXT_TRY
    return OG_OK;
}

static int domain_keys(const float *pos, uint64_t n, float box, uint64_t **keys, cudaStream_t st)
{
    *keys = nullptr;
    if (n == 0) return OG_OK;
    if (!pos || !(box > 0.0f) || n >= (1ull << 31)) { og_set_error("bad pos / box / n"); return OG_ERR_INVALID_ARG; }
    cudaError_t e = og_malloc_async((void **)keys, n * sizeof(uint64_t), st);
    if (e != cudaSuccess) { og_set_error("cudaMallocAsync failed: %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return OG_ERR_OUT_OF_MEMORY; }
    OG_CUDA_TRY(ogk_keys(pos, n, box, *keys, nullptr, nullptr, false, st), { cudaFreeAsync(*keys, st); return OG_ERR_CUDA; });
    return OG_OK;
}

extern "C" int og_domain_cell_hist(const float *pos, uint64_t n, float box, uint32_t *hist, og_stream stream)
{
    g_err[0] = 0;
    if (!hist) { og_set_error("hist is NULL"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t *keys = nullptr;
    const int rc = domain_keys(pos, n, box, &keys, st);
    if (rc != OG_OK) return rc;
    OG_CUDA_TRY(ogk_cell_hist(keys, n, hist, st), { if (keys) cudaFreeAsync(keys, st); return OG_ERR_CUDA; });
    if (keys) OG_CUDA_TRY(cudaFreeAsync(keys, st), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_domain_owner(const float *pos, uint64_t n, float box, const uint32_t *splitters, uint32_t n_domains,
                               uint32_t *owner, og_stream stream)
{
    g_err[0] = 0;
    if (n == 0) return OG_OK;
    if (!splitters || !owner || n_domains == 0) { og_set_error("splitters / owner NULL or n_domains == 0"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    uint64_t *keys = nullptr;
    const int rc = domain_keys(pos, n, box, &keys, st);
    if (rc != OG_OK) return rc;
    OG_CUDA_TRY(ogk_owner(keys, n, splitters, n_domains, owner, st), { cudaFreeAsync(keys, st); return OG_ERR_CUDA; });
    OG_CUDA_TRY(cudaFreeAsync(keys, st), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_let_export_list(const float *tpos, uint64_t n_t, const float *boxes, uint32_t n_boxes, float r_cut,
                                  float box, uint32_t *list_out, uint64_t *count_host, og_stream stream)
{
    g_err[0] = 0;
    if (!count_host) { og_set_error("count_host is NULL"); return OG_ERR_INVALID_ARG; }
    *count_host = 0;
    if (n_t == 0 || n_boxes == 0) return OG_OK;
    if (!tpos || !boxes || !list_out || n_boxes > 1024 || !(box > 0.0f) || n_t >= (1ull << 31)) {
        og_set_error("bad tpos / boxes / list_out, or n_boxes > 1024"); return OG_ERR_INVALID_ARG;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t o_sc = align_up((size_t)n_t), total = o_sc + align_up(ogk_flag_scratch_bytes(n_t));
    char *tmp = nullptr;
    cudaError_t e = og_malloc_async((void **)&tmp, total, st);
    if (e != cudaSuccess) { og_set_error("cudaMallocAsync failed: %s", cudaGetErrorString(e)); (void)cudaGetLastError(); return OG_ERR_OUT_OF_MEMORY; }
    uint32_t *total_dev = nullptr, cnt = 0;
#define OG_LET_TRY(expr) OG_CUDA_TRY(expr, { cudaFreeAsync(tmp, st); return OG_ERR_CUDA; })
    OG_LET_TRY(ogk_let_mark(tpos, n_t, boxes, n_boxes, r_cut, box, (uint8_t *)tmp, st));
    OG_LET_TRY(ogk_flag_compact((const uint8_t *)tmp, n_t, list_out, (uint32_t *)(tmp + o_sc), &total_dev, st));
    OG_LET_TRY(cudaMemcpyAsync(&cnt, total_dev, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    OG_LET_TRY(cudaStreamSynchronize(st));
    OG_LET_TRY(cudaFreeAsync(tmp, st));
#undef OG_LET_TRY
    *count_host = cnt;
    return OG_OK;
}

extern "C" int og_let_accumulate(float *acc, float *pot, const uint32_t *idx, const float *part_acc, const float *part_pot,
                                 uint64_t m, uint64_t n, og_stream stream)
{
    g_err[0] = 0;
    if (m == 0) return OG_OK;
    if (!acc || !idx || !part_acc) { og_set_error("acc / idx / part_acc NULL"); return OG_ERR_INVALID_ARG; }
    OG_CUDA_TRY(ogk_let_accumulate(acc, pot, idx, part_acc, part_pot, m, n, (cudaStream_t)stream), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_tree_get(const og_tree *t, int field, const void **dev_ptr, uint64_t *count)
{
    g_err[0] = 0;
    if (!t || !dev_ptr || !count) { og_set_error("NULL argument"); return OG_ERR_INVALID_ARG; }
    if (t->n_nodes_host < 0) {
        const int rc = tree_sync(t, nullptr);
        if (rc != OG_OK) return rc;
    }
    const uint64_t nn = (uint64_t)t->n_nodes_host;
    switch (field) {
    case OG_F_KEYS_SORTED: *dev_ptr = t->keys; *count = t->n; break;
    case OG_F_PERM: *dev_ptr = t->perm; *count = t->n; break;
    case OG_F_INV_PERM: *dev_ptr = t->inv_perm; *count = t->n; break;
    case OG_F_SPOS: *dev_ptr = t->spos; *count = t->n * 4; break;
    case OG_F_SH: *dev_ptr = t->sh; *count = t->n; break;
    case OG_F_NODE_LEVEL: *dev_ptr = t->node_level; *count = nn; break;
    case OG_F_NODE_FIRST: *dev_ptr = t->node_first; *count = nn; break;
    case OG_F_NODE_COUNT: *dev_ptr = t->node_count; *count = nn; break;
    case OG_F_NODE_FIRST_CHILD: *dev_ptr = t->node_first_child; *count = nn; break;
    case OG_F_NODE_NCHILD: *dev_ptr = t->node_nchild; *count = nn; break;
    case OG_F_NODE_COM: *dev_ptr = t->node_com; *count = nn * 4; break;
    case OG_F_NODE_CELL: *dev_ptr = t->node_cell; *count = nn * 4; break;
    case OG_F_NODE_LO: *dev_ptr = t->node_lo; *count = nn * 4; break;
    case OG_F_NODE_HI: *dev_ptr = t->node_hi; *count = nn * 4; break;
    case OG_F_LEVEL_START: *dev_ptr = t->d_level_start; *count = 23; break;
    case OG_F_WALK_COST:
        if (!t->walk_cost) { og_set_error("OG_F_WALK_COST needs a tree built with OG_COUNT"); return OG_ERR_INVALID_ARG; }
        *dev_ptr = t->walk_cost; *count = t->n; break;
    default: og_set_error("unknown field %d", field); return OG_ERR_INVALID_ARG;
    }
    return OG_OK;
}

extern "C" int og_tree_status(const og_tree *t)
{
    g_err[0] = 0;
    if (!t) { og_set_error("tree is NULL"); return OG_ERR_INVALID_ARG; }
    uint32_t bits = 0;
    const int rc = tree_sync(t, &bits);
    if (rc != OG_OK) return rc;
    const int s = status_from_bits(bits);
    if (s != OG_OK) og_set_error("device-latched status bits 0x%x", bits);
    return s;
}

extern "C" int og_tree_stats(const og_tree *t, og_stats *out)
{
    g_err[0] = 0;
    if (!t || !out) { og_set_error("NULL argument"); return OG_ERR_INVALID_ARG; }
    const int rc = tree_sync(t, nullptr);
    if (rc != OG_OK) return rc;
    unsigned long long c[OGC_N];
    OG_CUDA_TRY(cudaMemcpy(c, t->d_counters, sizeof(c), cudaMemcpyDeviceToHost), return OG_ERR_CUDA);
    memset(out, 0, sizeof(*out));
    out->n = t->n; out->n_nodes = (uint64_t)t->n_nodes_host; out->max_level = t->max_level_host;
    out->V_full = c[OGC_V_FULL]; out->V_cull = c[OGC_V_CULL]; out->A_in = c[OGC_A_IN];
    out->P_in = c[OGC_P_IN]; out->P_soft = c[OGC_P_SOFT]; out->P_out = c[OGC_P_OUT];
    out->fp64_rechecks = c[OGC_FP64];
    out->cl_drop = c[OGC_CL_DROP]; out->cl_open = c[OGC_CL_OPEN]; out->cl_accept = c[OGC_CL_ACCEPT];
    out->cl_generic = c[OGC_CL_GENERIC]; out->pt_drop = c[OGC_PT_DROP]; out->pt_shift = c[OGC_PT_SHIFT];
    out->pt_wrap = c[OGC_PT_WRAP]; out->batches = c[OGC_BATCHES];
    out->stack_spills = c[OGC_SPILLS];
    if (t->walk_kind == 2) {
        uint32_t sparse = 0;
        OG_CUDA_TRY(cudaMemcpy(&sparse, t->d_status + 2, sizeof(sparse), cudaMemcpyDeviceToHost), return OG_ERR_CUDA);
        out->walk_targets_per_warp = sparse ? 8u : 32u;
    } else {
        out->walk_targets_per_warp = t->walk_kind == 1 ? 32u : 0u;
    }
    return OG_OK;
}

extern "C" void og_tree_free(og_tree *t, og_stream stream)
{
    if (!t) return;
    if (t->owns_arena && t->arena) {
        // the arena may still be in use by the build or the last walk on another stream: order the free after them
        cudaStreamWaitEvent((cudaStream_t)stream, t->ev_built, 0);
        if (t->walked) cudaStreamWaitEvent((cudaStream_t)stream, t->ev_walked, 0);
        cudaFreeAsync(t->arena, (cudaStream_t)stream);
    }
    tree_delete(t);
}

extern "C" int og_morton_keys(const float *pos, uint64_t n, float box, uint64_t *keys, uint32_t *idx,
                              og_stream stream)
{
    g_err[0] = 0;
    if (!pos || !keys || n == 0 || n >= (1ull << 31) || !(box > 0.0f)) {
        og_set_error("og_morton_keys: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    OG_CUDA_TRY(ogk_keys(pos, n, box, keys, idx, nullptr, false, (cudaStream_t)stream), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" size_t og_radix_sort_scratch_bytes(uint64_t n) { return ogk_sort_scratch_bytes(n); }

extern "C" int og_radix_sort_pairs(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt,
                                   uint64_t n, int begin_bit, int end_bit, void *scratch, size_t scratch_bytes,
                                   int *result_in_alt, og_stream stream)
{
    g_err[0] = 0;
    if (!keys || !vals || !keys_alt || !vals_alt || !scratch || n == 0 || n >= (1ull << 31) || begin_bit < 0 ||
        end_bit > 64 || begin_bit >= end_bit || scratch_bytes < ogk_sort_scratch_bytes(n)) {
        og_set_error("og_radix_sort_pairs: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    OG_CUDA_TRY(ogk_radix_sort(keys, vals, keys_alt, vals_alt, n, begin_bit, end_bit, scratch, result_in_alt,
                               (cudaStream_t)stream),
                return OG_ERR_CUDA);
    return OG_OK;
}

// The variant of og_radix_sort_pairs whose scratch is a fixed array inside the library (radix_sort.cu): argument checks
// here, nothing allocated anywhere on the path.
extern "C" int og_radix_sort_pairs_noalloc(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt,
                                           uint64_t n, int begin_bit, int end_bit, int *result_in_alt, og_stream stream)
{
    g_err[0] = 0;
    if (!keys || !vals || !keys_alt || !vals_alt || n == 0 || begin_bit < 0 || end_bit > 64 || begin_bit >= end_bit) {
        og_set_error("og_radix_sort_pairs_noalloc: bad argument");
        return OG_ERR_INVALID_ARG;
    }
    if (n > (uint64_t)ogk_sort_noalloc_max_n()) {
        og_set_error("og_radix_sort_pairs_noalloc: n = %llu exceeds OG_SORT_NOALLOC_MAX_N = %llu, the capacity of the "
                     "library's built-in scratch array (use og_radix_sort_pairs with caller-supplied scratch)",
                     (unsigned long long)n, (unsigned long long)ogk_sort_noalloc_max_n());
        return OG_ERR_INVALID_ARG;
    }
    OG_CUDA_TRY(ogk_radix_sort_noalloc(keys, vals, keys_alt, vals_alt, n, begin_bit, end_bit, result_in_alt,
                                       (cudaStream_t)stream),
                return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_shortrange_accel_host(const float *pos, const float *mass, const float *soft, uint64_t n,
                                        float box, const og_params *params, const uint32_t *active_idx,
                                        uint64_t n_active, const float *a_old, float *acc_out, float *pot_out,
                                        og_stream stream)
{
    g_err[0] = 0;
    if (!check_params(params, n, box)) return OG_ERR_INVALID_ARG;
    if (!pos || !mass || !soft || !acc_out) { og_set_error("NULL host pointer"); return OG_ERR_INVALID_ARG; }
    if (!active_idx && n_active != n) { og_set_error("active_idx == NULL requires n_active == n"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t na = (size_t)n_active;
    const size_t o_pos = 0, o_m = o_pos + align_up(n * 12), o_s = o_m + align_up(n * 4), o_ai = o_s + align_up(n * 4),
                 o_ao = o_ai + align_up(na * 4), o_acc = o_ao + align_up(na * 4), o_pot = o_acc + align_up(na * 12),
                 total = o_pot + align_up(na * 4);
    char *d = nullptr;
    cudaError_t e = og_malloc_async((void **)&d, total, st);
    if (e != cudaSuccess) {
        og_set_error("cudaMallocAsync(%zu bytes) failed: %s", total, cudaGetErrorString(e));
        (void)cudaGetLastError();
        return OG_ERR_OUT_OF_MEMORY;
    }
    int rc = OG_OK;
    og_tree *t = nullptr;
    // Host-to-device copies run on a second stream so that they overlap the build: the keys and the sort
    // need only pos, the gather waits for mass / soft, the walk for active_idx / a_old.
    cudaStream_t cs = nullptr;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};   // buffer allocated, pos, mass + soft, the rest
#define OG_H_TRY(expr) OG_CUDA_TRY(expr, { rc = OG_ERR_CUDA; goto done; })
    OG_H_TRY(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    for (int i = 0; i < 4; ++i) OG_H_TRY(cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming));
    OG_H_TRY(cudaEventRecord(ev[0], st));
    OG_H_TRY(cudaStreamWaitEvent(cs, ev[0], 0));
    OG_H_TRY(cudaMemcpyAsync(d + o_pos, pos, n * 12, cudaMemcpyHostToDevice, cs));
    OG_H_TRY(cudaEventRecord(ev[1], cs));
    OG_H_TRY(cudaMemcpyAsync(d + o_m, mass, n * 4, cudaMemcpyHostToDevice, cs));
    OG_H_TRY(cudaMemcpyAsync(d + o_s, soft, n * 4, cudaMemcpyHostToDevice, cs));
    OG_H_TRY(cudaEventRecord(ev[2], cs));
    if (active_idx) OG_H_TRY(cudaMemcpyAsync(d + o_ai, active_idx, na * 4, cudaMemcpyHostToDevice, cs));
    if (a_old) OG_H_TRY(cudaMemcpyAsync(d + o_ao, a_old, na * 4, cudaMemcpyHostToDevice, cs));
    OG_H_TRY(cudaEventRecord(ev[3], cs));
    OG_H_TRY(cudaStreamWaitEvent(st, ev[1], 0));
    {
        og_params p = *params;
        p.workspace = nullptr; p.workspace_bytes = 0;
        t = tree_build_impl((const float *)(d + o_pos), (const float *)(d + o_m), (const float *)(d + o_s), n, box,
                            &p, stream, ev[2]);
    }
    if (t) OG_H_TRY(cudaStreamWaitEvent(st, ev[3], 0));
    if (!t) { rc = OG_ERR_CUDA; goto done; }
    rc = og_shortrange_accel(t, active_idx ? (const uint32_t *)(d + o_ai) : nullptr, n_active,
                             a_old ? (const float *)(d + o_ao) : nullptr, (float *)(d + o_acc),
                             pot_out ? (float *)(d + o_pot) : nullptr, stream);
    if (rc != OG_OK) goto done;
    OG_H_TRY(cudaMemcpyAsync(acc_out, d + o_acc, na * 12, cudaMemcpyDeviceToHost, st));
    if (pot_out) OG_H_TRY(cudaMemcpyAsync(pot_out, d + o_pot, na * 4, cudaMemcpyDeviceToHost, st));
    {
        const int s = og_tree_status(t);  // synchronises
        if (s != OG_OK) rc = s;
    }
#undef OG_H_TRY
done:
    if (cs) cudaStreamSynchronize(cs);   // (on the error paths copies may still be in flight)
    if (t) og_tree_free(t, stream);
    cudaFreeAsync(d, st);
    cudaStreamSynchronize(st);
    for (int i = 0; i < 4; ++i) if (ev[i]) cudaEventDestroy(ev[i]);
    if (cs) cudaStreamDestroy(cs);
    return rc;
}

extern "C" int og_trim(void)
{
    g_err[0] = 0;
    int dev = 0;
    OG_CUDA_TRY(cudaGetDevice(&dev), return OG_ERR_CUDA);
    if (dev < 0 || dev >= 64) return OG_OK;
    cudaMemPool_t pool;
    {
        std::lock_guard<std::mutex> lk(g_pool_mu);
        pool = g_pools[dev];
    }
    if (pool) OG_CUDA_TRY(cudaMemPoolTrimTo(pool, 0), return OG_ERR_CUDA);
    return OG_OK;
}
