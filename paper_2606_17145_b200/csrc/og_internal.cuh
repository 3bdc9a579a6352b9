// og_internal.cuh -- shared declarations of the CUDA path (sm_100a only).
// Nothing here is used by, or taken from, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include "og.h"

#define OG_MAX_LEVEL 21
#define OG_COVER_L5 4681u     // offset of the level-5 cells in og_tree::cover

// Latched device-side status bits (og_tree::d_status[0]).
#define OG_DEV_NODE_OVERFLOW 1u
#define OG_DEV_BAD_POSITION 2u
#define OG_DEV_STACK_OVERFLOW 4u
#define OG_DEV_BAD_INDEX 8u
#define OG_DEV_NGB_OVERFLOW 16u   // og_sph_density: the neighbour candidates of a target do not fit its list

// Counter slots (og_tree::d_counters), see og_stats.
enum { OGC_V_FULL = 0, OGC_V_CULL, OGC_A_IN, OGC_P_IN, OGC_P_SOFT, OGC_P_OUT, OGC_FP64,
       // group-walk diagnostics: nodes per class, particles per class, batches
       OGC_CL_DROP, OGC_CL_OPEN, OGC_CL_ACCEPT, OGC_CL_GENERIC, OGC_PT_DROP, OGC_PT_SHIFT, OGC_PT_WRAP, OGC_BATCHES,
       OGC_SPILLS, OGC_N };

// Packed node record read by the walk: 4 x float4 + uint2.
//   com  = (s_x, s_y, s_z, M)                 R9: fp32 rounding of the fp64 upward pass
//   cell = (c_x, c_y, c_z, l)                 geometric centre and side
//   lo   = (lo_x, lo_y, lo_z, h_max)          tight AABB (R10: culling only)
//   hi   = (hi_x, hi_y, hi_z, 0)
//   info = (start, count | leaf bit)          leaf: first slot / particle count
//                                             internal: first child / n_child
#define OG_LEAF_BIT 0x80000000u

struct og_tree {
    // problem
    uint64_t n;
    float box;
    og_params prm;
    uint32_t max_nodes;
    int device;
    int sm_count;
    // memory
    void *arena;            // base of the device allocation (or caller workspace)
    size_t arena_bytes;
    int owns_arena;
    // sorted particles
    uint64_t *keys;         // sorted keys
    uint32_t *perm;
    uint32_t *inv_perm;
    float4 *spos;           // (x, y, z, m)
    float *sh;
    // canonical topology
    uint8_t *node_level;
    uint32_t *node_first;
    uint32_t *node_count;
    uint32_t *node_first_child;
    uint8_t *node_nchild;
    // packed records
    float4 *node_com;
    float4 *node_cell;
    float4 *node_lo;
    float4 *node_hi;
    uint2 *node_info;
    // packed walk records (read by the group walk; written by the last phase of k_upward):
    //   n0 = node_com (copied, so that the three quadwords of a node are contiguous)
    //   n1 = (R, ng, first, meta): R = largest distance from s to a corner of the AABB (rounded up),
    //        ng = max(h_max, largest |x - s| over the 0.6 l guard box of R15) (rounded up), first = first
    //        child / first slot, meta = level << 27 | leaf << 26 | (n_child or particle count)
    //   n2 = (c_x, c_y, c_z, h_max)
    uint4 *node_rec;           // [3 n_nodes]: n0, n1, n2 of node j at 3 j, 3 j + 1, 3 j + 2 (48 contiguous bytes)
    // small device state
    uint32_t *d_level_start;   // [24]: start index per level, [22] = n_nodes, [23] = max level
    uint32_t *d_status;        // [16]: [0] latched status bits, [1] walk work counter, [2] sparse-active-list flag, [3] SPH ticket
    uint32_t *cover;           // [37449] cell (level 0..5, Morton index; level l starts at (8^l - 1) / 7) -> the node that covers it
                               // (of that level, or the leaf above; 0xffffffff: empty cell): entry points of the walks
    uint32_t *walk_cost;       // [n] OG_COUNT only: interactions evaluated per target of the last walk, caller's order
    unsigned long long *d_counters;  // [OGC_N]
    // walk scratch (spill stacks), allocated lazily
    void *walk_spill;
    size_t walk_spill_bytes;
    uint32_t walk_spill_cap;   // ranges per warp in the slab
    // stream ordering (og.h "Streams and a tree"): built = end of og_tree_build on build_stream; walked = end of
    // the last og_shortrange_accel (recorded on its stream), waited for by the next walk and by og_tree_free
    cudaStream_t build_stream;
    cudaEvent_t ev_built;
    cudaEvent_t ev_walked;
    mutable bool walked;
    mutable int walk_kind;     // last og_shortrange_accel[_ext]: 0 none yet, 1 identity list / external targets (32 per warp),
                               // 2 explicit active list (d_status[2] holds the choice: 0 -> 32, 1 -> 8 targets per warp)
    mutable bool cover_built;  // the cell table has been written (by the first og_sph_density on this tree)
    mutable int64_t n_nodes_host;   // -1 until read back
    mutable uint32_t max_level_host;
};

// ---- error plumbing (api.cu) ----
void og_set_error(const char *fmt, ...);
#define OG_CUDA_TRY(expr, onfail)                                                        \
    do {                                                                                 \
        cudaError_t _e = (expr);                                                         \
        if (_e != cudaSuccess) {                                                         \
            og_set_error("%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e),         \
                         __FILE__, __LINE__);                                            \
            onfail;                                                                      \
        }                                                                                \
    } while (0)

// SMs of the current device (cached per device; 148 when none is visible): grid-stride kernels size their grids by it
int ogk_sm_count(void);

// ---- kernel launchers (one per row of SURVEY.md Sec. 8(a)) ----
// a1
cudaError_t ogk_keys(const float *pos, uint64_t n, float box, uint64_t *keys, uint32_t *idx,
                     uint32_t *d_status, bool validate, cudaStream_t st);
// a2
size_t ogk_sort_scratch_bytes(uint64_t n);
cudaError_t ogk_radix_sort(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt,
                           uint64_t n, int begin_bit, int end_bit, void *scratch, int *in_alt,
                           cudaStream_t st);
// a2 with the scratch in a fixed array of the library image (og_radix_sort_pairs_noalloc)
size_t ogk_sort_noalloc_max_n(void);
cudaError_t ogk_radix_sort_noalloc(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt, uint64_t n,
                                   int begin_bit, int end_bit, int *in_alt, cudaStream_t st);
// a3
cudaError_t ogk_gather(const float *pos, const float *mass, const float *soft,
                       const uint32_t *perm, uint64_t n, float4 *spos, float *sh,
                       uint32_t *inv_perm, cudaStream_t st);
// a4 + a5
size_t ogk_octree_scratch_bytes(uint32_t max_nodes);
cudaError_t ogk_octree_upward(og_tree *t, void *scratch, cudaStream_t st);
cudaError_t ogk_cover(const og_tree *t, cudaStream_t st);
// a6 + a7
cudaError_t ogk_walk(const og_tree *t, const uint32_t *tgt_slot, const uint32_t *tgt_out,
                     uint64_t n_active, const float *a_old, float *acc_out, float *pot_out,
                     cudaStream_t st, const float4 *ext = nullptr, const uint32_t *ext_sparse = nullptr);
size_t ogk_walk_spill_bytes(int sm_count, uint32_t spill_entries);
uint32_t ogk_walk_spill_entries(const og_params *p);
// f3
cudaError_t ogk_sph_density(const og_tree *t, const uint32_t *active_idx, uint64_t n_active, float n_des, float tol_n,
                            const float *h_guess, float *h_out, float *rho_out, float *nn_out, cudaStream_t st);
// f4 (let.cu)
cudaError_t ogk_ext_gather(const float *tpos, const float *tsoft, const uint32_t *order, uint64_t n_t, float4 *ext,
                           cudaStream_t st);
cudaError_t ogk_cell_hist(const uint64_t *keys, uint64_t n, uint32_t *hist, cudaStream_t st);
cudaError_t ogk_owner(const uint64_t *keys, uint64_t n, const uint32_t *S, uint32_t R, uint32_t *owner, cudaStream_t st);
cudaError_t ogk_let_mark(const float *tpos, uint64_t n_t, const float *boxes, uint32_t nb, float r_cut, float L,
                         uint8_t *flag, cudaStream_t st);
size_t ogk_flag_scratch_bytes(uint64_t n);
cudaError_t ogk_flag_compact(const uint8_t *flag, uint64_t n, uint32_t *out, uint32_t *scratch, uint32_t **total_dev,
                             cudaStream_t st);
cudaError_t ogk_let_accumulate(float *acc, float *pot, const uint32_t *idx, const float *pacc, const float *ppot, uint64_t m,
                               uint64_t n, cudaStream_t st);
// helpers for the active subset
cudaError_t ogk_active_slots(const uint32_t *active_idx, const uint32_t *inv_perm, uint64_t n,
                             uint64_t n_active, uint64_t *keys, uint32_t *vals, uint32_t *d_status,
                             cudaStream_t st);
cudaError_t ogk_unpack_slots(const uint64_t *keys, uint64_t n_active, uint32_t *slots, uint32_t sparse_div,
                             uint32_t *sparse, cudaStream_t st);
cudaError_t ogk_ext_sparse(const uint64_t *tkeys_sorted, uint64_t n_t, const uint64_t *tree_keys, uint64_t n, uint32_t sparse_div,
                           uint32_t *sparse, cudaStream_t st);
#define OG_SPARSE_DIV 16u  // an active list that fills fewer than 1 / 16 of its Morton range counts as sparse (8 targets per warp)
