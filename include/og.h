/*
 * og.h -- C ABI of libogtree.so: B200-native TreePM short-range gravity
 *         (tree construction + Barnes-Hut tree walk), single GPU, sm_100a.
 *
 * What the calls compute.  The paper states the problem only qualitatively: "for each
 * dynamically active particle, a tree walk is performed to compute the forces acting on
 * it" (Sec. 2), Barnes & Hut gravity opened by a criterion,
 * TreePM with the long-range part done elsewhere.  It prints no formula;
 * the arithmetic is the reading fixed in SURVEY.md Sec. 8.3 (C0..C7, R1..R30) and listed
 * in DESIGN.md Sec. 3.  Each entry point below cites the item it implements.
 *
 * Conventions (all entry points)
 *  - Every pointer says DEVICE or HOST.  Device pointers must be valid on the current
 *    CUDA device; inputs are borrowed and only read; outputs are caller-owned.
 *  - `stream` is a cudaStream_t passed as an opaque pointer (NULL = legacy default
 *    stream).  Calls only ENQUEUE work on `stream` and return; the library never calls
 *    cudaDeviceSynchronize.  Inputs must stay valid until the stream has passed the call.
 *  - Streams and a tree: og_shortrange_accel may be called on any stream.  The library orders it
 *    after the tree's build and after the previous walk on the same tree (events; no host
 *    synchronisation), because a walk uses scratch state owned by the tree (group counter,
 *    traversal-stack slabs, OG_COUNT counters): walks on ONE tree therefore run one after the
 *    other even when issued on different streams; walks on different trees overlap freely.
 *    og_tree_free orders the release after the last walk.  Calls on one tree from several host
 *    threads at the same time are not supported.
 *  - `int` functions return OG_OK (0) or a negative og_status; og_tree_build returns NULL
 *    on synchronous failure.  og_last_error() holds a thread-local message for the last
 *    failing call.  No C++ exception crosses the ABI; nothing aborts.
 *  - Conditions detected on the device (node capacity exceeded, walk stack overflow,
 *    position outside [0, box) when OG_VALIDATE_POS) are latched in the tree and returned
 *    by og_tree_status().
 *  - There is no CPU fallback: without a CUDA device every compute call fails with
 *    OG_ERR_CUDA.
 */
#ifndef OG_H
#define OG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct og_tree og_tree;         /* opaque; device-resident; owned by the library */
typedef struct CUstream_st *og_stream;  /* == cudaStream_t */

typedef enum {
    OG_OK = 0,
    OG_ERR_INVALID_ARG = -1,
    OG_ERR_OUT_OF_MEMORY = -2,
    OG_ERR_NODE_OVERFLOW = -3,   /* canonical octree needs more than max_nodes nodes (R6)  */
    OG_ERR_CUDA = -4,
    OG_ERR_BAD_POSITION = -5,    /* OG_VALIDATE_POS: some x not in [0, box)                */
    OG_ERR_STACK_OVERFLOW = -6,  /* walk traversal stack exceeded its spill capacity       */
    OG_ERR_NGB_OVERFLOW = -7     /* og_sph_density: no root / neighbour stack exceeded      */
} og_status;

/* og_params.flags */
#define OG_PERIODIC 1u      /* required in this build (nearest-image distances, R13)      */
#define OG_VALIDATE_POS 2u  /* device-side check 0 <= x < box during key generation       */
#define OG_COUNT 4u         /* walk also accumulates interaction counters (og_stats)      */
#define OG_WALK_G32 8u      /* og_shortrange_accel with an active list: always 32 targets per warp ...       */
#define OG_WALK_G8 16u      /* ... always 8 targets per warp (neither bit: chosen per call from the list, see  */
                            /* og_shortrange_accel; both bits: invalid)                                         */

typedef struct {
    uint32_t struct_size;   /* = sizeof(og_params); ABI guard                              */
    uint32_t flags;         /* OG_PERIODIC | ...                                           */
    float G;                /* gravitational constant (R12; 1 in all configs)              */
    float r_s;              /* force-split scale, same units as box                        */
    float rcut_over_rs;     /* 4.5 (BASELINE.json north_star); must be <= 5 (range of the  */
                            /* split-factor polynomial)                */
    float alpha;            /* relative opening criterion (R14), used iff a_old != NULL    */
    float theta;            /* geometric criterion (R22), used iff a_old == NULL           */
    uint32_t leaf_max;      /* bucket size of the canonical octree (R7), default 8         */
    uint32_t max_nodes;     /* node capacity; 0 -> default (R6)                            */
    /* additions over SURVEY.md Sec. 8.2 (capacity knobs of the walk's traversal stack; 0 -> default): */
    uint32_t walk_stack_entries;  /* pending node ranges a warp keeps in shared memory before it spills the
                                     older half to its global slab (default and maximum 256)               */
    uint32_t walk_spill_entries;  /* capacity of that global slab per warp, in ranges (default 3072);
                                     exceeding it latches OG_ERR_STACK_OVERFLOW                            */
    void *workspace;        /* DEVICE scratch supplied by the caller, or NULL -> the       */
    size_t workspace_bytes; /* library allocates with cudaMallocAsync on `stream`          */
} og_params;

typedef struct {
    uint64_t n;             /* particles                                                   */
    uint64_t n_nodes;       /* nodes of the canonical octree                               */
    uint32_t max_level;     /* deepest level holding a node (root = 0)                     */
    uint32_t walk_targets_per_warp;  /* grouping the last og_shortrange_accel on this tree used: 32 or 8 (0: no walk yet) */
    /* sums over the targets of the last og_shortrange_accel with OG_COUNT (else 0):       */
    uint64_t V_full;        /* visits that passed the cull                                 */
    uint64_t V_cull;        /* visits removed by the cutoff-box test                       */
    uint64_t A_in;          /* accepted nodes with r < r_cut                               */
    uint64_t P_in;          /* particle pairs with r < r_cut                               */
    uint64_t P_soft;        /* ... of which r < h                                          */
    uint64_t P_out;         /* particle pairs evaluated with r >= r_cut                    */
    uint64_t fp64_rechecks; /* decisions re-evaluated in fp64           */
    /* group-walk diagnostics (OG_COUNT): nodes classified at group level as dropped / opened by
     * all / accepted by all / undecided; particles dropped / staged shifted / staged for per-lane
     * wrap; node batches popped                                                              */
    uint64_t cl_drop, cl_open, cl_accept, cl_generic, pt_drop, pt_shift, pt_wrap, batches;
    uint64_t stack_spills;  /* times a warp moved half of its traversal stack to its global slab        */
} og_stats;

/* og_tree_get field selectors.  Pointers are DEVICE pointers into the tree, valid until
 * og_tree_free; `count` is the number of ELEMENTS of the stated type.                    */
typedef enum {
    OG_F_KEYS_SORTED = 0,   /* u64 [n]     Morton keys in sorted order (C1, C2)            */
    OG_F_PERM = 1,          /* u32 [n]     perm[s] = original index of sorted slot s (C2)  */
    OG_F_INV_PERM = 2,      /* u32 [n]     inverse permutation                             */
    OG_F_SPOS = 3,          /* f32 [n][4]  sorted (x, y, z, m)                             */
    OG_F_SH = 4,            /* f32 [n]     sorted h = fl32(2.8 eps) (R9)                   */
    OG_F_NODE_LEVEL = 5,    /* u8  [n_nodes]                                               */
    OG_F_NODE_FIRST = 6,    /* u32 [n_nodes] first sorted slot                             */
    OG_F_NODE_COUNT = 7,    /* u32 [n_nodes] particle count                                */
    OG_F_NODE_FIRST_CHILD = 8, /* u32 [n_nodes] (0 for leaves)                             */
    OG_F_NODE_NCHILD = 9,   /* u8  [n_nodes] 0 for leaves, else 1..8                       */
    OG_F_NODE_COM = 10,     /* f32 [n_nodes][4]  (s_x, s_y, s_z, M)        fp32 record R9  */
    OG_F_NODE_CELL = 11,    /* f32 [n_nodes][4]  (c_x, c_y, c_z, l)                        */
    OG_F_NODE_LO = 12,      /* f32 [n_nodes][4]  (lo_x, lo_y, lo_z, h_max)  tight AABB     */
    OG_F_NODE_HI = 13,      /* f32 [n_nodes][4]  (hi_x, hi_y, hi_z, unused)                */
    OG_F_LEVEL_START = 14,  /* u32 [23]    node index where each level starts (BFS)        */
    OG_F_WALK_COST = 15     /* u32 [n]     OG_COUNT trees only: interactions (accepted nodes + particle pairs)
                               evaluated for each target of the LAST walk, in the caller's active order (the first
                               n_active entries); the per-target work figure a host code balances its next step by
                               (not written by a walk of more than n targets or of external targets)              */
} og_field;

/* Bytes of DEVICE workspace og_tree_build needs for n particles (0 on invalid input).    */
size_t og_tree_workspace_bytes(uint64_t n, const og_params *params);

/*
 * Rows a1..a5 of SURVEY.md Sec. 8: Morton keys (C1) -> stable LSD radix sort with index
 * tie-break (C2) -> gather to sorted float4 (x,y,z,m) + h -> canonical sparse octree (C3)
 * -> upward pass (C4: M, centre of mass, cell centre/side, tight AABB, h_max; fp64
 * accumulation in slot / child order, stored fp32).
 *   pos   DEVICE f32 [n][3], 0 <= x < box       (borrowed)
 *   mass  DEVICE f32 [n]                        (borrowed)
 *   soft  DEVICE f32 [n]  Plummer-equivalent eps; h = 2.8 eps (borrowed)
 *   n     1 <= n < 2^31;   box > 0;   requires rcut_over_rs * r_s < box / 2 (R13)
 * Returns a tree that owns sorted copies (inputs may be released once the stream has
 * passed the call), or NULL (bad struct_size / sizes / pointers, r_cut >= box/2,
 * leaf_max == 0, allocation failure).  Cite: PAPER.md:88, :322 (the reference builds its
 * tree on the CPU and re-uploads it; here it is built on the device).
 */
og_tree *og_tree_build(const float *pos, const float *mass, const float *soft, uint64_t n,
                       float box, const og_params *params, og_stream stream);

/*
 * Rows a6..a7: short-range tree walk (C5, C6) for the active targets and scatter of the
 * results in the caller's order.  PAPER.md:59 ("for each dynamically active particle a
 * tree walk"), :74 (per-node interaction, opening criterion).
 *   active_idx DEVICE u32 [n_active] ORIGINAL particle indices, any order, no duplicates
 *              required; NULL -> all n particles in identity order (n_active must be n)
 *   a_old      DEVICE f32 [n_active] |a| of the previous step in active order (R23);
 *              NULL -> geometric criterion l^2 > theta^2 r^2 (R22)
 *   acc_out    DEVICE f32 [n_active][3], overwritten (n_active == 0: nothing is done, OG_OK)
 *   pot_out    DEVICE f32 [n_active], overwritten, or NULL
 * Returns OG_OK or a negative og_status; conditions detected on the device (bad index, traversal stack
 * capacity) are latched and reported by og_tree_status().  n_active == 0 is a no-op.  Implementation note:
 * the targets are taken in Morton order, 32 per warp; an active list that fills fewer than 1 / 16 of the Morton
 * range it covers is walked with 8 targets per warp (4 lanes per target), decided on the device from THAT list's
 * first and last target (OG_WALK_G32 / OG_WALK_G8 in og_params.flags fix the grouping instead; og_stats.
 * walk_targets_per_warp tells which one the last call used).  Results do not depend on the launch order
 * (bit-reproducible run to run), and a call on a sub-list that covers whole warps of the full list's order (a
 * multiple of 32 consecutive targets of the sorted active list) returns the same bits as the full call does for those
 * targets PROVIDED both calls use the same grouping: the partial sums of a target are added in an order that depends
 * on it.  The automatic choice does not guarantee that (a list made of two distant clumps counts as sparse, each clump
 * alone as dense), so a caller who splits a list over several calls or ranks builds the sub-list trees with the flag
 * that matches the full call's og_stats.walk_targets_per_warp (bench.py --scaling strong does).
 */
int og_shortrange_accel(const og_tree *tree, const uint32_t *active_idx, uint64_t n_active,
                        const float *a_old, float *acc_out, float *pot_out, og_stream stream);

/* DEVICE pointer + element count of one tree array (og_field).  Synchronises the tree's
 * build stream once (to learn n_nodes).                                                   */
int og_tree_get(const og_tree *tree, int field, const void **dev_ptr, uint64_t *count);

/* Synchronises the stream(s) the tree was used on; returns the latched status.           */
int og_tree_status(const og_tree *tree);

/* Synchronises like og_tree_status and fills *stats.                                     */
int og_tree_stats(const og_tree *tree, og_stats *stats);

/* Releases the tree (stream-ordered on `stream`).  NULL is ignored.                      */
void og_tree_free(og_tree *tree, og_stream stream);

/* Thread-local message of the last failing call ("" if none).                            */
const char *og_last_error(void);

/* ---- single rows, exposed for parity tests and per-kernel measurement ---------------- */

/* Row a1 (C1, R1, R2): key[i] = Morton(quantise(pos[i])), idx[i] = i.
 *   pos DEVICE f32 [n][3];  keys DEVICE u64 [n];  idx DEVICE u32 [n] or NULL.            */
int og_morton_keys(const float *pos, uint64_t n, float box, uint64_t *keys, uint32_t *idx,
                   og_stream stream);

/* Bytes of DEVICE scratch og_radix_sort_pairs needs for n pairs.                          */
size_t og_radix_sort_scratch_bytes(uint64_t n);

/* Row a2 (C2, R3): stable LSD radix sort of (key, val) pairs by key bits
 * [begin_bit, end_bit), 8 bits per pass.  keys/vals are DEVICE ping-pong buffers of n
 * elements each; on return *result_in_alt = 1 if the sorted data is in (keys_alt,
 * vals_alt), else 0 (it is in keys/vals).  Stability gives the index tie-break.           */
int og_radix_sort_pairs(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt,
                        uint64_t n, int begin_bit, int end_bit, void *scratch,
                        size_t scratch_bytes, int *result_in_alt, og_stream stream);

/*
 * Row a2 for callers that cannot allocate device memory: the same sort, same result bit for bit, but without a
 * scratch argument and without a single allocation inside the library (no cudaMalloc / cudaFree / cudaMallocAsync,
 * no library routine that allocates).  Who needs this: a simulation code that claims the whole device for its own
 * arena at start-up and has nothing left to allocate from; a step that runs where an allocation would stall or
 * deadlock (another thread holds the allocator, or the allocation would synchronise the device in the middle of
 * overlapped work); a component that is only lent buffers and owns no allocator.  Such a caller can still pass the four
 * ping-pong buffers -- those are its inputs and outputs -- but not a scratch buffer sized per call.
 *   The scratch (digit histograms, tile tickets and look-back words of the one-sweep passes) lives in a fixed array
 * compiled into the library: every GPU on which libogtree.so is loaded carries it (about 4 MiB) until the process
 * exits, whether or not this call is ever used.  That fixes the limit: n <= OG_SORT_NOALLOC_MAX_N.  A larger n is
 * refused with OG_ERR_INVALID_ARG and a message naming the limit; nothing is enqueued.  Use og_radix_sort_pairs then.
 *   keys / vals / keys_alt / vals_alt, begin_bit, end_bit, result_in_alt, stream: exactly as og_radix_sort_pairs.
 *   First call on a device: the library looks up the array's device address (cudaGetSymbolAddress, with the caller's
 * current device) and remembers it per device.  The runtime may load the library's device code at that moment, so
 * make the first call on each device during set-up, before any stream capture begins.
 *   Sharing: all calls on one device use the same array.  Each call zeroes what it needs on `stream` before its
 * kernels run, so a call never depends on what an earlier one left there.  Calls that can be in flight on the GPU at
 * the same time (two streams, two host threads) race on the array: order them (one stream, or events).
 */
#define OG_SORT_NOALLOC_MAX_N 1048576u   /* 2^20 pairs */
int og_radix_sort_pairs_noalloc(uint64_t *keys, uint32_t *vals, uint64_t *keys_alt, uint32_t *vals_alt, uint64_t n,
                                int begin_bit, int end_bit, int *result_in_alt, og_stream stream);

/*
 * End-to-end convenience with HOST buffers (bench.py's `e2e` leg): copies pos/mass/soft
 * (and active_idx, a_old if given) to the device, runs og_tree_build + og_shortrange_accel,
 * copies acc/pot back, frees everything, and synchronises `stream` before returning.
 * All pointers HOST (pinned memory recommended); semantics as the two calls above.
 */
int og_shortrange_accel_host(const float *pos, const float *mass, const float *soft, uint64_t n,
                             float box, const og_params *params, const uint32_t *active_idx,
                             uint64_t n_active, const float *a_old, float *acc_out,
                             float *pot_out, og_stream stream);

/* ---- row f1: the PM long-range part of the TreePM force ------------------------------- */

/*
 * PAPER.md:124 keeps the long-range PM force on the CPU (FFTW); here it runs on the device.  Together with
 * og_shortrange_accel (same r_s, same G) it gives the full periodic Newtonian force within the TreePM error.
 * Steps (readings R31..R34; Gadget-2 lineage): CIC assignment of the masses to
 * ng^3 grid points -> DFT (cuFFT, the one library step) -> phi_k = -4 pi G / (V k^2) exp(-k^2 r_s^2) M_k / W(k)^2
 * (W = CIC window, divided out twice; phi_0 = 0) -> inverse DFT -> 4-point finite-difference gradient ->
 * CIC interpolation of acceleration and potential to the targets.  fp32 throughout.
 *
 * og_pm_create: plans and grids for an ng^3 mesh (ng even, 8..2048; Gadget's choice is r_s = 1.25 box / ng).
 *   Device memory: ONE allocation of 28 ng^3 bytes owned by the handle -- 24 ng^3 of grids (mass / potential 4,
 *   spectrum 4, acceleration + potential 16) and one cuFFT work area of 4 ng^3 that the forward and the inverse
 *   transform share (they never run at the same time) -- measured on a B200: 0.47 GB at ng = 256, 3.8 GB at 512,
 *   30 GB at 1024, 101.5 GB at 1536.  ng = 2048 would need 240.6 GB and fails on a 180 GB B200 like any size that does
 *   not fit: NULL, with the byte counts in og_last_error().  Synchronises `stream` once.  NULL on failure.
 * og_pm_longrange: all pointers DEVICE.  pos f32 [n][3] in [0, box), mass f32 [n] (all n particles are sources);
 *   active_idx u32 [n_active] original indices of the targets, or NULL -> all n in identity order
 *   (n_active == n); acc_out f32 [n_active][3], pot_out f32 [n_active] or NULL, overwritten.  Enqueues on `stream`.
 *   The mass assignment uses floating-point atomics: results are reproducible to fp32 rounding, not bit for bit.
 *   An active_idx entry >= n cannot be served: that target gets a zero force and potential, and the mistake is latched
 *   in the handle (the call itself only enqueues and still returns OG_OK).
 * og_pm_status: synchronises `stream` and returns OG_OK, or OG_ERR_INVALID_ARG if any og_pm_longrange on this handle met
 *   an active_idx entry >= n (og_last_error says so); latched until og_pm_free, like og_tree_status for a tree.
 * og_pm_free: synchronises `stream`, releases plans and grids.  NULL is ignored.
 */
typedef struct og_pm og_pm;
og_pm *og_pm_create(uint32_t ng, float box, float r_s, float G, og_stream stream);
int og_pm_longrange(og_pm *pm, const float *pos, const float *mass, uint64_t n, const uint32_t *active_idx,
                    uint64_t n_active, float *acc_out, float *pot_out, og_stream stream);
int og_pm_status(const og_pm *pm, og_stream stream);
void og_pm_free(og_pm *pm, og_stream stream);

/* ---- row f2: the time-step shell around the force calls --------------------------------- */

/*
 * PAPER.md:80 (time bins with few active particles), :82 (all particles are drifted at the onset of a GPU step),
 * :320 (find_sync_point_and_drift).  Gadget-2's individual power-of-two time steps (readings R37..R42, DESIGN.md
 * Sec. 11): one tick = dt_max / 2^bmax; a particle in bin b (u8, 0..bmax) has a step of 2^(bmax - b) ticks and is
 * active at the ticks its step divides.  One step of a host loop is
 *     og_ts_next_tick -> og_ts_drift (all particles, dt = (next - tick) dt_max / 2^bmax) -> og_ts_active_list ->
 *     og_tree_build + og_shortrange_accel (active_idx, a_old gathered by the caller) [+ og_pm_longrange] -> og_ts_kick.
 * All array pointers DEVICE; state arrays (pos, vel, bin, a_old) are caller-owned and updated in place.
 *
 * og_ts_drift       pos f32 [n][3] += vel f32 [n][3] * dt, wrapped into [0, box).  Enqueues.
 * og_ts_next_tick   *next_tick_host (HOST) = the next tick > `tick` at which some particle is active (`tick` must be a
 *                   synchronisation point, 0 at the start).  Synchronises `stream`.
 * og_ts_active_list active_idx u32 [>= n] receives, ascending, the particles active at `tick`; *n_active_host (HOST)
 *                   their number.  Synchronises `stream` (the host sizes the force call with it).
 * og_ts_kick        for the active particles (active_idx NULL -> all n in identity order), with acc f32 [n_active][3]
 *                   in active order and soft f32 [n] (eps): |a| in fp32; wanted bin = smallest b with
 *                   4^b >= dt_max^2 |a| / (2 eta eps) (fp32, fixed operation order); the step shrinks freely and grows
 *                   by one level only at a tick the larger step divides; vel += acc (dt_old + dt_new) / 2 (first != 0:
 *                   start of the integration, wanted bin taken as is, opening half kick dt_new / 2 only); bin and
 *                   a_old f32 [n] (= |a|, the next walk's opening-criterion input) updated.  Enqueues.
 *                   status: DEVICE u32 [1] owned (and zeroed) by the caller, or NULL.  An active_idx entry >= n is
 *                   skipped (no particle is touched for it); with a status word the mistake is also recorded there, the bit
 *                   OG_TS_BAD_INDEX OR-ed in, for the caller to read when it next synchronises -- a corrupted
 *                   active list otherwise shows only as particles that stop moving.
 * scratch: DEVICE, og_ts_scratch_bytes(n) bytes.  bmax <= 40.
 */
size_t og_ts_scratch_bytes(uint64_t n);
int og_ts_drift(float *pos, const float *vel, uint64_t n, float dt, float box, og_stream stream);
int og_ts_next_tick(const uint8_t *bin, uint64_t n, uint64_t tick, uint32_t bmax, uint64_t *next_tick_host,
                    void *scratch, size_t scratch_bytes, og_stream stream);
int og_ts_active_list(const uint8_t *bin, uint64_t n, uint64_t tick, uint32_t bmax, uint32_t *active_idx,
                      uint64_t *n_active_host, void *scratch, size_t scratch_bytes, og_stream stream);
int og_ts_kick(float *vel, uint8_t *bin, float *a_old, const uint32_t *active_idx, uint64_t n, uint64_t n_active,
               const float *acc, const float *soft, float eta, float dt_max, uint32_t bmax, uint64_t tick, int first,
               uint32_t *status, og_stream stream);
#define OG_TS_BAD_INDEX 8u   /* og_ts_kick status bit: some active_idx entry was >= n */

/* ---- row f3: SPH density / smoothing length on the same tree -------------------------------- */

/*
 * PAPER.md:61 ("the SPH density module ... operates as an iterative process, aiming to determine a smoothing length
 * containing a fixed number of neighbours"), :74 ("collects all neighbours within a sphere around the target
 * particle").  Readings R43..R47 (Gadget-2's SPH): cubic-spline kernel with compact
 * support h, W(r, h) = (8 / (pi h^3)) w(r / h); kernel-weighted neighbour number N_i(h) = (4 pi / 3) h^3 sum_j
 * W(r_ij, h) over ALL particles of the tree (j = i included, nearest periodic image); h_i = the root of
 * N_i(h) = n_des; rho_i = sum_j m_j W(r_ij, h_i).  The root is found per target on the neighbours collected by a
 * walk of the tree; the iteration stops at |N - n_des| <= tol_n or at fp32 resolution of h (tol_n = 0: always the
 * latter).  fp32 arithmetic, fixed summation order (bit-reproducible run to run).
 *   tree       a tree from og_tree_build (its particles are the SPH particles; masses from the tree)
 *   active_idx DEVICE u32 [n_active] ORIGINAL indices of the targets, or NULL -> all n in identity order
 *   n_des      32/3 < n_des <= 256 (N(h) -> 32/3 as h -> 0 for an isolated particle)
 *   h_guess    DEVICE f32 [n_active] an estimate of h per target in active order (e.g. the previous step's h; the search
 *              starts at 1.05 x this; any positive value reaches the same root), or NULL -> derived from the tree (the
 *              radius that holds 1.5 n_des at the mean density of the deepest ancestor cell with n_des particles)
 *   h_out      DEVICE f32 [n_active]; rho_out, nn_out (N at the returned h): DEVICE f32 [n_active] or NULL
 * Enqueues on `stream` (ordered after the tree's build and the previous call on the tree; the first call on a tree also
 * writes the tree's table of level-5 cells, where the neighbour walks start).  Neighbour candidates are kept in a per-warp list of 512
 * entries; a target whose root sphere holds more (a void particle whose kernel rim grazes a dense clump) is solved
 * by re-walking the tree for every trial h instead (same result, slower).  A target with more than 3 n_des / 32
 * coincident particles (N(h) > n_des for every h: no root), or whose pending nodes exceed even the fallback's stack,
 * latches OG_ERR_NGB_OVERFLOW (og_tree_status) and gets h = rho = N = 0.
 */
int og_sph_density(const og_tree *tree, const uint32_t *active_idx, uint64_t n_active, float n_des, float tol_n,
                   const float *h_guess, float *h_out, float *rho_out, float *nn_out, og_stream stream);

/* ---- row f4: domain-decomposed short-range force (several GPUs, one tree per domain) ---------- */

/*
 * "the tree walk is executed for particles that reside on the same MPI rank ('primary') ... particles
 * that require tree nodes of other MPI ranks are exported ... ('secondary')", :80 (export buffers).  Readings R49..R53
 * (DESIGN.md Sec. 13): domains are contiguous Morton ranges made of whole level-5 cells (the top 15 key bits); every
 * domain builds the tree of its own particles in the full box (og_tree_build); the force on a target is the sum of the
 * walks of all domains' trees with the target's own (x, h, a_old): og_shortrange_accel on its home tree (self excluded),
 * og_shortrange_accel_ext on the others, where it is an external point.  A target is exported to a domain only if it is
 * within r_cut of one of that domain's top-cell boxes: the tight boxes of its tree's nodes at level 2 when
 * r_cut <= 0.05 box, at level 1 otherwise (and of shallower leaves).  A domain farther away then contributes exactly
 * nothing: nodes at that level and below are culled, and a shallower node that is accepted instead of opened has the
 * target outside its 0.6 l guard box, at least 0.1 l >= r_cut from its centre of mass (R52).  The ranks
 * exchange particles, boxes, targets and results with NCCL all-to-all / all-gather in the host layer
 * (paper_2606_17145_b200/let.py); the calls below are its device-side steps.  All pointers DEVICE unless named HOST.
 *
 * og_shortrange_accel_ext  walk of `tree` for n_t targets that are NOT particles of the tree: tpos f32 [n_t][3] in
 *     [0, box), tsoft f32 [n_t] (eps; h = 2.8 eps as in the tree), a_old f32 [n_t] or NULL (geometric criterion);
 *     acc_out f32 [n_t][3], pot_out f32 [n_t] or NULL, overwritten, in the caller's order.  Nothing is excluded.  The
 *     targets are walked in their own Morton order, 32 per warp, or 8 per warp when they are sparse against this tree:
 *     fewer than 1 / 16 of the tree's particles whose keys lie between the first and the last target's key (decided on
 *     the device; OG_WALK_G32 / OG_WALK_G8 fix it; og_stats.walk_targets_per_warp reports it).  Enqueues; stream rules
 *     as og_shortrange_accel.
 * og_domain_cell_hist      hist u32 [32768] = particles per level-5 cell of pos f32 [n][3] (overwritten).  Enqueues.
 * og_domain_owner          owner u32 [n] = the d with splitters[d] <= cell < splitters[d + 1]; splitters u32
 *     [n_domains + 1], ascending, splitters[0] = 0, splitters[n_domains] = 32768.  Enqueues.
 * og_let_export_list       list_out u32 [>= n_t] receives, ascending, the targets t with tpos[t] within r_cut (nearest
 *     periodic image, point-to-box distance, conservative by a relative 1e-5) of one of the n_boxes <= 1024 boxes
 *     f32 [n_boxes][6] = (lo_x, lo_y, lo_z, hi_x, hi_y, hi_z); *count_host (HOST) their number.  Synchronises `stream`.
 * og_let_accumulate        acc[idx[k]] += part_acc[k], pot[idx[k]] += part_pot[k] for k < m (idx u32 [m], distinct,
 *     < n; pot / part_pot may be NULL).  Enqueues.
 */
int og_shortrange_accel_ext(const og_tree *tree, const float *tpos, const float *tsoft, uint64_t n_t, const float *a_old,
                            float *acc_out, float *pot_out, og_stream stream);
int og_domain_cell_hist(const float *pos, uint64_t n, float box, uint32_t *hist, og_stream stream);
int og_domain_owner(const float *pos, uint64_t n, float box, const uint32_t *splitters, uint32_t n_domains,
                    uint32_t *owner, og_stream stream);
int og_let_export_list(const float *tpos, uint64_t n_t, const float *boxes, uint32_t n_boxes, float r_cut, float box,
                       uint32_t *list_out, uint64_t *count_host, og_stream stream);
int og_let_accumulate(float *acc, float *pot, const uint32_t *idx, const float *part_acc, const float *part_pot,
                      uint64_t m, uint64_t n, og_stream stream);

/* Returns the device memory that freed trees / finished calls left cached in the library's
 * stream-ordered pool of the current device to the driver (the pool keeps arenas for reuse by
 * the next og_tree_build; a host code that needs the memory for something else calls this).
 * Synchronises nothing; memory still in use stays.                                         */
int og_trim(void);

#ifdef __cplusplus
}
#endif
#endif /* OG_H */
