// keys.cu -- rows a1 (Morton keys) and a3 (gather to sorted SoA) of SURVEY.md Sec. 8(a).
//
// a1 (C1, R1, R2): S = fl32(2^21 / L); per axis t = x *_{fp32,RN} S (one IEEE multiply, no
// FMA contraction -> __fmul_rn); clamp to [0, 2^21 - 1]; truncate; bit b of q_x -> key bit
// 3b+2, q_y -> 3b+1, q_z -> 3b.  HBM-bound: 12 B read + 12 B written per particle.
//
// a3: spos[s] = (pos[perm[s]], mass[perm[s]]), sh[s] = fl32(2.8 * eps[perm[s]]) (R9),
// inv_perm[perm[s]] = s.  Random 20 B gathers, 24 B coalesced writes per particle.
#include "og_internal.cuh"

__device__ __forceinline__ uint64_t og_spread3(uint32_t v)
{
    uint64_t x = v & 0x1fffffu;
    x = (x | (x << 32)) & 0x001f00000000ffffull;
    x = (x | (x << 16)) & 0x001f0000ff0000ffull;
    x = (x | (x << 8)) & 0x100f00f00f00f00full;
    x = (x | (x << 4)) & 0x10c30c30c30c30c3ull;
    x = (x | (x << 2)) & 0x1249249249249249ull;
    return x;
}

__device__ __forceinline__ uint32_t og_quantise(float x, float S)
{
    float t = __fmul_rn(x, S);
    if (!(t >= 0.0f)) t = 0.0f;
    if (t > 2097151.0f) t = 2097151.0f;
    return (uint32_t)t;  // truncation (cvt.rzi)
}

__device__ __forceinline__ uint64_t og_key3(float x, float y, float z, float S)
{
    return (og_spread3(og_quantise(x, S)) << 2) | (og_spread3(og_quantise(y, S)) << 1) |
           og_spread3(og_quantise(z, S));
}

// 4 particles per thread: 3 x LDG.128 in, 2 x STG.128 (keys) + 1 x STG.128 (idx) out.
__global__ void __launch_bounds__(256)
k_keys(const float *__restrict__ pos, uint64_t n, float S, float box, uint64_t *__restrict__ keys,
       uint32_t *__restrict__ idx, uint32_t *d_status, int validate, int vec)
{
    const uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;  // quad index
    const uint64_t i0 = q * 4;
    if (i0 >= n) return;
    bool bad = false;
    if (vec && i0 + 4 <= n) {
        const float4 *p4 = reinterpret_cast<const float4 *>(pos) + q * 3;
        const float4 a = __ldg(p4), b = __ldg(p4 + 1), c = __ldg(p4 + 2);
        const float xs[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
        uint64_t k[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            k[j] = og_key3(xs[3 * j], xs[3 * j + 1], xs[3 * j + 2], S);
            if (validate)
#pragma unroll
                for (int d = 0; d < 3; ++d) bad |= !(xs[3 * j + d] >= 0.0f && xs[3 * j + d] < box);
        }
        ulonglong2 *k2 = reinterpret_cast<ulonglong2 *>(keys + i0);
        k2[0] = make_ulonglong2(k[0], k[1]);
        k2[1] = make_ulonglong2(k[2], k[3]);
        if (idx)
            *reinterpret_cast<uint4 *>(idx + i0) =
                make_uint4((uint32_t)i0, (uint32_t)i0 + 1, (uint32_t)i0 + 2, (uint32_t)i0 + 3);
    } else {
        const uint64_t i1 = (i0 + 4 < n) ? i0 + 4 : n;
        for (uint64_t i = i0; i < i1; ++i) {
            const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
            keys[i] = og_key3(x, y, z, S);
            if (idx) idx[i] = (uint32_t)i;
            if (validate)
                bad |= !(x >= 0.0f && x < box && y >= 0.0f && y < box && z >= 0.0f && z < box);
        }
    }
    if (validate && bad) atomicOr(d_status, OG_DEV_BAD_POSITION);
}

cudaError_t ogk_keys(const float *pos, uint64_t n, float box, uint64_t *keys, uint32_t *idx,
                     uint32_t *d_status, bool validate, cudaStream_t st)
{
    const float S = (float)(2097152.0 / (double)box);
    const uint64_t quads = (n + 3) / 4;
    const unsigned grid = (unsigned)((quads + 255) / 256);
    // vector path needs 16-byte aligned buffers (torch allocations are)
    const int vec = (((uintptr_t)pos | (uintptr_t)keys | (uintptr_t)idx) & 15u) == 0;
    k_keys<<<grid, 256, 0, st>>>(pos, n, S, box, keys, idx, d_status, validate ? 1 : 0, vec);
    return cudaGetLastError();
}

// ---- a3 gather --------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_gather(const float *__restrict__ pos, const float *__restrict__ mass, const float *__restrict__ soft,
         const uint32_t *__restrict__ perm, uint64_t n, float4 *__restrict__ spos,
         float *__restrict__ sh, uint32_t *__restrict__ inv_perm)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint32_t i = perm[s];
    const float x = __ldg(pos + 3 * (uint64_t)i), y = __ldg(pos + 3 * (uint64_t)i + 1),
                z = __ldg(pos + 3 * (uint64_t)i + 2);
    spos[s] = make_float4(x, y, z, __ldg(mass + i));
    // R9: h = fl32(2.8 * eps), product formed in fp64
    sh[s] = __double2float_rn(__dmul_rn(2.8, (double)__ldg(soft + i)));
    inv_perm[i] = (uint32_t)s;
}

cudaError_t ogk_gather(const float *pos, const float *mass, const float *soft, const uint32_t *perm,
                       uint64_t n, float4 *spos, float *sh, uint32_t *inv_perm, cudaStream_t st)
{
    const unsigned grid = (unsigned)((n + 255) / 256);
    k_gather<<<grid, 256, 0, st>>>(pos, mass, soft, perm, n, spos, sh, inv_perm);
    return cudaGetLastError();
}

// ---- active subset helpers --------------------------------------------------------------
// key = sorted slot of the target (so that a stable sort by key groups spatial neighbours),
// val = position in the caller's active list.
__global__ void __launch_bounds__(256)
k_active_slots(const uint32_t *__restrict__ active_idx, const uint32_t *__restrict__ inv_perm, uint64_t n,
               uint64_t n_active, uint64_t *__restrict__ keys, uint32_t *__restrict__ vals,
               uint32_t *d_status)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_active) return;
    uint32_t i = __ldg(active_idx + t);
    if (i >= n) {  // latch and clamp: never read out of bounds
        atomicOr(d_status, OG_DEV_BAD_INDEX);
        i = (uint32_t)(n - 1);
    }
    keys[t] = (uint64_t)__ldg(inv_perm + i);
    vals[t] = (uint32_t)t;
}

// Also decides (on the device: no host round trip) how the walk groups these targets: `*sparse` = 1 if the active
// targets fill fewer than 1 / sparse_div of the sorted slots between the first and the last of them (the walk then
// takes 8 targets per warp), else 0.  The density is that of the Morton range the list covers, so a contiguous range
// of a larger set (one rank's share, a spatial region) is walked like the full set.
__global__ void __launch_bounds__(256)
k_unpack_slots(const uint64_t *__restrict__ keys, uint64_t n_active, uint32_t *__restrict__ slots, uint32_t sparse_div,
               uint32_t *__restrict__ sparse)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_active) return;
    slots[t] = (uint32_t)keys[t];
    if (t == 0) {
        const uint64_t span = keys[n_active - 1] - keys[0] + 1;
        *sparse = (n_active * (uint64_t)sparse_div < span) ? 1u : 0u;
    }
}

// The same decision for targets that are not particles of the tree (og_shortrange_accel_ext): their density is
// measured against the tree they walk -- `*sparse` = 1 if the n_t targets are fewer than 1 / sparse_div of the tree's
// particles whose keys lie between the first and the last target key (two binary searches over the tree's sorted keys).
__global__ void k_ext_sparse(const uint64_t *__restrict__ tkeys, uint64_t n_t, const uint64_t *__restrict__ keys, uint64_t n,
                             uint32_t sparse_div, uint32_t *__restrict__ sparse)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    const uint64_t k_first = tkeys[0], k_last = tkeys[n_t - 1];
    uint64_t lo = 0, hi = n;                       // first tree slot with key >= k_first
    while (lo < hi) { const uint64_t m = (lo + hi) >> 1; if (keys[m] < k_first) lo = m + 1; else hi = m; }
    const uint64_t first = lo;
    lo = first; hi = n;                            // first tree slot with key > k_last
    while (lo < hi) { const uint64_t m = (lo + hi) >> 1; if (keys[m] <= k_last) lo = m + 1; else hi = m; }
    *sparse = (sparse_div == 0u || n_t * (uint64_t)sparse_div < lo - first) ? 1u : 0u;   // 0: forced (OG_WALK_G8)
}

cudaError_t ogk_ext_sparse(const uint64_t *tkeys_sorted, uint64_t n_t, const uint64_t *tree_keys, uint64_t n, uint32_t sparse_div,
                           uint32_t *sparse, cudaStream_t st)
{
    k_ext_sparse<<<1, 32, 0, st>>>(tkeys_sorted, n_t, tree_keys, n, sparse_div, sparse);
    return cudaGetLastError();
}

cudaError_t ogk_active_slots(const uint32_t *active_idx, const uint32_t *inv_perm, uint64_t n,
                             uint64_t n_active, uint64_t *keys, uint32_t *vals, uint32_t *d_status,
                             cudaStream_t st)
{
    const unsigned grid = (unsigned)((n_active + 255) / 256);
    k_active_slots<<<grid, 256, 0, st>>>(active_idx, inv_perm, n, n_active, keys, vals, d_status);
    return cudaGetLastError();
}

cudaError_t ogk_unpack_slots(const uint64_t *keys, uint64_t n_active, uint32_t *slots, uint32_t sparse_div,
                             uint32_t *sparse, cudaStream_t st)
{
    const unsigned grid = (unsigned)((n_active + 255) / 256);
    k_unpack_slots<<<grid, 256, 0, st>>>(keys, n_active, slots, sparse_div, sparse);
    return cudaGetLastError();
}
