// pm.cu -- row f1 of SURVEY.md Sec. 8: the particle-mesh LONG-RANGE part of the TreePM force on the device.
// the reference keeps the PM on the CPU with FFTW; here every step runs on the GPU:
//
//   k_pm_deposit   R31  CIC assignment of the particle masses to the Ng^3 grid points (fp32 atomics)
//   cuFFT R2C           the DFT itself is the library's
//   k_pm_green     R32  phi_k = -4 pi G / (V k^2) exp(-k^2 r_s^2) M_k / W(k)^2, phi_0 = 0
//   cuFFT C2R           (unnormalised inverse = the sum over k that R33 asks for)
//   k_pm_gradient  R33  4-point finite difference, a = -grad phi, stored with phi as one float4 per grid point
//   k_pm_interp    R34  CIC interpolation of (a, phi) to the targets: 8 x LDG.128 per target
//
// The readings R31..R34 are those of DESIGN.md Sec. 10 (Gadget-2 lineage, Springel 2005, cited PAPER.md:296);
// oracle/pm.py restates them in fp64 NumPy and shares nothing with this file.
#include <cufft.h>
#include <cmath>
#include <new>
#include <vector>
#include "og_internal.cuh"

struct og_pm {
    uint32_t ng;
    float box, r_s, G;
    int device;
    cufftHandle plan_r2c, plan_c2r;
    bool have_plans;
    float *mgrid;          // [ng^3] mass grid, then the potential grid (in place after the inverse transform)
    float2 *kgrid;         // [ng^2 (ng/2 + 1)]
    float4 *fgrid;         // [ng^3] (a_x, a_y, a_z, phi)
    float *k2tab;          // [ng] (2 pi n / L)^2, n in (-ng/2, ng/2]
    float *dctab;          // [ng] 1 / sinc^4(pi n / ng): the CIC window divided out twice, per axis
    size_t arena_bytes;    // grids + tables + the cuFFT work area shared by the two plans
    uint32_t *d_status;    // [1] latched OG_DEV_* bits of the calls on this handle (og_pm_status)
    void *arena;
};

namespace {

__device__ __forceinline__ uint32_t wrap_idx(int i, int ng) { return (uint32_t)(i < 0 ? i + ng : (i >= ng ? i - ng : i)); }

// R31.  One thread per particle.  Particles that are neighbours in the input and share their base grid point (the usual
// case when the caller keeps its particles in space-filling-curve order, as a tree code does: the points of a 2^k mesh
// are octree cells, so such particles are consecutive) are summed inside the warp first -- a segmented scan over the
// runs of equal base points, eight weights at once -- and only the last lane of a run issues the 8 red.global.add.f32;
// unordered input (no runs) skips the scan.
__global__ void __launch_bounds__(256)
k_pm_deposit(const float *__restrict__ pos, const float *__restrict__ mass, uint64_t n, float inv_delta, int ng,
             float *__restrict__ mgrid)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t lane = threadIdx.x & 31u;
    const bool ok = i < n;
    const uint64_t ii = ok ? i : n - 1;
    const float x = __ldg(pos + 3 * ii) * inv_delta, y = __ldg(pos + 3 * ii + 1) * inv_delta, z = __ldg(pos + 3 * ii + 2) * inv_delta;
    const float m = ok ? __ldg(mass + ii) : 0.0f;
    const float fx0 = floorf(x), fy0 = floorf(y), fz0 = floorf(z);
    const float fx = x - fx0, fy = y - fy0, fz = z - fz0;
    int ix = (int)fx0, iy = (int)fy0, iz = (int)fz0;
    ix = ix >= ng ? ix - ng : ix; iy = iy >= ng ? iy - ng : iy; iz = iz >= ng ? iz - ng : iz;   // x * inv_delta may round up to ng
    const uint32_t x0 = wrap_idx(ix, ng), x1 = wrap_idx(ix + 1, ng), y0 = wrap_idx(iy, ng), y1 = wrap_idx(iy + 1, ng),
                   z0 = wrap_idx(iz, ng), z1 = wrap_idx(iz + 1, ng);
    const float wx[2] = {1.0f - fx, fx}, wy[2] = {1.0f - fy, fy}, wz[2] = {1.0f - fz, fz};
    const uint32_t xs[2] = {x0, x1}, ys[2] = {y0, y1}, zs[2] = {z0, z1};
    float v[8];
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int c = 0; c < 2; ++c) v[4 * a + 2 * b + c] = m * wx[a] * wy[b] * wz[c];
    const uint32_t base = ok ? (x0 * (uint32_t)ng + y0) * (uint32_t)ng + z0 : 0xffffffffu;
    const uint32_t prev = __shfl_up_sync(0xffffffffu, base, 1);
    const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0u || base != prev);
    if (heads != 0xffffffffu) {
        // inclusive segmented scan over the runs; my_head = the lane that starts this lane's run
        const uint32_t my_head = 31u - (uint32_t)__clz(heads & (0xffffffffu >> (31u - lane)));
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const bool take = lane >= my_head + (uint32_t)o;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const float up = __shfl_up_sync(0xffffffffu, v[c], o);
                if (take) v[c] += up;
            }
        }
    }
    const bool tail = lane == 31u || ((heads >> (lane + 1u)) & 1u);
    if (ok && tail) {
#pragma unroll
        for (int a = 0; a < 2; ++a)
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int c = 0; c < 2; ++c)
                    atomicAdd(mgrid + ((size_t)xs[a] * ng + ys[b]) * ng + zs[c], v[4 * a + 2 * b + c]);
    }
}

// R32.  One thread per complex element of the half spectrum [ng][ng][ng/2 + 1].
__global__ void __launch_bounds__(256)
k_pm_green(float2 *__restrict__ kg, int ng, const float *__restrict__ k2tab, const float *__restrict__ dctab,
           float pref /* -4 pi G / V */, float rs2)
{
    const int nzh = ng / 2 + 1;
    const size_t total = (size_t)ng * ng * nzh;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const int kz = (int)(e % nzh);
    const size_t r = e / nzh;
    const int ky = (int)(r % ng), kx = (int)(r / ng);
    const float k2 = __ldg(k2tab + kx) + __ldg(k2tab + ky) + __ldg(k2tab + kz);
    float g = 0.0f;
    if (k2 > 0.0f) g = pref / k2 * __expf(-k2 * rs2) * (__ldg(dctab + kx) * __ldg(dctab + ky) * __ldg(dctab + kz));
    float2 v = kg[e];
    v.x *= g; v.y *= g;
    kg[e] = v;
}

// R33.  One thread per grid point; the z line is contiguous.
__global__ void __launch_bounds__(256)
k_pm_gradient(const float *__restrict__ phi, int ng, float c1 /* (4/3) / (2 Delta) */, float c2 /* (1/3) / (4 Delta) */,
              float4 *__restrict__ fg)
{
    const size_t total = (size_t)ng * ng * ng;
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const int z = (int)(e % ng);
    const size_t r = e / ng;
    const int y = (int)(r % ng), x = (int)(r / ng);
    auto at = [&](int xx, int yy, int zz) {
        return __ldg(phi + ((size_t)wrap_idx(xx, ng) * ng + wrap_idx(yy, ng)) * ng + wrap_idx(zz, ng));
    };
    const float ax = -(c1 * (at(x + 1, y, z) - at(x - 1, y, z)) - c2 * (at(x + 2, y, z) - at(x - 2, y, z)));
    const float ay = -(c1 * (at(x, y + 1, z) - at(x, y - 1, z)) - c2 * (at(x, y + 2, z) - at(x, y - 2, z)));
    const float az = -(c1 * (at(x, y, z + 1) - at(x, y, z - 1)) - c2 * (at(x, y, z + 2) - at(x, y, z - 2)));
    fg[e] = make_float4(ax, ay, az, __ldg(phi + e));
}

// R34.  One thread per target.
__global__ void __launch_bounds__(256)
k_pm_interp(const float *__restrict__ pos, const uint32_t *__restrict__ active_idx, uint64_t n, uint64_t n_active,
            float inv_delta, int ng, const float4 *__restrict__ fg, float *__restrict__ acc_out,
            float *__restrict__ pot_out, uint32_t *status)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_active) return;
    uint64_t i = t;
    if (active_idx) {
        i = __ldg(active_idx + t);
        if (i >= n) {
            if (status) atomicOr(status, OG_DEV_BAD_INDEX);
            acc_out[3 * t] = acc_out[3 * t + 1] = acc_out[3 * t + 2] = 0.0f;
            if (pot_out) pot_out[t] = 0.0f;
            return;
        }
    }
    const float x = __ldg(pos + 3 * i) * inv_delta, y = __ldg(pos + 3 * i + 1) * inv_delta, z = __ldg(pos + 3 * i + 2) * inv_delta;
    const float fx0 = floorf(x), fy0 = floorf(y), fz0 = floorf(z);
    const float fx = x - fx0, fy = y - fy0, fz = z - fz0;
    int ix = (int)fx0, iy = (int)fy0, iz = (int)fz0;
    ix = ix >= ng ? ix - ng : ix; iy = iy >= ng ? iy - ng : iy; iz = iz >= ng ? iz - ng : iz;
    const uint32_t xs[2] = {wrap_idx(ix, ng), wrap_idx(ix + 1, ng)}, ys[2] = {wrap_idx(iy, ng), wrap_idx(iy + 1, ng)},
                   zs[2] = {wrap_idx(iz, ng), wrap_idx(iz + 1, ng)};
    const float wx[2] = {1.0f - fx, fx}, wy[2] = {1.0f - fy, fy}, wz[2] = {1.0f - fz, fz};
    float ax = 0.f, ay = 0.f, az = 0.f, ph = 0.f;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const float4 v = __ldg(fg + ((size_t)xs[a] * ng + ys[b]) * ng + zs[c]);
                const float wgt = wx[a] * wy[b] * wz[c];
                ax = fmaf(wgt, v.x, ax); ay = fmaf(wgt, v.y, ay); az = fmaf(wgt, v.z, az); ph = fmaf(wgt, v.w, ph);
            }
    acc_out[3 * t] = ax; acc_out[3 * t + 1] = ay; acc_out[3 * t + 2] = az;
    if (pot_out) pot_out[t] = ph;
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

extern "C" og_pm *og_pm_create(uint32_t ng, float box, float r_s, float G, og_stream stream)
{
    og_set_error("%s", "");
    if (ng < 8 || ng > 2048 || (ng & 1u)) { og_set_error("og_pm_create: ng = %u must be even and in [8, 2048]", ng); return nullptr; }
    if (!(box > 0.0f) || !(r_s > 0.0f)) { og_set_error("og_pm_create: box and r_s must be > 0"); return nullptr; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); og_set_error("no CUDA device available (there is no CPU fallback)"); return nullptr; }
    cudaStream_t st = (cudaStream_t)stream;
    og_pm *pm = new (std::nothrow) og_pm();
    if (!pm) { og_set_error("host allocation failed"); return nullptr; }
    pm->ng = ng; pm->box = box; pm->r_s = r_s; pm->G = G; pm->device = dev; pm->have_plans = false; pm->arena = nullptr;
    const size_t n3 = (size_t)ng * ng * ng, nk = (size_t)ng * ng * (ng / 2 + 1);
    // The two plans are made first, without cuFFT's own work areas: the forward and the inverse transform of a call
    // run one after the other on one stream, so ONE work area of the larger size serves both and sits in the arena.
    size_t ws_f = 0, ws_b = 0;
    bool planned = cufftCreate(&pm->plan_r2c) == CUFFT_SUCCESS;
    if (planned) {
        planned = cufftCreate(&pm->plan_c2r) == CUFFT_SUCCESS;
        if (!planned) cufftDestroy(pm->plan_r2c);
    }
    if (planned) {
        planned = cufftSetAutoAllocation(pm->plan_r2c, 0) == CUFFT_SUCCESS && cufftSetAutoAllocation(pm->plan_c2r, 0) == CUFFT_SUCCESS &&
                  cufftMakePlan3d(pm->plan_r2c, (int)ng, (int)ng, (int)ng, CUFFT_R2C, &ws_f) == CUFFT_SUCCESS &&
                  cufftMakePlan3d(pm->plan_c2r, (int)ng, (int)ng, (int)ng, CUFFT_C2R, &ws_b) == CUFFT_SUCCESS;
        if (!planned) { cufftDestroy(pm->plan_r2c); cufftDestroy(pm->plan_c2r); }
    }
    if (!planned) {
        (void)cudaGetLastError();
        og_set_error("og_pm_create: cuFFT plan creation failed for ng = %u", ng);
        delete pm;
        return nullptr;
    }
    pm->have_plans = true;
    const size_t work = ws_f > ws_b ? ws_f : ws_b;
    const size_t o_m = 0, o_k = o_m + align256(n3 * 4), o_f = o_k + align256(nk * 8), o_t = o_f + align256(n3 * 16),
                 o_d = o_t + align256(ng * 4), o_s = o_d + align256(ng * 4), o_w = o_s + 256, total = o_w + align256(work);
    pm->arena_bytes = total;
    if (cudaMalloc(&pm->arena, total) != cudaSuccess) {
        (void)cudaGetLastError();
        og_set_error("og_pm_create: cudaMalloc(%zu bytes) failed (ng = %u: %zu bytes of grids + %zu bytes of cuFFT work area)",
                     total, ng, total - align256(work), work);
        cufftDestroy(pm->plan_r2c); cufftDestroy(pm->plan_c2r);
        delete pm;
        return nullptr;
    }
    char *b = (char *)pm->arena;
    pm->mgrid = (float *)(b + o_m); pm->kgrid = (float2 *)(b + o_k); pm->fgrid = (float4 *)(b + o_f);
    pm->k2tab = (float *)(b + o_t); pm->dctab = (float *)(b + o_d); pm->d_status = (uint32_t *)(b + o_s);
    // per-axis tables in fp64 on the host (R32): k^2 and the doubly divided CIC window
    std::vector<float> k2(ng), dc(ng);
    const double PI = 3.14159265358979323846;
    for (uint32_t j = 0; j < ng; ++j) {
        const int n = (j <= ng / 2) ? (int)j : (int)j - (int)ng;           // (-ng/2, ng/2]
        const double k = 2.0 * PI * n / (double)box;
        k2[j] = (float)(k * k);
        const double a = PI * n / (double)ng;
        const double s = (n == 0) ? 1.0 : sin(a) / a;
        dc[j] = (float)(1.0 / (s * s * s * s));
    }
    bool ok = cudaMemsetAsync(pm->d_status, 0, 256, st) == cudaSuccess &&
              cudaMemcpyAsync(pm->k2tab, k2.data(), ng * 4, cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaMemcpyAsync(pm->dctab, dc.data(), ng * 4, cudaMemcpyHostToDevice, st) == cudaSuccess &&
              cudaStreamSynchronize(st) == cudaSuccess;      // the host tables go out of scope
    if (ok && work)
        ok = cufftSetWorkArea(pm->plan_r2c, b + o_w) == CUFFT_SUCCESS && cufftSetWorkArea(pm->plan_c2r, b + o_w) == CUFFT_SUCCESS;
    if (!ok) {
        (void)cudaGetLastError();
        og_set_error("og_pm_create: table upload or cuFFT work-area set-up failed");
        cufftDestroy(pm->plan_r2c); cufftDestroy(pm->plan_c2r);
        cudaFree(pm->arena);
        delete pm;
        return nullptr;
    }
    return pm;
}

extern "C" int og_pm_longrange(og_pm *pm, const float *pos, const float *mass, uint64_t n, const uint32_t *active_idx,
                               uint64_t n_active, float *acc_out, float *pot_out, og_stream stream)
{
    og_set_error("%s", "");
    if (!pm || !pos || !mass || n == 0 || n >= (1ull << 31)) { og_set_error("og_pm_longrange: bad argument"); return OG_ERR_INVALID_ARG; }
    if (n_active == 0) return OG_OK;   // empty target list: nothing to do (pointers of empty buffers may be NULL)
    if (!active_idx && n_active != n) { og_set_error("active_idx == NULL requires n_active == n"); return OG_ERR_INVALID_ARG; }
    if (!acc_out) { og_set_error("acc_out is NULL"); return OG_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)stream;
    const int ng = (int)pm->ng;
    const size_t n3 = (size_t)ng * ng * ng, nk = (size_t)ng * ng * (ng / 2 + 1);
    const float delta = pm->box / (float)ng, inv_delta = (float)ng / pm->box;
    OG_CUDA_TRY(cudaMemsetAsync(pm->mgrid, 0, n3 * 4, st), return OG_ERR_CUDA);
    k_pm_deposit<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(pos, mass, n, inv_delta, ng, pm->mgrid);
    if (cufftSetStream(pm->plan_r2c, st) != CUFFT_SUCCESS || cufftSetStream(pm->plan_c2r, st) != CUFFT_SUCCESS ||
        cufftExecR2C(pm->plan_r2c, pm->mgrid, (cufftComplex *)pm->kgrid) != CUFFT_SUCCESS) {
        og_set_error("cuFFT forward transform failed");
        return OG_ERR_CUDA;
    }
    const double V = (double)pm->box * pm->box * pm->box;
    const float pref = (float)(-4.0 * 3.14159265358979323846 * (double)pm->G / V);
    k_pm_green<<<(unsigned)((nk + 255) / 256), 256, 0, st>>>(pm->kgrid, ng, pm->k2tab, pm->dctab, pref, pm->r_s * pm->r_s);
    if (cufftExecC2R(pm->plan_c2r, (cufftComplex *)pm->kgrid, pm->mgrid) != CUFFT_SUCCESS) {
        og_set_error("cuFFT inverse transform failed");
        return OG_ERR_CUDA;
    }
    k_pm_gradient<<<(unsigned)((n3 + 255) / 256), 256, 0, st>>>(pm->mgrid, ng, (4.0f / 3.0f) / (2.0f * delta),
                                                                (1.0f / 3.0f) / (4.0f * delta), pm->fgrid);
    k_pm_interp<<<(unsigned)((n_active + 255) / 256), 256, 0, st>>>(pos, active_idx, n, n_active, inv_delta, ng, pm->fgrid,
                                                                   acc_out, pot_out, pm->d_status);
    OG_CUDA_TRY(cudaGetLastError(), return OG_ERR_CUDA);
    return OG_OK;
}

extern "C" int og_pm_status(const og_pm *pm, og_stream stream)
{
    og_set_error("%s", "");
    if (!pm) { og_set_error("og_pm_status: pm is NULL"); return OG_ERR_INVALID_ARG; }
    uint32_t bits = 0;
    OG_CUDA_TRY(cudaMemcpyAsync(&bits, pm->d_status, sizeof(bits), cudaMemcpyDeviceToHost, (cudaStream_t)stream), return OG_ERR_CUDA);
    OG_CUDA_TRY(cudaStreamSynchronize((cudaStream_t)stream), return OG_ERR_CUDA);
    if (bits & OG_DEV_BAD_INDEX) {
        og_set_error("og_pm_longrange: an active_idx entry was >= n (such targets were given a zero force)");
        return OG_ERR_INVALID_ARG;
    }
    return OG_OK;
}

extern "C" void og_pm_free(og_pm *pm, og_stream stream)
{
    if (!pm) return;
    cudaStreamSynchronize((cudaStream_t)stream);   // the grids may still be in use on the caller's stream
    if (pm->have_plans) { cufftDestroy(pm->plan_r2c); cufftDestroy(pm->plan_c2r); }
    if (pm->arena) cudaFree(pm->arena);
    delete pm;
}
