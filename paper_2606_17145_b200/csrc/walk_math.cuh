// walk_math.cuh -- per-target arithmetic of the short-range walk (rows a6 of SURVEY.md
// Sec. 8(a); readings C5, C6, R13..R22 of Sec. 8.3, listed in DESIGN.md Sec. 3).
//
// All arithmetic is fp32.  Every *decision* that is discontinuous in the result (open /
// accept, inside r_cut or not) is taken in fp32 first; if the fp32 operands are within a
// relative band OG_BAND of the threshold the same test is re-evaluated in fp64 from the same
// fp32 inputs, in the order the method states it, so that the decision equals the one an
// exact evaluation takes.  The band is ~30x the worst fp32 error of the
// tests, and only ~1e-5 of all tests fall inside it.
#pragma once
#include "og_internal.cuh"

#define OG_BAND 1.0e-5f
#define OG_WMAX 2.5f  // the split-factor polynomial is fitted on w = r / (2 r_s) in [0, OG_WMAX]: rcut_over_rs <= 5

struct WalkConst {
    float L, invL;
    float rcut, rcut2;
    float rcut2_lo, rcut2_hi;   // rcut2 * (1 -+ OG_BAND): outside this band the fp32 cutoff test is final
    float cull_r;        // r_cut * (1 + 1e-5) + 1e-6 L : conservative cull radius
    float G;
    float alpha;
    float theta2;
    float k_w;           // 1 / (2 r_s): w = r k_w
    float k_e;           // -log2(e) / (4 r_s^2): exp(-w^2) = ex2(r^2 k_e)
    float hmax2g;        // (largest softening length h of any particle)^2 (1 + 1e-5): r^2 above it is Newtonian
    // fp64 copies for the re-evaluation path (C0: fp32 parameters promoted to fp64)
    double dL, drcut, dG, dalpha, dtheta2;
};

struct Target {
    float x, y, z;
    float h;       // fl32(2.8 eps_i)
    float A;       // alpha * a_old (fp32 product); unused in geometric mode
    float aold;    // a_old as given (for the fp64 path)
    uint32_t slot; // own sorted slot (self exclusion)
};

struct Accum {
    float ax, ay, az, pot;
};

__device__ __forceinline__ float og_wrap(float d, const WalkConst &c)
{
    return fmaf(-c.L, rintf(d * c.invL), d);  // R13: d - L round(d / L); exact for |d| < 1.5 L
}

__device__ __forceinline__ double og_wrap64(double d, double L) { return d - L * round(d / L); }

// Split factors (R18) in registers: E(w) = erfc(w) = exp(-w^2) P(w), T(w) = E(w) + (2 / sqrt(pi)) w exp(-w^2),
// w = r / (2 r_s).  P = degree-10 polynomial, weighted-minimax fit of erfcx on [0, OG_WMAX] (weight exp(-w^2));
// exp(-w^2) = ex2.approx(r^2 k_e).  Max abs error of T and E in fp32 Horner: 1.8e-7 (budget 1e-6).
// Coefficients of P (degree 10, highest first: OG_SP10 .. OG_SP0), shared by og_split and og_split2.
#define OG_SP10 1.651949088e-04f
#define OG_SP9 -2.225770333e-03f
#define OG_SP8 1.362162625e-02f
#define OG_SP7 -5.118135848e-02f
#define OG_SP6 1.361394758e-01f
#define OG_SP5 -2.828231287e-01f
#define OG_SP4 4.931623193e-01f
#define OG_SP3 -7.507289497e-01f
#define OG_SP2 9.998254850e-01f
#define OG_SP1 -1.128371385e+00f
#define OG_SP0 9.999999427e-01f
#define OG_TWO_OVER_SQRTPI 1.1283791670955126f
__device__ __forceinline__ float og_ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// rsqrt.approx without the denormal-range rescaling of rsqrtf (arguments here are >= 1e-20).
__device__ __forceinline__ float og_rsqrt(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void og_split(float r, float r2, const WalkConst &c, float &T, float &E)
{
    const float w = r * c.k_w;
    const float ex = og_ex2(r2 * c.k_e);
    float p = OG_SP10;
    p = fmaf(p, w, OG_SP9);
    p = fmaf(p, w, OG_SP8);
    p = fmaf(p, w, OG_SP7);
    p = fmaf(p, w, OG_SP6);
    p = fmaf(p, w, OG_SP5);
    p = fmaf(p, w, OG_SP4);
    p = fmaf(p, w, OG_SP3);
    p = fmaf(p, w, OG_SP2);
    p = fmaf(p, w, OG_SP1);
    p = fmaf(p, w, OG_SP0);
    E = p * ex;
    T = fmaf(OG_TWO_OVER_SQRTPI * w, ex, E);
}

// ---- packed fp32 pairs (sm_100: fma/mul/add/sub.rn.f32x2 -> FFMA2 / FMUL2 / FADD2) ---------------
// One instruction, two independent IEEE fp32 operations on a 64-bit register pair: the two source chains
// of the consume loop and the two nodes of an undecided-node test are pairs of identical operations, so
// packing them halves their issue slots (the walk is issue-bound).  Each half rounds
// exactly like the scalar instruction.
typedef unsigned long long f32x2;

__device__ __forceinline__ f32x2 pk2(float a, float b)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float &a, float &b)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 bc2(float a) { return pk2(a, a); }

// og_split for two sources at once, same coefficients.  The polynomial is evaluated as even and odd part
// in w^2 (two independent Horner chains, depth 7 instead of 10: the walk is latency-bound at its occupancy),
// P(w) = Pe(w^2) + w Po(w^2); tests/test_split_poly.py evaluates this order in fp32 against the R18 budget.
__device__ __forceinline__ void og_split2(f32x2 r, f32x2 r2, const WalkConst &c, f32x2 &T, f32x2 &E)
{
    const f32x2 w = mul2(r, bc2(c.k_w));
    const f32x2 a = mul2(r2, bc2(c.k_e));
    float a0, a1;
    upk2(a, a0, a1);
    const f32x2 ex = pk2(og_ex2(a0), og_ex2(a1));
    const f32x2 w2 = mul2(w, w);
    f32x2 pe = bc2(OG_SP10), po = bc2(OG_SP9);
    pe = fma2(pe, w2, bc2(OG_SP8));
    po = fma2(po, w2, bc2(OG_SP7));
    pe = fma2(pe, w2, bc2(OG_SP6));
    po = fma2(po, w2, bc2(OG_SP5));
    pe = fma2(pe, w2, bc2(OG_SP4));
    po = fma2(po, w2, bc2(OG_SP3));
    pe = fma2(pe, w2, bc2(OG_SP2));
    po = fma2(po, w2, bc2(OG_SP1));
    pe = fma2(pe, w2, bc2(OG_SP0));
    const f32x2 p = fma2(po, w, pe);
    E = mul2(p, ex);
    T = fma2(mul2(w, bc2(OG_TWO_OVER_SQRTPI)), ex, E);
}

// ---- cutoff decision r < r_cut (R17, strict) ------------------------------------------------
__device__ __noinline__ bool og_inside_rcut64(float sx, float sy, float sz, const Target &t,
                                              const WalkConst &c, unsigned long long *counters)
{
    const double dx = og_wrap64((double)sx - (double)t.x, c.dL);
    const double dy = og_wrap64((double)sy - (double)t.y, c.dL);
    const double dz = og_wrap64((double)sz - (double)t.z, c.dL);
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    if (counters) atomicAdd(&counters[OGC_FP64], 1ull);
    return sqrt(r2) < c.drcut;
}

__device__ __forceinline__ bool og_inside_rcut(float r2, float sx, float sy, float sz, const Target &t,
                                               const WalkConst &c, unsigned long long *counters)
{
    bool in = r2 < c.rcut2_lo;
    if (!in && r2 < c.rcut2_hi) in = og_inside_rcut64(sx, sy, sz, t, c, counters);
    return in;
}

// ---- pair kernel C5 ------------------------------------------------------------------------
// Interaction with a source at nearest-image offset d (|d|^2 = r2, already known to be inside
// r_cut), gm = G * mass, softening length ph (0 for a node monopole: R16 guarantees r >= h_i there,
// so node interactions are Newtonian, R21).  Returns 1 for r >= h, 2 for r < h.
template <bool POT>
__device__ __forceinline__ int og_pair_core(float dx, float dy, float dz, float r2, float gm, float ph,
                                            const Target &t, const WalkConst &c, Accum &acc)
{
    r2 = fmaxf(r2, 1.0e-36f);           // distinct coincident particles: force 0, potential -14/5 m/h
    const float rinv = rsqrtf(r2);
    const float r = r2 * rinv;
    const float h = fmaxf(t.h, ph);     // R19
    float T, E;
    og_split(r, r2, c, T, E);
    float g, pp;
    int kind = 1;
    if (r >= h) {
        g = rinv * rinv * rinv;
        pp = -rinv;
    } else {
        kind = 2;
        const float hinv = __frcp_rn(h);
        const float u = r * hinv, u2 = u * u;
        const float h3inv = hinv * hinv * hinv;
        if (u < 0.5f) {
            g = h3inv * fmaf(u2, fmaf(32.0f, u, -38.4f), 10.666666666666666f);
            pp = hinv * fmaf(u2, fmaf(u2, fmaf(6.4f, u, -9.6f), 5.333333333333333f), -2.8f);
        } else {
            const float uinv = __frcp_rn(u);
            const float u3inv = uinv * uinv * uinv;
            g = h3inv * (fmaf(u, fmaf(u, fmaf(-10.666666666666666f, u, 38.4f), -48.0f), 21.333333333333332f) -
                         0.06666666666666667f * u3inv);
            pp = hinv * (fmaf(u2, fmaf(u, fmaf(u, fmaf(-2.1333333333333333f, u, 9.6f), -16.0f), 10.666666666666666f),
                              -3.2f) +
                         0.06666666666666667f * uinv);
        }
    }
    const float f = gm * g * T;
    acc.ax = fmaf(f, dx, acc.ax);
    acc.ay = fmaf(f, dy, acc.ay);
    acc.az = fmaf(f, dz, acc.az);
    if (POT) acc.pot = fmaf(gm * pp, E, acc.pot);
    return kind;
}

// Source particle p = (x, y, z, m) in any periodic image; adds to acc if r < r_cut.  Returns 0
// outside, 1 inside with r >= h, 2 inside with r < h.
template <bool POT>
__device__ __forceinline__ int og_pair(const float4 p, float ph, const Target &t, const WalkConst &c,
                                       Accum &acc, unsigned long long *counters)
{
    const float dx = og_wrap(p.x - t.x, c), dy = og_wrap(p.y - t.y, c), dz = og_wrap(p.z - t.z, c);
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if (!og_inside_rcut(r2, p.x, p.y, p.z, t, c, counters)) return 0;
    return og_pair_core<POT>(dx, dy, dz, r2, c.G * p.w, ph, t, c, acc);
}

// ---- node: cull, opening decision, monopole ------------------------------------------------
struct NodeRec {
    float4 com;   // s, M
    float4 cell;  // c, l
    float4 lo;    // lo, h_max
    float4 hi;    // hi, -
};

// Conservative cutoff-box test against the tight AABB (C6 step 1; result-neutral, R17).
__device__ __forceinline__ bool og_cull(const NodeRec &n, const Target &t, const WalkConst &c)
{
    const float mx = 0.5f * (n.lo.x + n.hi.x), my = 0.5f * (n.lo.y + n.hi.y), mz = 0.5f * (n.lo.z + n.hi.z);
    const float hx = 0.5f * (n.hi.x - n.lo.x), hy = 0.5f * (n.hi.y - n.lo.y), hz = 0.5f * (n.hi.z - n.lo.z);
    const float ex = fabsf(og_wrap(t.x - mx, c)) - hx;
    const float ey = fabsf(og_wrap(t.y - my, c)) - hy;
    const float ez = fabsf(og_wrap(t.z - mz, c)) - hz;
    return fmaxf(ex, fmaxf(ey, ez)) > c.cull_r;
}

// fp64 re-evaluation of C6 step 3, exactly in the stated order, from the fp32 inputs.
template <bool GEOM>
__device__ __noinline__ bool og_open64(const NodeRec &n, const Target &t, const WalkConst &c,
                                       unsigned long long *counters)
{
    const double x[3] = {(double)t.x, (double)t.y, (double)t.z};
    const double s[3] = {(double)n.com.x, (double)n.com.y, (double)n.com.z};
    const double cc[3] = {(double)n.cell.x, (double)n.cell.y, (double)n.cell.z};
    double d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) d[k] = og_wrap64(s[k] - x[k], c.dL);
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2]));
    const double M = (double)n.com.w, l = (double)n.cell.w;
    bool open = false;
    if (GEOM) {
        if (__dmul_rn(l, l) > __dmul_rn(c.dtheta2, r2)) open = true;
    } else {
        const double A = __dmul_rn(c.dalpha, (double)t.aold);
        if (__dmul_rn(__dmul_rn(__dmul_rn(c.dG, M), l), l) > __dmul_rn(__dmul_rn(A, r2), r2)) open = true;
    }
    bool inside = true;
#pragma unroll
    for (int k = 0; k < 3; ++k)
        if (!(fabs(og_wrap64(cc[k] - x[k], c.dL)) < __dmul_rn(0.6, l))) inside = false;
    if (inside) open = true;
    const double hm = (double)n.lo.w, hi = (double)t.h;
    const double hh = hi > hm ? hi : hm;
    if (r2 < __dmul_rn(hh, hh)) open = true;
    if (counters) atomicAdd(&counters[OGC_FP64], 1ull);
    return open;
}

// C6 steps 2-3 in fp32 (+ band re-evaluation).  Outputs d = wrap(s - x) and r2.
template <bool GEOM>
__device__ __forceinline__ bool og_open(const NodeRec &n, const Target &t, const WalkConst &c, float &dx,
                                        float &dy, float &dz, float &r2, unsigned long long *counters)
{
    dx = og_wrap(n.com.x - t.x, c);
    dy = og_wrap(n.com.y - t.y, c);
    dz = og_wrap(n.com.z - t.z, c);
    r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const float l = n.cell.w;
    const float l2 = l * l;
    float lhs, rhs;
    if (GEOM) {
        lhs = l2;
        rhs = c.theta2 * r2;
    } else {
        lhs = c.G * n.com.w * l2;   // R14: G M l^2 > alpha a_old r^4, strict
        rhs = t.A * r2 * r2;
    }
    bool open = lhs > rhs;
    bool amb = fabsf(lhs - rhs) <= OG_BAND * fmaxf(lhs, rhs);
    // inside guard R15: |wrap(c_k - x_k)| < 0.6 l for all k
    const float lim = 0.6f * l;
    const float cx = fabsf(og_wrap(n.cell.x - t.x, c)), cy = fabsf(og_wrap(n.cell.y - t.y, c)),
                cz = fabsf(og_wrap(n.cell.z - t.z, c));
    const float cmax = fmaxf(cx, fmaxf(cy, cz));
    open |= cmax < lim;
    // only the largest component can sit on the threshold in a way that matters
    amb |= fabsf(cmax - lim) <= OG_BAND * l;
    // softening guard R16: r^2 < max(h_i, h_max)^2
    const float hh = fmaxf(t.h, n.lo.w);
    const float hh2 = hh * hh;
    open |= r2 < hh2;
    amb |= fabsf(r2 - hh2) <= OG_BAND * hh2;
    if (amb) open = og_open64<GEOM>(n, t, c, counters);
    return open;
}

// Monopole of mass GM = G * M at offset d (r2 inside r_cut), Newtonian force times the split
// factor (R21).
template <bool POT>
__device__ __forceinline__ void og_monopole_core(float GM, float dx, float dy, float dz, float r2,
                                                 const WalkConst &c, Accum &acc)
{
    const float rinv = rsqrtf(r2);
    const float r = r2 * rinv;
    float T, E;
    og_split(r, r2, c, T, E);
    const float gr = GM * rinv;
    const float f = gr * T * (rinv * rinv);
    acc.ax = fmaf(f, dx, acc.ax);
    acc.ay = fmaf(f, dy, acc.ay);
    acc.az = fmaf(f, dz, acc.az);
    if (POT) acc.pot = fmaf(-gr, E, acc.pot);
}

// C6 step 4: accepted node, Newtonian monopole times the split factor (R21).  Returns 1 if
// r < r_cut.
template <bool POT>
__device__ __forceinline__ int og_monopole(const NodeRec &n, const Target &t, const WalkConst &c,
                                           float dx, float dy, float dz,
                                           float r2, Accum &acc, unsigned long long *counters)
{
    if (!og_inside_rcut(r2, n.com.x, n.com.y, n.com.z, t, c, counters)) return 0;
    og_monopole_core<POT>(c.G * n.com.w, dx, dy, dz, r2, c, acc);
    return 1;
}
