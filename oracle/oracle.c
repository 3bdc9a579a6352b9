/*
 * oracle/oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the TreePM short-range gravity path
 * (Morton keys -> stable sort -> canonical octree -> monopole upward pass ->
 * per-target tree walk) plus the O(N^2) direct short-range sum.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant generator with the CUDA path in
 * paper_2606_17145_b200/csrc/.
 *
 * What it follows.  The paper states the method only qualitatively:
 * "for each dynamically active particle, a tree walk is performed to compute the
 * forces acting on it" (Sec. 2), Barnes & Hut gravity "opened with an
 * angular criterion", lineage Gadget3 <- Gadget-2, Springel 2005
 * (PAPER.md:57).  It prints no formula.  The arithmetic below is therefore the
 * reading fixed in SURVEY.md Sec. 8.3 (C0..C7, R1..R30) from BASELINE.json's
 * north_star and the Gadget-2 formulas; every function cites its item, and
 * DESIGN.md lists every such reading.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P15 of SURVEY.md Sec. 8.3.
 * "Parity unpinned": none of the arithmetic; the *choice* among the conventions
 * R14..R16 (strict '>' in the opening test, guard factor 0.6, softening-guard
 * form) cannot be pinned by anything in the paper -- they are conventions.
 *
 * Build:  gcc -O2 -std=c11 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC
 * (-ffp-contract=off matters: C1 needs a single-rounded fp32 multiply, C4 needs
 * separately rounded fp64 products.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_LEVEL 21
#define ORC_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------------- */
/* C0: parameters.  The scalar parameters are the fp32 fields of the caller's  */
/* parameter block promoted to fp64; derived constants are formed in fp64.     */
/* ------------------------------------------------------------------------- */
typedef struct {
    float G;            /* gravitational constant (R12: 1 in all configs)      */
    float L;            /* periodic box side                                   */
    float r_s;          /* force-split scale                                   */
    float rcut_over_rs; /* 4.5 (north_star)                                    */
    float alpha;        /* relative opening criterion parameter                */
    float theta;        /* geometric criterion, used iff a_old == NULL         */
    uint32_t leaf_max;  /* bucket size of the canonical octree (R7)            */
    uint32_t want_pot;  /* unused by the arithmetic; kept for symmetry         */
} orc_params;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------- */
/* C1: 64-bit Morton keys (R1, R2).                                            */
/* S = (float)(2^21 / L); per axis t = x *_{fp32,RN} S (one IEEE binary32      */
/* multiply, no FMA); clamp to [0, 2^21-1]; truncate; interleave so that bit b */
/* of q_x -> key bit 3b+2, q_y -> 3b+1, q_z -> 3b; key bit 63 = 0.             */
/* ------------------------------------------------------------------------- */
static uint32_t orc_quantise(float x, float S)
{
    volatile float t = x * S; /* volatile: force the rounding to binary32 */
    float u = t;
    if (!(u >= 0.0f)) u = 0.0f;
    if (u > 2097151.0f) u = 2097151.0f;
    return (uint32_t)u;
}

uint64_t orc_interleave(uint32_t qx, uint32_t qy, uint32_t qz)
{
    uint64_t key = 0;
    for (int b = 0; b < ORC_MAX_LEVEL; ++b) {
        key |= (uint64_t)((qx >> b) & 1u) << (3 * b + 2);
        key |= (uint64_t)((qy >> b) & 1u) << (3 * b + 1);
        key |= (uint64_t)((qz >> b) & 1u) << (3 * b);
    }
    return key;
}

void orc_deinterleave(uint64_t key, uint32_t *qx, uint32_t *qy, uint32_t *qz)
{
    uint32_t x = 0, y = 0, z = 0;
    for (int b = 0; b < ORC_MAX_LEVEL; ++b) {
        x |= (uint32_t)((key >> (3 * b + 2)) & 1u) << b;
        y |= (uint32_t)((key >> (3 * b + 1)) & 1u) << b;
        z |= (uint32_t)((key >> (3 * b)) & 1u) << b;
    }
    *qx = x; *qy = y; *qz = z;
}

void orc_keys(const float *pos, uint64_t n, float L, uint64_t *keys)
{
    const float S = (float)(2097152.0 / (double)L);
    for (uint64_t i = 0; i < n; ++i) {
        uint32_t qx = orc_quantise(pos[3 * i + 0], S);
        uint32_t qy = orc_quantise(pos[3 * i + 1], S);
        uint32_t qz = orc_quantise(pos[3 * i + 2], S);
        keys[i] = orc_interleave(qx, qy, qz);
    }
}

/* ------------------------------------------------------------------------- */
/* C2: sort (R3).  Ascending (key, original index), lexicographic.             */
/* perm[s] = original index of sorted slot s.                                  */
/* ------------------------------------------------------------------------- */
typedef struct { uint64_t key; uint32_t idx; } orc_kv;

static int orc_kv_cmp(const void *a, const void *b)
{
    const orc_kv *p = (const orc_kv *)a, *q = (const orc_kv *)b;
    if (p->key < q->key) return -1;
    if (p->key > q->key) return 1;
    if (p->idx < q->idx) return -1;
    if (p->idx > q->idx) return 1;
    return 0;
}

int orc_sort(const uint64_t *keys, uint64_t n, uint32_t *perm, uint64_t *keys_sorted)
{
    orc_kv *kv = (orc_kv *)malloc((size_t)n * sizeof(orc_kv));
    if (!kv) return -1;
    for (uint64_t i = 0; i < n; ++i) { kv[i].key = keys[i]; kv[i].idx = (uint32_t)i; }
    qsort(kv, (size_t)n, sizeof(orc_kv), orc_kv_cmp);
    for (uint64_t s = 0; s < n; ++s) { perm[s] = kv[s].idx; keys_sorted[s] = kv[s].key; }
    free(kv);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* C3: canonical sparse octree (R5..R7).                                       */
/* cell (l, p) = sorted slots whose key >> (63 - 3l) == p.  Root = node 0.     */
/* leaf iff count <= leaf_max or l == 21; otherwise one child per non-empty    */
/* octant in ascending octant order; breadth-first numbering.                  */
/* Pass NULL arrays to count nodes only.  Returns the node count, or           */
/* -(needed) if cap is too small.                                              */
/* ------------------------------------------------------------------------- */
int64_t orc_tree_build(const uint64_t *keys_sorted, uint64_t n, uint32_t leaf_max,
                       int64_t cap, uint8_t *level, uint32_t *first, uint32_t *count,
                       uint32_t *first_child, uint8_t *n_child)
{
    /* counting pass keeps only a queue of (level, first, count) */
    int64_t qcap = 1024, nn = 0;
    uint8_t *qlev = (uint8_t *)malloc((size_t)qcap);
    uint32_t *qfirst = (uint32_t *)malloc((size_t)qcap * 4);
    uint32_t *qcount = (uint32_t *)malloc((size_t)qcap * 4);
    if (!qlev || !qfirst || !qcount) return 0;
    qlev[0] = 0; qfirst[0] = 0; qcount[0] = (uint32_t)n; nn = 1;
    const int fill = (level != NULL);
    for (int64_t j = 0; j < nn; ++j) {
        const uint32_t lv = qlev[j], f = qfirst[j], c = qcount[j];
        uint32_t nch = 0, fch = 0;
        if (c > leaf_max && lv < ORC_MAX_LEVEL) {
            /* split the slot range by the octant digit of level lv -> lv+1 */
            const int shift = 60 - 3 * (int)lv;
            uint32_t cnt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (uint32_t s = f; s < f + c; ++s) cnt[(keys_sorted[s] >> shift) & 7u]++;
            fch = (uint32_t)nn;
            uint32_t start = f;
            for (int o = 0; o < 8; ++o) {
                if (cnt[o] == 0) continue;
                if (nn == qcap) {
                    qcap *= 2;
                    qlev = (uint8_t *)realloc(qlev, (size_t)qcap);
                    qfirst = (uint32_t *)realloc(qfirst, (size_t)qcap * 4);
                    qcount = (uint32_t *)realloc(qcount, (size_t)qcap * 4);
                    if (!qlev || !qfirst || !qcount) return 0;
                }
                qlev[nn] = (uint8_t)(lv + 1); qfirst[nn] = start; qcount[nn] = cnt[o];
                start += cnt[o]; ++nn; ++nch;
            }
        }
        if (fill && j < cap) {
            level[j] = (uint8_t)lv; first[j] = f; count[j] = c;
            first_child[j] = fch; n_child[j] = (uint8_t)nch;
        }
    }
    free(qlev); free(qfirst); free(qcount);
    if (fill && nn > cap) return -nn;
    return nn;
}

/* ------------------------------------------------------------------------- */
/* C4: upward pass (R8..R11).  Leaves: sums over their slots in slot order;    */
/* internal nodes: over children in order; all fp64.  M = sum m;               */
/* s = (sum m x)/M; l = L/2^level; c_k = (p_k + 1/2) l; AABB lo/hi; h_max.     */
/* R9: the record the walk reads is the fp32 rounding of these results, and    */
/* per particle h_i = fl32(2.8 eps_i).                                         */
/* Inputs are in SORTED order (spos[s] = pos[perm[s]] etc.).                   */
/* ------------------------------------------------------------------------- */
void orc_particle_h(const float *eps, uint64_t n, float *h)
{
    for (uint64_t i = 0; i < n; ++i) h[i] = (float)(2.8 * (double)eps[i]);
}

int orc_upward(const uint64_t *keys_sorted, const float *spos, const float *smass,
               const float *sh, float L, int64_t n_nodes, const uint8_t *level,
               const uint32_t *first, const uint32_t *count, const uint32_t *first_child,
               const uint8_t *n_child,
               /* fp64 results */
               double *M64, double *s64 /* [n][3] */,
               /* fp32 node record (R9) */
               float *M32, float *s32 /* [n][3] */, float *c32 /* [n][3] */, float *l32,
               float *hmax32, float *lo32 /* [n][3] */, float *hi32 /* [n][3] */)
{
    double *mx = (double *)malloc((size_t)n_nodes * 3 * sizeof(double));
    if (!mx) return -1;
    for (int64_t j = n_nodes - 1; j >= 0; --j) {
        double M = 0.0, ax = 0.0, ay = 0.0, az = 0.0;
        float lo[3], hi[3], hm;
        if (n_child[j] == 0) {
            const uint32_t f = first[j];
            lo[0] = hi[0] = spos[3 * f]; lo[1] = hi[1] = spos[3 * f + 1];
            lo[2] = hi[2] = spos[3 * f + 2]; hm = sh[f];
            for (uint32_t s = f; s < f + count[j]; ++s) {
                const double m = (double)smass[s];
                M += m;
                ax += m * (double)spos[3 * s]; ay += m * (double)spos[3 * s + 1];
                az += m * (double)spos[3 * s + 2];
                for (int k = 0; k < 3; ++k) {
                    if (spos[3 * s + k] < lo[k]) lo[k] = spos[3 * s + k];
                    if (spos[3 * s + k] > hi[k]) hi[k] = spos[3 * s + k];
                }
                if (sh[s] > hm) hm = sh[s];
            }
        } else {
            const uint32_t fc = first_child[j];
            for (int k = 0; k < 3; ++k) { lo[k] = lo32[3 * fc + k]; hi[k] = hi32[3 * fc + k]; }
            hm = hmax32[fc];
            for (uint32_t ch = fc; ch < fc + n_child[j]; ++ch) {
                M += M64[ch];
                ax += mx[3 * ch]; ay += mx[3 * ch + 1]; az += mx[3 * ch + 2];
                for (int k = 0; k < 3; ++k) {
                    if (lo32[3 * ch + k] < lo[k]) lo[k] = lo32[3 * ch + k];
                    if (hi32[3 * ch + k] > hi[k]) hi[k] = hi32[3 * ch + k];
                }
                if (hmax32[ch] > hm) hm = hmax32[ch];
            }
        }
        M64[j] = M; mx[3 * j] = ax; mx[3 * j + 1] = ay; mx[3 * j + 2] = az;
        s64[3 * j] = ax / M; s64[3 * j + 1] = ay / M; s64[3 * j + 2] = az / M;
        /* geometric cell: side and centre from the key prefix of the first slot */
        const int lv = level[j];
        const double l = (double)L / (double)((uint64_t)1 << lv);
        uint32_t qx, qy, qz;
        orc_deinterleave(keys_sorted[first[j]], &qx, &qy, &qz);
        const uint32_t px = lv ? (qx >> (ORC_MAX_LEVEL - lv)) : 0;
        const uint32_t py = lv ? (qy >> (ORC_MAX_LEVEL - lv)) : 0;
        const uint32_t pz = lv ? (qz >> (ORC_MAX_LEVEL - lv)) : 0;
        M32[j] = (float)M;
        s32[3 * j] = (float)s64[3 * j]; s32[3 * j + 1] = (float)s64[3 * j + 1];
        s32[3 * j + 2] = (float)s64[3 * j + 2];
        c32[3 * j] = (float)(((double)px + 0.5) * l);
        c32[3 * j + 1] = (float)(((double)py + 0.5) * l);
        c32[3 * j + 2] = (float)(((double)pz + 0.5) * l);
        l32[j] = (float)l;
        hmax32[j] = hm;
        for (int k = 0; k < 3; ++k) { lo32[3 * j + k] = lo[k]; hi32[3 * j + k] = hi[k]; }
    }
    free(mx);
    return 0;
}

/* ------------------------------------------------------------------------- */
/* C5: pair kernel (R12, R17..R21, R24).                                       */
/* Cubic-spline softened force/potential factors with h = 2.8 eps (Gadget-2,   */
/* Springel 2005, the paper's citation PAPER.md:296), and the TreePM split     */
/* factors T(w) = erfc(w) + (2w/sqrt(pi)) exp(-w^2), E(w) = erfc(w),           */
/* w = r / (2 r_s).                                                            */
/* ------------------------------------------------------------------------- */
double orc_spline_g(double r, double h) /* a = G m d g */
{
    const double u = r / h;
    if (u >= 1.0) return 1.0 / (r * r * r);
    const double h3 = h * h * h;
    if (u < 0.5) return (32.0 / 3.0 + u * u * (32.0 * u - 192.0 / 5.0)) / h3;
    return (64.0 / 3.0 - 48.0 * u + (192.0 / 5.0) * u * u - (32.0 / 3.0) * u * u * u
            - 1.0 / (15.0 * u * u * u)) / h3;
}

double orc_spline_p(double r, double h) /* phi = G m p */
{
    const double u = r / h;
    if (u >= 1.0) return -1.0 / r;
    if (u < 0.5)
        return (-14.0 / 5.0 + u * u * (16.0 / 3.0 + u * u * ((32.0 / 5.0) * u - 48.0 / 5.0))) / h;
    return (-16.0 / 5.0 + 1.0 / (15.0 * u)
            + u * u * (32.0 / 3.0 + u * (-16.0 + u * (48.0 / 5.0 - (32.0 / 15.0) * u)))) / h;
}

double orc_split_T(double w)
{
    return erfc(w) + (2.0 * w / sqrt(ORC_PI)) * exp(-w * w);
}

double orc_split_E(double w) { return erfc(w); }

/* nearest image, R13: d -= L round(d / L) */
static inline double orc_wrap(double d, double L) { return d - L * round(d / L); }

typedef struct {
    double G, L, r_s, r_cut, inv2rs, alpha, theta2;
} orc_derived;

static orc_derived orc_derive(const orc_params *p)
{
    orc_derived d;
    d.G = (double)p->G; d.L = (double)p->L; d.r_s = (double)p->r_s;
    d.r_cut = (double)p->rcut_over_rs * (double)p->r_s;
    d.inv2rs = 1.0 / (2.0 * d.r_s);
    d.alpha = (double)p->alpha;
    d.theta2 = (double)p->theta * (double)p->theta;
    return d;
}

/* One pair: target at x (softening length h_i) feels source j at xj, mass mj,   */
/* h_j.  Adds to acc/pot if r < r_cut (strict, R17).  Returns 0 beyond r_cut,    */
/* 1 inside with r >= h, 2 inside with r < h.                                   */
static inline int orc_pair(const orc_derived *D, const double x[3], double hi,
                           const double xj[3], double mj, double hj, double acc[3],
                           double *pot)
{
    double d[3];
    for (int k = 0; k < 3; ++k) d[k] = orc_wrap(xj[k] - x[k], D->L);
    const double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(r < D->r_cut)) return 0;
    const double h = hi > hj ? hi : hj; /* R19 */
    const double w = r * D->inv2rs;
    const double g = orc_spline_g(r, h) * orc_split_T(w);
    const double p = orc_spline_p(r, h) * orc_split_E(w);
    for (int k = 0; k < 3; ++k) acc[k] += D->G * mj * d[k] * g;
    *pot += D->G * mj * p;
    return r < h ? 2 : 1;
}

/* exported single-pair evaluation for the closed-form pins (P3..P5, P13) */
int orc_pair_eval(const orc_params *p, const double x[3], double h_i, const double xj[3],
                  double mj, double h_j, double acc[3], double *pot)
{
    orc_derived D = orc_derive(p);
    acc[0] = acc[1] = acc[2] = 0.0; *pot = 0.0;
    return orc_pair(&D, x, h_i, xj, mj, h_j, acc, pot);
}

/* ------------------------------------------------------------------------- */
/* C6: walk for one target.  Counters per target (Sec. 8.3, needed by 8.4):    */
/*  0 V_full  1 V_cull  2 A_in  3 A_out  4 P_in  5 P_out  6 P_soft             */
/*  7 O_int (opened internal)  8 O_leaf (opened leaves)                        */
/*  9 sum of n_child over opened internal nodes  10 sum of count over opened   */
/*  leaves  11 number of opened leaves that hold the target itself (0 or 1)    */
/* ------------------------------------------------------------------------- */
#define ORC_NCOUNT 12

typedef struct {
    const orc_derived *D;
    const uint8_t *n_child; const uint32_t *first, *count, *first_child;
    const float *M32, *s32, *c32, *l32, *hmax32, *lo32, *hi32;
    const float *spos, *smass, *sh;
    double x[3]; double h_i; double A; int geometric; uint32_t self_slot;
    double acc[3]; double pot; uint64_t cnt[ORC_NCOUNT];
} orc_walk_ctx;

static void orc_visit(orc_walk_ctx *W, uint32_t n)
{
    const orc_derived *D = W->D;
    /* 1. cull by the cutoff box around the node's tight AABB (R10, R17) */
    for (int k = 0; k < 3; ++k) {
        const double lo = (double)W->lo32[3 * n + k], hi = (double)W->hi32[3 * n + k];
        const double mid = 0.5 * (lo + hi), half = 0.5 * (hi - lo);
        double e = fabs(orc_wrap(W->x[k] - mid, D->L)) - half;
        if (e < 0.0) e = 0.0;
        if (e > D->r_cut) { W->cnt[1]++; return; }
    }
    W->cnt[0]++;
    /* 2. distance to the centre of mass */
    double d[3];
    for (int k = 0; k < 3; ++k) d[k] = orc_wrap((double)W->s32[3 * n + k] - W->x[k], D->L);
    const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    const double M = (double)W->M32[n], l = (double)W->l32[n];
    /* 3. open? */
    int open = 0;
    if (W->geometric) {
        if (l * l > D->theta2 * r2) open = 1;                 /* R22 */
    } else {
        if (D->G * M * l * l > W->A * r2 * r2) open = 1;      /* R14, strict */
    }
    {   /* inside guard, R15 */
        int inside = 1;
        for (int k = 0; k < 3; ++k)
            if (!(fabs(orc_wrap((double)W->c32[3 * n + k] - W->x[k], D->L)) < 0.6 * l)) inside = 0;
        if (inside) open = 1;
    }
    {   /* softening guard, R16 */
        const double hm = (double)W->hmax32[n];
        const double hh = W->h_i > hm ? W->h_i : hm;
        if (r2 < hh * hh) open = 1;
    }
    /* 4. accept: Newtonian monopole times the split factor (R21) */
    if (!open) {
        const double r = sqrt(r2);
        if (r < D->r_cut) {
            const double w = r * D->inv2rs;
            const double f = D->G * M * orc_split_T(w) / (r2 * r);
            for (int k = 0; k < 3; ++k) W->acc[k] += f * d[k];
            W->pot -= D->G * M * orc_split_E(w) / r;
            W->cnt[2]++;
        } else {
            W->cnt[3]++;
        }
        return;
    }
    /* 5. open */
    if (W->n_child[n] == 0) {
        W->cnt[8]++;
        W->cnt[10] += W->count[n];
        const uint32_t f = W->first[n];
        for (uint32_t s = f; s < f + W->count[n]; ++s) {
            if (s == W->self_slot) { W->cnt[11]++; continue; }
            const double xj[3] = {(double)W->spos[3 * s], (double)W->spos[3 * s + 1],
                                  (double)W->spos[3 * s + 2]};
            const int kind = orc_pair(D, W->x, W->h_i, xj, (double)W->smass[s],
                                      (double)W->sh[s], W->acc, &W->pot);
            if (kind == 0) W->cnt[5]++;
            else { W->cnt[4]++; if (kind == 2) W->cnt[6]++; }
        }
    } else {
        W->cnt[7]++;
        W->cnt[9] += W->n_child[n];
        const uint32_t fc = W->first_child[n];
        for (uint32_t ch = fc; ch < fc + W->n_child[n]; ++ch) orc_visit(W, ch);
    }
}

/* target_slot[t] = sorted slot of target t; a_old[t] (fp32, R23) or NULL ->    */
/* geometric criterion.  Outputs acc[t][3], pot[t] (fp64), counters[t][9].     */
void orc_walk(const orc_params *p, uint64_t n_targets, const uint32_t *target_slot,
              const float *a_old, const uint8_t *n_child, const uint32_t *first,
              const uint32_t *count, const uint32_t *first_child, const float *M32,
              const float *s32, const float *c32, const float *l32, const float *hmax32,
              const float *lo32, const float *hi32, const float *spos, const float *smass,
              const float *sh, double *acc, double *pot, uint64_t *counters)
{
    const orc_derived D = orc_derive(p);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < (int64_t)n_targets; ++t) {
        orc_walk_ctx W;
        memset(&W, 0, sizeof(W));
        W.D = &D; W.n_child = n_child; W.first = first; W.count = count;
        W.first_child = first_child; W.M32 = M32; W.s32 = s32; W.c32 = c32; W.l32 = l32;
        W.hmax32 = hmax32; W.lo32 = lo32; W.hi32 = hi32; W.spos = spos; W.smass = smass;
        W.sh = sh;
        const uint32_t slot = target_slot[t];
        for (int k = 0; k < 3; ++k) W.x[k] = (double)spos[3 * slot + k];
        W.h_i = (double)sh[slot];
        W.self_slot = slot;
        W.geometric = (a_old == NULL);
        W.A = a_old ? D.alpha * (double)a_old[t] : 0.0;
        orc_visit(&W, 0);
        acc[3 * t] = W.acc[0]; acc[3 * t + 1] = W.acc[1]; acc[3 * t + 2] = W.acc[2];
        if (pot) pot[t] = W.pot;
        if (counters)
            for (int c = 0; c < ORC_NCOUNT; ++c) counters[ORC_NCOUNT * t + c] = W.cnt[c];
    }
}

/* ------------------------------------------------------------------------- */
/* C7: direct short-range sum, a_i = sum_{j != i} C5.  O(n_targets * N).       */
/* Works on any ordering; j == i is skipped by index.                          */
/* ------------------------------------------------------------------------- */
void orc_direct(const orc_params *p, uint64_t n, const float *pos, const float *mass,
                const float *h, uint64_t n_targets, const uint32_t *target_idx, double *acc,
                double *pot)
{
    const orc_derived D = orc_derive(p);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < (int64_t)n_targets; ++t) {
        const uint32_t i = target_idx ? target_idx[t] : (uint32_t)t;
        const double x[3] = {(double)pos[3 * i], (double)pos[3 * i + 1], (double)pos[3 * i + 2]};
        double a[3] = {0.0, 0.0, 0.0}, ph = 0.0;
        for (uint64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            const double xj[3] = {(double)pos[3 * j], (double)pos[3 * j + 1],
                                  (double)pos[3 * j + 2]};
            orc_pair(&D, x, (double)h[i], xj, (double)mass[j], (double)h[j], a, &ph);
        }
        acc[3 * t] = a[0]; acc[3 * t + 1] = a[1]; acc[3 * t + 2] = a[2];
        if (pot) pot[t] = ph;
    }
}

/* ------------------------------------------------------------------------- */
/* Row f4 ("secondary" phase): the same  */
/* walk (orc_visit, unchanged) and the same direct sum for targets that are NOT */
/* particles of the tree -- targets imported from another domain.  A target is  */
/* (x, h, a_old); nothing is excluded (no particle of this tree is the target). */
/* ------------------------------------------------------------------------- */
void orc_walk_ext(const orc_params *p, uint64_t n_targets, const float *tpos, const float *th,
                  const float *a_old, const uint8_t *n_child, const uint32_t *first,
                  const uint32_t *count, const uint32_t *first_child, const float *M32,
                  const float *s32, const float *c32, const float *l32, const float *hmax32,
                  const float *lo32, const float *hi32, const float *spos, const float *smass,
                  const float *sh, double *acc, double *pot, uint64_t *counters)
{
    const orc_derived D = orc_derive(p);
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t t = 0; t < (int64_t)n_targets; ++t) {
        orc_walk_ctx W;
        memset(&W, 0, sizeof(W));
        W.D = &D; W.n_child = n_child; W.first = first; W.count = count;
        W.first_child = first_child; W.M32 = M32; W.s32 = s32; W.c32 = c32; W.l32 = l32;
        W.hmax32 = hmax32; W.lo32 = lo32; W.hi32 = hi32; W.spos = spos; W.smass = smass;
        W.sh = sh;
        for (int k = 0; k < 3; ++k) W.x[k] = (double)tpos[3 * t + k];
        W.h_i = (double)th[t];
        W.self_slot = 0xffffffffu;   /* no slot of the tree is the target */
        W.geometric = (a_old == NULL);
        W.A = a_old ? D.alpha * (double)a_old[t] : 0.0;
        orc_visit(&W, 0);
        acc[3 * t] = W.acc[0]; acc[3 * t + 1] = W.acc[1]; acc[3 * t + 2] = W.acc[2];
        if (pot) pot[t] = W.pot;
        if (counters)
            for (int c = 0; c < ORC_NCOUNT; ++c) counters[ORC_NCOUNT * t + c] = W.cnt[c];
    }
}

void orc_direct_ext(const orc_params *p, uint64_t n, const float *pos, const float *mass,
                    const float *h, uint64_t n_targets, const float *tpos, const float *th,
                    double *acc, double *pot)
{
    const orc_derived D = orc_derive(p);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < (int64_t)n_targets; ++t) {
        const double x[3] = {(double)tpos[3 * t], (double)tpos[3 * t + 1], (double)tpos[3 * t + 2]};
        double a[3] = {0.0, 0.0, 0.0}, ph = 0.0;
        for (uint64_t j = 0; j < n; ++j) {
            const double xj[3] = {(double)pos[3 * j], (double)pos[3 * j + 1],
                                  (double)pos[3 * j + 2]};
            orc_pair(&D, x, (double)th[t], xj, (double)mass[j], (double)h[j], a, &ph);
        }
        acc[3 * t] = a[0]; acc[3 * t + 1] = a[1]; acc[3 * t + 2] = a[2];
        if (pot) pot[t] = ph;
    }
}
