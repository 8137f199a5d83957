/*
 * sw_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See sw_oracle.h.
 *
 * Sequential CPU Swendsen-Wang step, written from arXiv 1403.7560 in the paper's
 * order: (1) active-bond generation, (2) cluster labelling, (3) spin flip,
 * then the observables of PAPER.md:142-157.  No blocking, no fusion: one plain loop per sub-step.
 * Compile with -O2 -ffp-contract=off (oracle/build.py) so that the fp32 reflection below is two
 * correctly rounded fp32 operations.
 */
#include "sw_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------
 * Random numbers.  The paper uses a linear congruential generator and says "any other
 * random-number generators can be used".  Reading S1: Philox4x32-10
 * (Salmon et al., SC'11), a counter-based generator, so that every random decision is a pure
 * function of (seed, step, site) and the CUDA path can reproduce it in any order.
 * ------------------------------------------------------------------------------------------ */
void swo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u; /* round multipliers  */
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u; /* Weyl key increments */
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Reading 6 (revised in round 2): key = (seed low, seed high); counter = (index, t low,
 * t high, domain).
 * Domain SITE (XY, clock): one call per site and step, index = site; word k (k < dim) decides the
 * bond in direction k, word 3 is the draw of the cluster whose root (minimum site index) is this site.
 * Domain GROUP (Ising, Potts -- the two models whose bond probability is one constant): the 32
 * sites with linear index 32 G .. 32 G + 31 (group G = site / 32, position b = site % 32) share one
 * stream of words W_G[n], n = 0, 1, 2, ...:
 *     W_G[n] = word n % 4 of the call with counter (G, t low, t high, GROUP + 256 (n / 4)).
 *   W_G[0]               bit b: Ising, the new value of the cluster whose root is site b of the group
 *   W_G[1 + s dim + k]   bit b: bit 31 - s (s = 0 is the most significant) of the 32-bit uniform
 *                        integer u(site, k) that decides bond k of the site, s = 0 .. 31
 *   W_G[128 + b]         Potts: the draw word of site b of the group
 * i.e. the uniform integers of a group are stored transposed, one word per binary digit, so that a
 * comparison u < P32 can be carried out for 32 sites at once, most significant digit first, and
 * stopped as soon as every site is decided.  The decision itself is the plain one of reading 16:
 * a bond between aligned neighbours is active iff u < P32.
 * Domain INIT: start configuration, word 0.  Domain XYDIR: the XY direction of step t, word 0.
 * (Domains 1 and 4 belonged to the round-1 Ising keying and are retired.) */
enum { DOM_SITE = 0, DOM_INIT = 2, DOM_XYDIR = 3, DOM_GROUP = 5 };
enum { GROUP_DRAW_BASE = 128, GROUP_WORDS = 160 };

struct swo_ctx {
    int dim, L, model, q;
    double beta;
    uint64_t seed;
    uint64_t t;      /* index of the next step to execute */
    size_t N;
    int8_t *s_ising;   /* +-1          */
    uint8_t *s_potts;  /* 0..q-1       */
    float *s_xy;       /* angle theta  */
    uint16_t *s_clock; /* clock state p, theta = 2 pi p / q */
    int mirror;        /* clock: mirror index m of the last step */
    uint8_t *bond;     /* bit k = bond (i, i+e_k) active, last step */
    uint32_t *label;   /* min site index of the cluster, last step  */
    uint32_t *queue;   /* BFS work list */
    double *proj;      /* XY: a_i = r . s_i of the last step (double) */
    float rx, ry, crefl; /* XY: direction and reflection constant of the last step */
    int force_phi;
    double forced_phi;
    /* statistics of the last step's bond configuration */
    double n_active, n_clusters, sum_nc2;
    /* the words W_G[0 .. 32 dim] of the group make_bonds is working on */
    uint32_t gw[GROUP_WORDS];
};

static void draw(const swo_ctx *o, uint32_t site, uint64_t t, uint32_t domain, uint32_t w[4])
{
    uint32_t ctr[4] = { site, (uint32_t)(t & 0xffffffffu), (uint32_t)(t >> 32), domain };
    uint32_t key[2] = { (uint32_t)(o->seed & 0xffffffffu), (uint32_t)(o->seed >> 32) };
    swo_philox4x32_10(ctr, key, w);
}

/* Neighbour of site i in direction +k (periodic; "Periodic boundary conditions").
 * Reading 8: i = x + L*y (+ L*L*z), x fastest; each site owns its +x,+y,+z bonds. */
static size_t nbr_plus(const swo_ctx *o, size_t i, int k)
{
    size_t L = (size_t)o->L;
    size_t stride = 1;
    for (int a = 0; a < k; ++a) stride *= L;
    size_t coord = (i / stride) % L;
    return (coord == L - 1) ? i - (L - 1) * stride : i + stride;
}
static size_t nbr_minus(const swo_ctx *o, size_t i, int k)
{
    size_t L = (size_t)o->L;
    size_t stride = 1;
    for (int a = 0; a < k; ++a) stride *= L;
    size_t coord = (i / stride) % L;
    return (coord == 0) ? i + (L - 1) * stride : i - stride;
}

static const double TWO_PI = 6.283185307179586476925286766559;

/* Start configuration (the paper's device_function_spinset, contents unspecified,
 * PAPER.md:108-112).  Reading S3: seeded random start from domain INIT, word 0 = w:
 * Ising s = +1 if the top bit of w is set else -1; Potts s = (w*q) >> 32;
 * XY theta = float(w >> 8) * float(2 pi / 2^24). */
static void init_spins(swo_ctx *o)
{
    for (size_t i = 0; i < o->N; ++i) {
        uint32_t w[4];
        draw(o, (uint32_t)i, 0, DOM_INIT, w);
        if (o->model == SWO_ISING) o->s_ising[i] = (w[0] >> 31) ? 1 : -1;
        else if (o->model == SWO_POTTS) o->s_potts[i] = (uint8_t)(((uint64_t)w[0] * (uint64_t)o->q) >> 32);
        else if (o->model == SWO_CLOCK) o->s_clock[i] = (uint16_t)(((uint64_t)w[0] * (uint64_t)o->q) >> 32);
        else {
            float scale = (float)(TWO_PI / 16777216.0);
            o->s_xy[i] = (float)(w[0] >> 8) * scale;
        }
    }
}

swo_ctx *swo_create(int dim, int L, int model, int q, double beta, uint64_t seed)
{
    if (dim != 2 && dim != 3) return NULL;
    if (L < 3) return NULL; /* L = 2 would double every bond under periodic wrap */
    if (model != SWO_ISING && model != SWO_POTTS && model != SWO_XY && model != SWO_CLOCK) return NULL;
    if (model == SWO_POTTS && (q < 2 || q > 255)) return NULL;
    if (model == SWO_CLOCK && (q < 2 || q > 512)) return NULL; /* q <= 512 */
    if (!(beta >= 0.0) || !isfinite(beta)) return NULL;
    double Nd = pow((double)L, dim);
    if (Nd > 4294967295.0) return NULL;
    swo_ctx *o = (swo_ctx *)calloc(1, sizeof(*o));
    if (!o) return NULL;
    o->dim = dim; o->L = L; o->model = model; o->q = (model == SWO_POTTS || model == SWO_CLOCK) ? q : 0;
    o->beta = beta; o->seed = seed; o->t = 0;
    o->N = 1;
    for (int a = 0; a < dim; ++a) o->N *= (size_t)L;
    if (model == SWO_ISING) o->s_ising = (int8_t *)malloc(o->N);
    if (model == SWO_POTTS) o->s_potts = (uint8_t *)malloc(o->N);
    if (model == SWO_XY) { o->s_xy = (float *)malloc(o->N * sizeof(float)); o->proj = (double *)malloc(o->N * sizeof(double)); }
    if (model == SWO_CLOCK) { o->s_clock = (uint16_t *)malloc(o->N * sizeof(uint16_t)); o->proj = (double *)malloc(o->N * sizeof(double)); }
    o->bond = (uint8_t *)calloc(o->N, 1);
    o->label = (uint32_t *)malloc(o->N * sizeof(uint32_t));
    o->queue = (uint32_t *)malloc(o->N * sizeof(uint32_t));
    if (!o->bond || !o->label || !o->queue || (!o->s_ising && !o->s_potts && !o->s_xy && !o->s_clock) ||
        ((model == SWO_XY || model == SWO_CLOCK) && !o->proj)) { swo_destroy(o); return NULL; }
    for (size_t i = 0; i < o->N; ++i) o->label[i] = (uint32_t)i;
    init_spins(o);
    return o;
}

void swo_destroy(swo_ctx *o)
{
    if (!o) return;
    free(o->s_ising); free(o->s_potts); free(o->s_xy); free(o->s_clock); free(o->proj);
    free(o->bond); free(o->label); free(o->queue);
    free(o);
}

/* Threshold for the integer bond decision.  PAPER.md:96 prints "p = 1 e^{2J/T}" (minus signs
 * lost); reading 1: p = 1 - exp(-2J/T) for Eq. (1).  Potts (Eq. 2): reading 2:
 * p = 1 - exp(-J/T).  Reading 16: a bond is active iff word < floor(p * 2^32) (clamped). */
static uint32_t threshold32(double p)
{
    double v = floor(p * 4294967296.0);
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

/* Reading 6, domain GROUP: word n of the stream of group G at step t. */
static uint32_t group_word(const swo_ctx *o, uint32_t G, uint64_t t, uint32_t n)
{
    uint32_t w[4];
    draw(o, G, t, (uint32_t)DOM_GROUP + 256u * (n >> 2), w);
    return w[n & 3u];
}

/* The words W_G[0 .. 32 dim] (draw bits and the 32 binary digits of every bond's uniform integer)
 * of group G, four per Philox call. */
static void group_fill(swo_ctx *o, uint32_t G, uint64_t t)
{
    const uint32_t nwords = 1u + 32u * (uint32_t)o->dim;
    for (uint32_t c = 0; 4u * c < nwords; ++c) draw(o, G, t, (uint32_t)DOM_GROUP + 256u * c, &o->gw[4u * c]);
}

/* u(site, k): digit s (bit 31 - s) is bit b of W_G[1 + s dim + k]. */
static uint32_t group_uniform(const swo_ctx *o, uint32_t b, int k)
{
    uint32_t u = 0;
    for (int s = 0; s < 32; ++s) u |= ((o->gw[1 + s * o->dim + k] >> b) & 1u) << (31 - s);
    return u;
}

/* Sub-step (1): active-bond generation. */
static void make_bonds(swo_ctx *o)
{
    const uint64_t t = o->t;
    double nact = 0.0;
    if (o->model == SWO_ISING || o->model == SWO_POTTS) {
        /* PAPER.md:96 (Ising), PAPER.md:152 + Eq. 2 (Potts): a bond between equal neighbours is active
         * with probability p; readings 1, 2, 16: active iff u(site, k) < floor(p 2^32). */
        const uint32_t P32 = threshold32(o->model == SWO_ISING ? -expm1(-2.0 * o->beta) : -expm1(-o->beta));
        for (size_t i = 0; i < o->N; ++i) {
            if ((i & 31u) == 0) group_fill(o, (uint32_t)(i >> 5), t);
            uint8_t b = 0;
            for (int k = 0; k < o->dim; ++k) {
                size_t j = nbr_plus(o, i, k);
                int equal = (o->model == SWO_ISING) ? (o->s_ising[i] == o->s_ising[j]) : (o->s_potts[i] == o->s_potts[j]);
                if (equal && group_uniform(o, (uint32_t)(i & 31u), k) < P32) {
                    b |= (uint8_t)(1u << k);
                    nact += 1.0;
                }
            }
            o->bond[i] = b;
        }
    } else if (o->model == SWO_CLOCK) {
        /* q-state clock model (theta = 2 pi p / q; "The variable ispr, which
         * is randomly chosen, specifies the direction for mirror projection").  Readings 23-25
         * (DESIGN.md): the mirror index m = (word * q) >> 32 from the XYDIR call of the step; the
         * mirror axis lies at angle pi m / q, so the reflection p -> (m - p) mod q maps clock states to
         * clock states; the embedded Ising variable is the component along the normal of the axis,
         * a(p) = sin(pi (2p - m) / q).  Written with k = (2p - m) mod 2q, u = k mod q:
         * a = +sin(pi u / q) for k < q and -sin(pi u / q) for k >= q (zero for u = 0).  A bond between
         * neighbours whose components have the same sign is active with
         * p = 1 - exp(-2 beta a_i a_j), decided as word < floor(p 2^32) like Ising / Potts. */
        uint32_t w[4];
        const int q = o->q;
        draw(o, 0, t, DOM_XYDIR, w);
        const int m = (int)(((uint64_t)w[0] * (uint64_t)q) >> 32);
        o->mirror = m;
        for (size_t i = 0; i < o->N; ++i) {
            int k = (2 * (int)o->s_clock[i] - m) % (2 * q);
            if (k < 0) k += 2 * q;
            int u = k % q;
            double mag = sin((TWO_PI / 2.0) * (double)u / (double)q);
            o->proj[i] = (u == 0) ? 0.0 : (k < q ? mag : -mag);
        }
        for (size_t i = 0; i < o->N; ++i) {
            draw(o, (uint32_t)i, t, DOM_SITE, w);
            uint8_t b = 0;
            for (int k = 0; k < o->dim; ++k) {
                size_t j = nbr_plus(o, i, k);
                double ai = o->proj[i], aj = o->proj[j];
                if ((ai > 0.0 && aj > 0.0) || (ai < 0.0 && aj < 0.0)) {
                    double prod = fabs(ai) * fabs(aj);
                    uint32_t P32 = threshold32(-expm1(-2.0 * o->beta * prod));
                    if (w[k] < P32) { b |= (uint8_t)(1u << k); nact += 1.0; }
                }
            }
            o->bond[i] = b;
        }
    } else {
        /* XY: "we project vector spins to form Ising spin clusters" (Wolff's
         * embedding).  Reading 3: with a_i = r . s_i, a bond between neighbours whose projections
         * have the same sign is active with p = 1 - exp(-2 beta a_i a_j).  Reading 20: the
         * direction r = (cos phi, sin phi), phi uniform from one XYDIR word, rounded to fp32. */
        uint32_t w[4];
        draw(o, 0, t, DOM_XYDIR, w);
        double phi = (double)w[0] * (TWO_PI / 4294967296.0);
        if (o->force_phi) phi = o->forced_phi;
        o->rx = (float)cos(phi);
        o->ry = (float)sin(phi);
        o->crefl = (float)fmod(2.0 * phi + TWO_PI / 2.0, TWO_PI);
        for (size_t i = 0; i < o->N; ++i) {
            double th = (double)o->s_xy[i];
            o->proj[i] = (double)o->rx * cos(th) + (double)o->ry * sin(th);
        }
        for (size_t i = 0; i < o->N; ++i) {
            draw(o, (uint32_t)i, t, DOM_SITE, w);
            uint8_t b = 0;
            for (int k = 0; k < o->dim; ++k) {
                size_t j = nbr_plus(o, i, k);
                double prod = o->proj[i] * o->proj[j];
                double u = (double)(w[k] >> 8) * (1.0 / 16777216.0);
                if (prod > 0.0 && u < -expm1(-2.0 * o->beta * prod)) { b |= (uint8_t)(1u << k); nact += 1.0; }
            }
            o->bond[i] = b;
        }
    }
    o->n_active = nact;
}

/* Sub-step (2): "The active bonds partition the spins into clusters".  Breadth-first
 * search over active bonds, start sites in increasing index: the first unvisited site of a
 * component is its minimum index and becomes the label of every site reached (reading 7: the
 * label a label-equivalence run with atomicMin from label = index converges to). */
static void label_clusters(swo_ctx *o)
{
    const uint32_t UNSEEN = 0xffffffffu;
    double nclus = 0.0, snc2 = 0.0;
    for (size_t i = 0; i < o->N; ++i) o->label[i] = UNSEEN;
    for (size_t start = 0; start < o->N; ++start) {
        if (o->label[start] != UNSEEN) continue;
        size_t head = 0, tail = 0;
        o->queue[tail++] = (uint32_t)start;
        o->label[start] = (uint32_t)start;
        double sum_a = 0.0;
        while (head < tail) {
            size_t i = o->queue[head++];
            if (o->model == SWO_XY || o->model == SWO_CLOCK) sum_a += o->proj[i];
            for (int k = 0; k < o->dim; ++k) {
                if (o->bond[i] & (1u << k)) {
                    size_t j = nbr_plus(o, i, k);
                    if (o->label[j] == UNSEEN) { o->label[j] = (uint32_t)start; o->queue[tail++] = (uint32_t)j; }
                }
                size_t m = nbr_minus(o, i, k);
                if (o->bond[m] & (1u << k)) {
                    if (o->label[m] == UNSEEN) { o->label[m] = (uint32_t)start; o->queue[tail++] = (uint32_t)m; }
                }
            }
        }
        nclus += 1.0;
        snc2 += (o->model == SWO_XY || o->model == SWO_CLOCK) ? sum_a * sum_a : (double)tail * (double)tail;
    }
    o->n_clusters = nclus;
    o->sum_nc2 = snc2;
}

/* Sub-step (3): "All spins in each cluster are set randomly to +1 or -1" (reading
 * 5: a fresh value, not "flip with probability 1/2").  One draw per cluster at its root (reading 6):
 * Ising the root's bit of W_G[0]; Potts the root's draw word w = W_G[128 + b], new state (w*q) >> 32;
 * XY and clock the top bit of word 3 of the root's SITE call.  XY (mirror
 * projection): if the top bit is set, reflect every spin of the cluster across the line
 * perpendicular to r: theta' = c - theta with c = (2 phi + pi) mod 2 pi, wrapped to [0, 2 pi]
 * -- two fp32 operations, done in float here exactly as the spec states them. */
static void flip_clusters(swo_ctx *o)
{
    const uint64_t t = o->t;
    const float two_pi_f = (float)TWO_PI;
    for (size_t i = 0; i < o->N; ++i) {
        uint32_t w[4];
        const uint32_t root = o->label[i];
        if (o->model == SWO_ISING) {
            o->s_ising[i] = ((group_word(o, root >> 5, t, 0) >> (root & 31u)) & 1u) ? 1 : -1;
            continue;
        }
        if (o->model == SWO_POTTS) {
            const uint32_t wd = group_word(o, root >> 5, t, (uint32_t)GROUP_DRAW_BASE + (root & 31u));
            o->s_potts[i] = (uint8_t)(((uint64_t)wd * (uint64_t)o->q) >> 32);
            continue;
        }
        draw(o, root, t, DOM_SITE, w);
        if (o->model == SWO_CLOCK) {
            /* mirror projection of the whole cluster with probability 1/2: p -> (m - p) mod q */
            if (w[3] >> 31) {
                int pn = (o->mirror - (int)o->s_clock[i]) % o->q;
                if (pn < 0) pn += o->q;
                o->s_clock[i] = (uint16_t)pn;
            }
            continue;
        }
        if (w[3] >> 31) {
            float th = o->crefl - o->s_xy[i];
            if (th < 0.0f) th = th + two_pi_f;
            o->s_xy[i] = th;
        }
    }
}

int swo_step(swo_ctx *o, int n)
{
    if (!o || n < 0) return -1;
    for (int s = 0; s < n; ++s) {
        make_bonds(o);
        label_clusters(o);
        flip_clusters(o);
        o->t += 1;
    }
    return 0;
}

/* Exact integer sums.  Ising: E = -sum_<ij> s_i s_j (Eq. 1, J = 1), M = sum_i s_i (Eq. 4).
 * Potts: E = -sum_<ij> (delta - 1) = number of unequal nearest-neighbour pairs (Eq. 2, J = 1),
 * n[k] = number of spins in state k (Eq. 5). */
int swo_counts(const swo_ctx *o, int64_t *E_int, int64_t *M_or_nk, int n)
{
    if (!o || o->model == SWO_XY || o->model == SWO_CLOCK) return -1;
    int64_t E = 0;
    if (o->model == SWO_ISING) {
        int64_t M = 0;
        for (size_t i = 0; i < o->N; ++i) {
            M += o->s_ising[i];
            for (int k = 0; k < o->dim; ++k) E -= (int64_t)o->s_ising[i] * o->s_ising[nbr_plus(o, i, k)];
        }
        if (M_or_nk && n >= 1) M_or_nk[0] = M;
    } else {
        for (int k = 0; k < n && M_or_nk; ++k) M_or_nk[k] = 0;
        for (size_t i = 0; i < o->N; ++i) {
            if (M_or_nk && o->s_potts[i] < n) M_or_nk[o->s_potts[i]] += 1;
            for (int k = 0; k < o->dim; ++k) E += (o->s_potts[i] != o->s_potts[nbr_plus(o, i, k)]);
        }
    }
    if (E_int) *E_int = E;
    return 0;
}

/* PAPER.md:142-157 and Eq. (1)-(5); conventions in DESIGN.md readings 11-14:
 * Ising M signed, M2 = M^2, M4 = M^4.  Potts M2 = (q sum n_k^2 - N^2)/(q-1) (Eq. 5),
 * M = sqrt(M2), M4 = M2^2.  XY E = -sum cos(theta_i - theta_j) (Eq. 3), M = |sum s_i|. */
void swo_observables(const swo_ctx *o, double *E, double *M, double *M2, double *M4)
{
    double e = 0.0, m = 0.0, m2 = 0.0;
    if (o->model == SWO_ISING) {
        int64_t Ei, Mi;
        swo_counts(o, &Ei, &Mi, 1);
        e = (double)Ei; m = (double)Mi; m2 = m * m;
    } else if (o->model == SWO_POTTS) {
        int64_t Ei, nk[256];
        swo_counts(o, &Ei, nk, o->q);
        double s2 = 0.0;
        for (int k = 0; k < o->q; ++k) s2 += (double)nk[k] * (double)nk[k];
        double Nd = (double)o->N;
        e = (double)Ei; m2 = ((double)o->q * s2 - Nd * Nd) / (double)(o->q - 1); m = sqrt(m2);
    } else if (o->model == SWO_CLOCK) {
        /* Eq. (3) with theta = 2 pi p / q, from the exact integer histograms (the paper's tables
         * rule[] and fmy[]): E = -sum_d D[d] cos(2 pi d / q),
         * M = | sum_p n[p] (cos, sin)(2 pi p / q) |, summed in increasing d and p. */
        int64_t D[512], nn[512];
        swo_clock_hist(o, D, nn, o->q);
        double mx = 0.0, my = 0.0;
        for (int d = 0; d < o->q; ++d) e -= (double)D[d] * cos(TWO_PI * (double)d / (double)o->q);
        for (int pp = 0; pp < o->q; ++pp) {
            mx += (double)nn[pp] * cos(TWO_PI * (double)pp / (double)o->q);
            my += (double)nn[pp] * sin(TWO_PI * (double)pp / (double)o->q);
        }
        m2 = mx * mx + my * my; m = sqrt(m2);
    } else {
        double mx = 0.0, my = 0.0;
        for (size_t i = 0; i < o->N; ++i) {
            double th = (double)o->s_xy[i];
            mx += cos(th); my += sin(th);
            for (int k = 0; k < o->dim; ++k) e -= cos(th - (double)o->s_xy[nbr_plus(o, i, k)]);
        }
        m2 = mx * mx + my * my; m = sqrt(m2);
    }
    if (E) *E = e;
    if (M) *M = m;
    if (M2) *M2 = m2;
    if (M4) *M4 = m2 * m2;
}

int swo_clock_hist(const swo_ctx *o, int64_t *D, int64_t *n, int q)
{
    if (!o || o->model != SWO_CLOCK || q != o->q) return -1;
    for (int k = 0; k < q; ++k) { if (D) D[k] = 0; if (n) n[k] = 0; }
    for (size_t i = 0; i < o->N; ++i) {
        int pi_ = (int)o->s_clock[i];
        if (n) n[pi_] += 1;
        for (int k = 0; k < o->dim && D; ++k) {
            int d = (pi_ - (int)o->s_clock[nbr_plus(o, i, k)]) % q;
            if (d < 0) d += q;
            D[d] += 1;
        }
    }
    return 0;
}

int swo_get_clock_mirror(const swo_ctx *o, int *m)
{
    if (!o || o->model != SWO_CLOCK) return -1;
    if (m) *m = o->mirror;
    return 0;
}

size_t swo_num_sites(const swo_ctx *o) { return o ? o->N : 0; }
uint64_t swo_step_index(const swo_ctx *o) { return o ? o->t : 0; }

static size_t spin_bytes(const swo_ctx *o)
{
    return o->model == SWO_XY ? o->N * sizeof(float) : o->model == SWO_CLOCK ? o->N * sizeof(uint16_t) : o->N;
}
static void *spin_ptr(const swo_ctx *o)
{
    return o->model == SWO_ISING ? (void *)o->s_ising : o->model == SWO_POTTS ? (void *)o->s_potts
         : o->model == SWO_CLOCK ? (void *)o->s_clock : (void *)o->s_xy;
}

int swo_get_spins(const swo_ctx *o, void *dst, size_t bytes)
{
    if (!o || !dst || bytes != spin_bytes(o)) return -1;
    memcpy(dst, spin_ptr(o), bytes);
    return 0;
}
int swo_set_spins(swo_ctx *o, const void *src, size_t bytes, uint64_t step)
{
    if (!o || !src || bytes != spin_bytes(o)) return -1;
    memcpy(spin_ptr(o), src, bytes);
    o->t = step;
    return 0;
}
int swo_get_bonds(const swo_ctx *o, uint8_t *dst, size_t bytes)
{
    if (!o || !dst || bytes != o->N) return -1;
    memcpy(dst, o->bond, bytes);
    return 0;
}
int swo_get_labels(const swo_ctx *o, uint32_t *dst, size_t bytes)
{
    if (!o || !dst || bytes != o->N * sizeof(uint32_t)) return -1;
    memcpy(dst, o->label, bytes);
    return 0;
}
int swo_get_xy_dir(const swo_ctx *o, float *rx, float *ry, float *c)
{
    if (!o || o->model != SWO_XY) return -1;
    if (rx) *rx = o->rx;
    if (ry) *ry = o->ry;
    if (c) *c = o->crefl;
    return 0;
}
int swo_force_xy_phi(swo_ctx *o, int enable, double phi)
{
    if (!o || o->model != SWO_XY) return -1;
    o->force_phi = enable; o->forced_phi = phi;
    return 0;
}

int swo_run_series(swo_ctx *o, int n, double *E, double *M, double *M2, double *n_active,
                   double *n_clusters, double *sum_nc2)
{
    if (!o || n < 0) return -1;
    for (int s = 0; s < n; ++s) {
        swo_step(o, 1);
        double e, m, m2, m4;
        swo_observables(o, &e, &m, &m2, &m4);
        if (E) E[s] = e;
        if (M) M[s] = m;
        if (M2) M2[s] = m2;
        if (n_active) n_active[s] = o->n_active;
        if (n_clusters) n_clusters[s] = o->n_clusters;
        if (sum_nc2) sum_nc2[s] = o->sum_nc2;
    }
    return 0;
}
