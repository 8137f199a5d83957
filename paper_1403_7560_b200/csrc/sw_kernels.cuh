// sw_kernels.cuh -- CUDA kernels (sm_100a) of one Swendsen-Wang step, arXiv 1403.7560 section 2
// (PAPER.md:94-98).  Independent of oracle/: nothing here is shared with or derived from it.
//
// Kernels of one step t:
//   k_bond_label_rows (sw_rows.cuh; Ising, Potts, clock)  /  k_bond_label (here; XY: the round-1 "quad" kernel)
//                 (1) bond activation fused with (2a) tile-local cluster labelling in shared
//                 memory; bonds through tile faces go to a global pair list.  In k_bond_label a thread owns
//                 "quads" of 4 consecutive sites along x; x-connectivity is resolved with two warp ballots,
//                 y/z bonds inside the tile by a CAS hook round, pointer jumping and an atomicMin union-find;
//   k_merge       (2b) global lock-free union-find (atomicCAS, min linear index wins) over the active
//                 bonds that cross tile faces incl. the periodic wrap;
//   k_flip        (2c) root chase fused with (3) the per-cluster new value / XY reflection
//                  and the magnetisation sums of PAPER.md:142-157;
//   k_measure4 / k_measure_xy / k_measure_clock   energy (Eq. 1-3) and magnetisation (Eq. 4, 5) of the
//                 current configuration, on request (sw_observables, sw_run_series);
//   k_sw_small (sw_small.cuh)  all of the above in one CTA for lattices of at most 32768 Ising / Potts sites.
// Models: Ising, q-state Potts, continuous XY, q-state clock (the discretisation the paper runs).
//
// Label array (HBM), one 32-bit word per site, TILE-MAJOR: the word of the site with tile-local
// index li = lx + TX (ly + TY lz) in tile T lives at address a = T * NS + li, and holds
//     (parent address << DB) | (the site's own cluster draw, DB bits, from its Philox call).
// A site is a root iff parent address == own address.  Hooking always puts the root with the larger
// LINEAR site index under the one with the smaller, so the final root of a cluster is its minimum
// linear site index (what label equivalence with atomicMin from label = index converges to,
// PAPER.md:102), and the cluster's new value is simply the draw field of the root's word.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// XY arithmetic (reading 20): the projections r . s_i and the bond probabilities 1 - exp(-2 beta a_i a_j)
// are evaluated with the SFU intrinsics __sincosf / __expf.  Measured against the fp64 oracle on 7.0e8 bonds
// (3D L = 256, T = 2.2019, 14 injected steps): 43 mismatching bonds = 6.1e-8 per bond, 16 x below north_star's
// budget of 1e-6 (full-precision sincosf / expm1f: 2 of 4.0e8 = 5e-9); what decides a bond is the ABSOLUTE error
// of p, about 1e-7 for the intrinsics on angles in [0, 2 pi].  SW_XY_FAST_MATH=0 builds the full-precision path.
#ifndef SW_XY_FAST_MATH
#define SW_XY_FAST_MATH 1
#endif
#if SW_XY_FAST_MATH
#define SW_SINCOSF(x, s, c) __sincosf((x), (s), (c))
// 1 - exp(x) for x <= 0 (x = -2 beta a_i a_j): __expf is ex2.approx(x log2 e) plus a rescaling for results below 2^-126, which
// 1 - r rounds to 1.0f either way; the .ftz form of the same SFU instruction gives the same bits without the rescaling.
__device__ __forceinline__ float sw_exp_le0(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x * 1.4426950408889634f));
    return r;
}
#define SW_NEG_EXPM1F(x) (1.0f - sw_exp_le0(x))
#else
#define SW_SINCOSF(x, s, c) sincosf((x), (s), (c))
#define SW_NEG_EXPM1F(x) (-expm1f(x))
#endif

namespace swk {

enum { ISING = 0, POTTS = 1, XY = 2, CLOCK = 3 };
constexpr uint32_t DOM_SITE = 0u, DOM_INIT = 2u, DOM_XYDIR = 3u, DOM_GROUP = 5u;  // DESIGN.md reading 6
constexpr uint32_t FULL = 0xffffffffu;
#ifndef SW_BL_THREADS_PER_SM
#define SW_BL_THREADS_PER_SM 1536  // resident threads per SM k_bond_label is compiled for (register cap)
#endif
#ifndef SW_BL_ROUNDS
#define SW_BL_ROUNDS 1  // uniform hook + flatten rounds before the general union-find loop
#endif
#ifndef SW_BL_HOOK_LOOP
#define SW_BL_HOOK_LOOP 1  // 3D hook round: 1 = loop over the active bonds, 0 = predicated code over all bond slots
#endif
#ifndef SW_BL_MIDJUMPS
#define SW_BL_MIDJUMPS 2  // pointer-jumping steps after a hook round
#endif
#ifndef SW_BL_JUMPS
#define SW_BL_JUMPS 2  // pointer-jumping rounds over the tile-local forest before it is stored
#endif

// Device accumulators of the observables and the labelling counters.
struct Acc {
    unsigned long long E_int;    // Ising: -sum s_i s_j (two's complement); Potts: #unequal pairs
    double E_xy;                 // XY: -sum cos(theta_i - theta_j)
    unsigned long long M_int;    // Ising: sum s_i (two's complement)
    double mx, my;               // XY: sum cos, sum sin
    unsigned long long nk[512];  // Potts: n_k (q <= 255); clock: number of sites in state p (q <= 512)
    unsigned long long dk[512];  // clock: number of nearest-neighbour pairs with (p_i - p_j) mod q = d
    unsigned long long stats[8]; // see sw_get_label_stats
    uint32_t npairs;             // length of the pair list of the current step
    unsigned long long t;        // index of the step being executed: read by k_bond_label, advanced by
                                 // k_flip, so a step's launches carry no per-step argument (CUDA graphs)
};

struct Params {
    void *spins;            // int8 (Ising) | uint8 (Potts) | float (XY angle), N elements, linear order
    uint8_t *bonds;         // N bytes, bit k = bond i -> i + e_k, linear order; NULL = not recorded
    uint32_t *labels;       // N packed parent words, tile-major (see above)
    uint2 *pairs;           // compact list of the active bonds through tile faces: (address i, address j)
    uint32_t *npairs;       // its length (reset by k_flip for the next step)
    uint32_t *tile_origin;  // per tile: linear index of its first site
    uint32_t *labels_out;   // k_export_labels: N canonical labels (minimum linear index), linear order
    Acc *acc;
    uint32_t L, N;
    uint32_t ntx, nty, ntz, ntiles;
    uint32_t k0, k1;   // Philox key = (seed low, seed high)
    uint32_t rk[20];   // its ten round keys (k0 + r 0x9E3779B9, k1 + r 0xBB67AE85), r = 0..9: constant-bank operands for the per-site generator
    uint32_t P32;      // Ising/Potts: bond active iff word < P32
    int q;
    int db;            // draw bits in a label word: 1 (Ising, XY), ceil(log2 q) (Potts)
    float rx, ry, crefl, m2beta;  // XY: direction, reflection constant, -2 beta
    const uint32_t *clock_T;      // clock: q x q bond thresholds T[u_i q + u_j] (see k_bond_label)
    int mirror;                   // clock: mirror index m of the step (the paper's ispr)
    int counting;
    int nk_clear;                 // number of n_k accumulators k_merge clears for k_flip (Potts: q, else 0)
};

// Philox4x32-10 (Salmon et al., SC'11): 10 rounds of two 32x32->64 multiplies and a key bump.
__host__ __device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                        uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long a = 0xD2511F53ull * c0;
        const unsigned long long b = 0xCD9E8D57ull * c2;
        const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)b;
        c3 = (uint32_t)a;
        c0 = n0;
        c2 = n2;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return make_uint4(c0, c1, c2, c3);
}

// The same numbers with the round keys read from the kernel parameters (constant bank): a loop that makes one call per
// iteration (XY, clock: one call per site) otherwise redoes the 18 key additions in every iteration.
__device__ __forceinline__ uint4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const Params &p)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long a = 0xD2511F53ull * c0;
        const unsigned long long b = 0xCD9E8D57ull * c2;
        const uint32_t n0 = (uint32_t)(b >> 32) ^ c1 ^ p.rk[2 * r];
        const uint32_t n2 = (uint32_t)(a >> 32) ^ c3 ^ p.rk[2 * r + 1];
        c1 = (uint32_t)b;
        c3 = (uint32_t)a;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ void decode(const Params &p, uint32_t i, uint32_t &x, uint32_t &y, uint32_t &z)
{
    x = i % p.L;
    const uint32_t r = i / p.L;
    y = r % p.L;
    z = r / p.L;
}

constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v / 2); }

// Geometry of a TX x TY x TZ tile (powers of two; TX a multiple of 32).
template <int DIM, int TX, int TY, int TZ>
struct TileGeom {
    static constexpr int NS = TX * TY * TZ;
    static constexpr int LOG2NS = ilog2(NS);
    static_assert((1 << LOG2NS) == NS, "tile sizes are powers of two");
    static_assert(TX % 32 == 0 && TX <= 128, "a tile row is 8, 16 or 32 quads");
    static_assert(DIM == 3 || TZ == 1, "2D tiles have TZ = 1");
    // face bit fields: +x face TY*TZ bonds, +y face TX*TZ bonds, +z face TX*TY bonds
    static constexpr int FXB = TY * TZ, FYB = TX * TZ, FZB = (DIM == 3) ? TX * TY : 0;
    static constexpr int FXW = (FXB + 31) / 32, FYW = (FYB + 31) / 32, FZW = (FZB + 31) / 32;
    static constexpr int NFW = FXW + FYW + FZW;
    static constexpr int NFWP = (NFW + 3) / 4 * 4;  // padded: what follows in smem stays 16-byte aligned
    static constexpr int NHALO = FXB + FYB + FZB;  // XY: projections of the three plus-faces
    // smem of k_bond_label (32-bit words): labels, face bit words, their popcount prefix (+ list base,
    // + leftover count), the list of leftover unions (16-bit entries), XY projections
    static constexpr int LEFT_CAP = NS / 4;
    static constexpr int OFF_FACE = NS, OFF_FPRE = NS + NFWP, OFF_LEFT = NS + 2 * NFWP + 4;
    static constexpr int OFF_VAL = OFF_LEFT + LEFT_CAP / 2;
    template <int MODEL> static constexpr size_t smem_bond_label()
    {
        return (size_t)OFF_VAL * 4 + (MODEL == XY ? ((size_t)NS + NHALO) * 4 : 0);
    }
};

// 4-bit mask of the byte positions where a and b hold equal bytes.
__device__ __forceinline__ uint32_t eq4(uint32_t a, uint32_t b)
{
    const uint32_t t = a ^ b;
    const uint32_t z = ~(((t & 0x7f7f7f7fu) + 0x7f7f7f7fu) | t | 0x7f7f7f7fu);  // 0x80 per zero byte
    return (((z >> 7) * 0x00204081u) >> 21) & 0xfu;
}
// bit s of a nibble -> bit 0 of byte s
__device__ __forceinline__ uint32_t spread4(uint32_t n) { return (n * 0x00204081u) & 0x01010101u; }

// ------------------------------------------------------------------------------------------------
// Shared-memory union-find (min-index roots).  Every link hangs the larger root under the smaller
// one, so the root of a finished tree is the minimum index of its set whatever the order in which
// concurrent unions land.  Tile-local indices are monotone in the linear site index.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void union_s(uint32_t *lab, uint32_t a, uint32_t b)
{
    for (;;) {
        {   // both chains in one loop: trip count max(hops a, hops b) instead of the sum, two loads in flight
            volatile uint32_t *vl = lab;
            uint32_t pa = vl[a], pb = vl[b];
            while (pa != a || pb != b) {
                a = pa; b = pb;
                pa = vl[a]; pb = vl[b];
            }
        }
        if (a == b) return;
        if (a < b) { const uint32_t t = a; a = b; b = t; }
        const uint32_t old = atomicMin(&lab[a], b);
        if (old == a) return;  // a was a root and now hangs under b
        a = old;               // a had been linked meanwhile: go on with (old parent, b)
    }
}


// One pointer-jumping step for the 4 sites of a quad: r <- parent(r) where the previous step still
// moved (r != prev); a site that has reached a fixed point (a root) issues no load, so roots and
// their direct children cost no shared-memory wavefronts.
__device__ __forceinline__ void jump4(volatile uint32_t *vl, uint4 &r, uint4 &prev)
{
    uint4 n;
    n.x = (r.x != prev.x) ? vl[r.x] : r.x;
    n.y = (r.y != prev.y) ? vl[r.y] : r.y;
    n.z = (r.z != prev.z) ? vl[r.z] : r.z;
    n.w = (r.w != prev.w) ? vl[r.w] : r.w;
    prev = r;
    r = n;
}

// ------------------------------------------------------------------------------------------------
// k_init: seeded random start (the paper's device_function_spinset).
// ------------------------------------------------------------------------------------------------
template <int MODEL>
__global__ void __launch_bounds__(256) k_init(const Params p)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= p.N) return;
    const uint32_t w = philox4x32_10(i, 0u, 0u, DOM_INIT, p.k0, p.k1).x;
    if (MODEL == ISING) ((int8_t *)p.spins)[i] = (w >> 31) ? 1 : -1;
    else if (MODEL == POTTS) ((uint8_t *)p.spins)[i] = (uint8_t)(((unsigned long long)w * (unsigned)p.q) >> 32);
    else if (MODEL == CLOCK) ((uint16_t *)p.spins)[i] = (uint16_t)(((unsigned long long)w * (unsigned)p.q) >> 32);
    else ((float *)p.spins)[i] = (float)(w >> 8) * (float)(6.283185307179586476925286766559 / 16777216.0);
}

// tile_origin[T] = linear index of the first site of tile T (T = tx + ntx (ty + nty tz)).
template <int TX, int TY, int TZ>
__global__ void __launch_bounds__(256) k_tile_origin(const Params p)
{
    const uint32_t T = blockIdx.x * 256u + threadIdx.x;
    if (T >= p.ntiles) return;
    const uint32_t tx = T % p.ntx, r = T / p.ntx, ty = r % p.nty, tz = r / p.nty;
    p.tile_origin[T] = tx * TX + p.L * (ty * TY + p.L * (tz * TZ));
}

// ------------------------------------------------------------------------------------------------
// k_bond_label: one CTA per tile, QPT quads per thread.
//   phase 0 (XY)  projections a_i = r . s_i of the tile and its three plus-faces into smem
//   phase 1       per quad: spins of the quad and of its +x/+y/+z neighbours, the Philox call(s)
//                 (reading 6), bond nibbles; two ballots give every site the
//                 start of its x-run; label_s[site] = run start; face bonds -> face bit words
//   phase 2a      hook round over the thread's active y/z bonds: CAS(larger root -> smaller root),
//                 failures stay pending; two pointer-jumping steps
//   phase 2b      pending bonds compacted into one list, handled by the general atomicMin union-find
//   phase 3       two more jumping steps, label word = (address of the parent << DB) | own draw with
//                 16-byte stores; active face bonds appended to the global pair list
// ------------------------------------------------------------------------------------------------
template <int DIM, int MODEL, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT, SW_BL_THREADS_PER_SM / NT) k_bond_label(const Params p)
{
    static_assert(MODEL == XY || MODEL == CLOCK, "Ising and Potts run k_bond_label_rows (sw_rows.cuh)");
    using G = TileGeom<DIM, TX, TY, TZ>;
    constexpr int NS = G::NS, NQ = NS / 4, QPT = NQ / NT, LPR = TX / 4;
    static_assert(NQ % NT == 0 && NT % 32 == 0, "whole quads per thread, whole rows per warp");
    static_assert(QPT * 4 <= 32, "the pending y bonds (and the pending z bonds) of a thread are one 32-bit mask");
    extern __shared__ __align__(16) uint32_t smem_u32[];
    static_assert(G::NFW <= 64, "two face words per lane of warp 0");
    static_assert(NS <= 32768, "a leftover entry keeps the site in 15 bits");
    uint32_t *lab_s = smem_u32;
    uint32_t *face_s = smem_u32 + G::OFF_FACE;
    uint32_t *fpre_s = smem_u32 + G::OFF_FPRE;  // NFW prefix counts, [NFWP] = base in the global list, [NFWP+1] = #leftovers, [NFWP+2] = valid part of their list
    uint16_t *left_s = reinterpret_cast<uint16_t *>(smem_u32 + G::OFF_LEFT);
    float *val_s = reinterpret_cast<float *>(smem_u32 + G::OFF_VAL);  // XY only: NS + NHALO floats

    const uint32_t L = p.L;
    const uint32_t bx = blockIdx.x, by = blockIdx.y, bz = (DIM == 3) ? blockIdx.z : 0u;
    const uint32_t x0 = bx * TX, y0 = by * TY, z0 = bz * TZ;
    const uint32_t tile = bx + p.ntx * (by + p.nty * bz);
    const uint32_t tile_base = tile << G::LOG2NS;
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t LL = L * L;
    const unsigned long long t_step = p.acc->t;
    const uint32_t t_lo = (uint32_t)t_step, t_hi = (uint32_t)(t_step >> 32);

    if (tid < G::NFW) face_s[tid] = 0u;
    if (tid == 0) { fpre_s[G::NFWP + 1] = 0u; fpre_s[G::NFWP + 2] = (uint32_t)G::LEFT_CAP; }

    if (MODEL == XY) {
        // a_i = r . s_i: interior, then the +x, +y, +z faces (periodic wrap)
        const float *th = (const float *)p.spins;
#pragma unroll
        for (int j = 0; j < QPT; ++j) {
            const int li = (tid + j * NT) * 4;
            const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
            const uint32_t g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
            const float4 t4 = *reinterpret_cast<const float4 *>(th + g);
            float4 a;
            float sn, cs;
            SW_SINCOSF(t4.x, &sn, &cs); a.x = p.rx * cs + p.ry * sn;
            SW_SINCOSF(t4.y, &sn, &cs); a.y = p.rx * cs + p.ry * sn;
            SW_SINCOSF(t4.z, &sn, &cs); a.z = p.rx * cs + p.ry * sn;
            SW_SINCOSF(t4.w, &sn, &cs); a.w = p.rx * cs + p.ry * sn;
            *reinterpret_cast<float4 *>(val_s + li) = a;
        }
        for (int h = tid; h < G::NHALO; h += NT) {
            uint32_t gx, gy, gz;
            if (h < G::FXB) {
                gx = x0 + TX; gy = y0 + h % TY; gz = z0 + h / TY;
            } else if (h < G::FXB + G::FYB) {
                const int k = h - G::FXB;
                gx = x0 + k % TX; gy = y0 + TY; gz = z0 + k / TX;
            } else {
                const int k = h - G::FXB - G::FYB;
                gx = x0 + k % TX; gy = y0 + k / TX; gz = z0 + TZ;
            }
            if (gx == L) gx = 0;
            if (gy == L) gy = 0;
            if (DIM == 3 && gz == L) gz = 0;
            float sn, cs;
            SW_SINCOSF(th[gx + L * (gy + L * gz)], &sn, &cs);
            val_s[NS + h] = p.rx * cs + p.ry * sn;
        }
    }
    __syncthreads();

    uint32_t bnd[QPT];   // per quad: bits 0-3 x bonds, 4-7 y bonds, 8-11 z bonds, 12-15 the four 1-bit draws
    // pending bonds that stay inside the tile: bit 4 j + s = site s of the thread's quad j, one mask for
    // the y bonds and one for the z bonds (32-bit masks, and the neighbour offset is a constant per mask)
    uint32_t work[2] = {0u, 0u};
    constexpr int db = 1;

#pragma unroll
    for (int j = 0; j < QPT; ++j) {
        const int li = (tid + j * NT) * 4;
        const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
        const uint32_t gx = x0 + lx, gy = y0 + ly, gz = z0 + lz;
        const uint32_t g = gx + L * (gy + L * gz);
        const bool rowend = (lane & (LPR - 1)) == LPR - 1;
        uint4 w[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) w[s] = philox4x32_10(g + s, t_lo, t_hi, DOM_SITE, p.k0, p.k1);
        uint32_t bxn, byn, bzn = 0u, d;
        if (MODEL == XY) {
            // Wolff embedding: aligned iff a_i a_j > 0, p = 1 - exp(-2 beta a_i a_j)
            const float scale = 5.9604644775390625e-8f;  // 2^-24
            const float4 a = *reinterpret_cast<const float4 *>(val_s + li);
            const float ax3 = (lx + 4 < TX) ? val_s[li + 4] : val_s[NS + ly + TY * lz];
            const float4 ay = (ly + 1 < TY) ? *reinterpret_cast<const float4 *>(val_s + li + TX)
                                            : *reinterpret_cast<const float4 *>(val_s + NS + G::FXB + lx + TX * lz);
            const float av[4] = {a.x, a.y, a.z, a.w};
            const float axv[4] = {a.y, a.z, a.w, ax3};
            const float ayv[4] = {ay.x, ay.y, ay.z, ay.w};
            bxn = byn = 0u;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const float px = av[s] * axv[s], py = av[s] * ayv[s];
                if (px > 0.f && (float)(w[s].x >> 8) * scale < SW_NEG_EXPM1F(p.m2beta * px)) bxn |= 1u << s;
                if (py > 0.f && (float)(w[s].y >> 8) * scale < SW_NEG_EXPM1F(p.m2beta * py)) byn |= 1u << s;
            }
            if (DIM == 3) {
                const float4 az = (lz + 1 < TZ) ? *reinterpret_cast<const float4 *>(val_s + li + TX * TY)
                                                : *reinterpret_cast<const float4 *>(val_s + NS + G::FXB + G::FYB + lx + TX * ly);
                const float azv[4] = {az.x, az.y, az.z, az.w};
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const float pz = av[s] * azv[s];
                    if (pz > 0.f && (float)(w[s].z >> 8) * scale < SW_NEG_EXPM1F(p.m2beta * pz)) bzn |= 1u << s;
                }
            }
            d = (w[0].w >> 31) | ((w[1].w >> 31) << 1) | ((w[2].w >> 31) << 2) | ((w[3].w >> 31) << 3);
        } else if (MODEL == CLOCK) {
            // q-state clock model (readings 23-25): state p, mirror index m.
            // k = (2p - m) mod 2q, u = k mod q: the component along the mirror normal is
            // +sin(pi u / q) for k < q, -sin(pi u / q) for k >= q, zero for u = 0.  A bond between
            // neighbours of the same non-zero sign is active iff word < T[u_i q + u_j], the table
            // floor((1 - exp(-2 beta sin sin)) 2^32) built once on the host.
            const uint16_t *sp = (const uint16_t *)p.spins;
            const int q = p.q, m = p.mirror;
            auto cls = [&](uint32_t pp) -> uint32_t {  // u | sign class << 16 (1: positive, 2: negative, 0: zero)
                int k = 2 * (int)pp - m;
                if (k < 0) k += 2 * q;
                const int u = k >= q ? k - q : k;
                return (uint32_t)u | (u == 0 ? 0u : (k >= q ? 2u : 1u) << 16);
            };
            const uint2 own2 = *reinterpret_cast<const uint2 *>(sp + g);
            const uint2 up2 = *reinterpret_cast<const uint2 *>(sp + ((gy + 1 == L) ? g - L * (L - 1) : g + L));
            uint32_t nbq = __shfl_down_sync(FULL, own2.x, 1) & 0xffffu;
            if (rowend) nbq = sp[(gx + 4 == L) ? g + 4 - L : g + 4];
            const uint32_t c0[5] = {cls(own2.x & 0xffffu), cls(own2.x >> 16), cls(own2.y & 0xffffu), cls(own2.y >> 16), cls(nbq)};
            const uint32_t cy[4] = {cls(up2.x & 0xffffu), cls(up2.x >> 16), cls(up2.y & 0xffffu), cls(up2.y >> 16)};
            uint32_t cz[4] = {0u, 0u, 0u, 0u};
            if (DIM == 3) {
                const uint2 fr2 = *reinterpret_cast<const uint2 *>(sp + ((gz + 1 == L) ? g - LL * (L - 1) : g + LL));
                cz[0] = cls(fr2.x & 0xffffu); cz[1] = cls(fr2.x >> 16); cz[2] = cls(fr2.y & 0xffffu); cz[3] = cls(fr2.y >> 16);
            }
            auto bond = [&](uint32_t a, uint32_t b, uint32_t word) -> uint32_t {
                if (((a & b) >> 16) == 0u) return 0u;  // different sign, or one component is zero
                return word < __ldg(p.clock_T + (a & 0xffffu) * (uint32_t)q + (b & 0xffffu)) ? 1u : 0u;
            };
            bxn = byn = 0u;
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                bxn |= bond(c0[s], c0[s + 1], w[s].x) << s;
                byn |= bond(c0[s], cy[s], w[s].y) << s;
                if (DIM == 3) bzn |= bond(c0[s], cz[s], w[s].z) << s;
            }
            d = (w[0].w >> 31) | ((w[1].w >> 31) << 1) | ((w[2].w >> 31) << 2) | ((w[3].w >> 31) << 3);
        }
        // the four 1-bit draws ride in bits 12-15 of the bond word (one register less per quad)
        bnd[j] = bxn | (byn << 4) | (bzn << 8) | (d << 12);

        // x-runs: link = my last site is bonded to the next quad of the row, thru = no break inside
        const uint32_t Lk = __ballot_sync(FULL, (bxn & 8u) && !rowend);
        const uint32_t Th = __ballot_sync(FULL, (bxn & 7u) == 7u);
        const uint32_t E = Th & (Lk << 1);                 // entering quad c from the right leaves it to the left
        const uint32_t z3 = ~bxn & 7u;
        const int tails = z3 ? 32 - __clz(z3) : 0;         // first site of the run that reaches my site 3
        const uint32_t below = (1u << lane) - 1u;
        const bool linked_prev = (Lk << 1) >> lane & 1u;
        const uint32_t zE = ~E & below;
        const int q0 = linked_prev ? 31 - __clz(zE) : lane;  // quad in which the run of my site 0 starts
        const int tq = __shfl_sync(FULL, tails, q0);
        const uint32_t s0 = linked_prev ? (uint32_t)(li - 4 * (lane - q0) + tq) : (uint32_t)li;
        const uint32_t s1 = (bxn & 1u) ? s0 : (uint32_t)li + 1u;
        const uint32_t s2 = (bxn & 2u) ? s1 : (uint32_t)li + 2u;
        const uint32_t s3 = (bxn & 4u) ? s2 : (uint32_t)li + 3u;
        *reinterpret_cast<uint4 *>(lab_s + li) = make_uint4(s0, s1, s2, s3);

        // bonds through the tile faces (incl. the periodic wrap) go to the global merge
        if (rowend && (bxn & 8u)) {
            const int r = ly + TY * lz;
            atomicOr(&face_s[r >> 5], 1u << (r & 31));
        }
        if (ly == TY - 1 && byn) {
            const int b = lx + TX * lz;
            atomicOr(&face_s[G::FXW + (b >> 5)], byn << (b & 31));
        }
        if (DIM == 3 && lz == TZ - 1 && bzn) {
            const int b = lx + TX * ly;
            atomicOr(&face_s[G::FXW + G::FYW + (b >> 5)], bzn << (b & 31));
        }
        if (ly < TY - 1) work[0] |= byn << (4 * j);
        if (DIM == 3 && lz < TZ - 1) work[1] |= bzn << (4 * j);
    }
    __syncthreads();

    if (tid < 32) {
        // face words are final: exclusive prefix of their popcounts, and room in the global pair list
        const uint32_t c0 = lane < G::NFW ? __popc(face_s[lane]) : 0u;
        const uint32_t c1 = lane + 32 < G::NFW ? __popc(face_s[lane + 32]) : 0u;
        uint32_t i0 = c0, i1 = c1;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u0 = __shfl_up_sync(FULL, i0, o), u1 = __shfl_up_sync(FULL, i1, o);
            if (lane >= o) { i0 += u0; i1 += u1; }
        }
        const uint32_t t0 = __shfl_sync(FULL, i0, 31), t1 = __shfl_sync(FULL, i1, 31);
        if (lane < G::NFW) fpre_s[lane] = i0 - c0;
        if (lane + 32 < G::NFW) fpre_s[lane + 32] = t0 + i1 - c1;
        if (lane == 0) fpre_s[G::NFWP] = (t0 + t1) ? atomicAdd(p.npairs, t0 + t1) : 0u;
    }

    // phase 2a: SW_BL_ROUNDS uniform hook rounds.  Every thread looks at its quads' bonds with two
    // 16-byte loads (parents of its 4 sites and of their 4 neighbours); a bond whose two parents differ
    // tries to hook the larger one under the smaller with a compare-and-swap (parent slot: itself ->
    // smaller): that succeeds only if the larger one still is a root, and a failure changes nothing
    // (the bond stays in the work mask).  Straight-line predicated code: no loops, no divergence.
    // Each round ends with a pointer-jumping pass that re-flattens the forest.
    const uint32_t lab_sa = (uint32_t)__cvta_generic_to_shared(lab_s);
#pragma unroll 1
    for (int round = 0; round < SW_BL_ROUNDS; ++round) {
        if (SW_BL_HOOK_LOOP && DIM == 3) {
            // one iteration per active bond of the thread (trip count = the largest popcount in the
            // warp): at 3D densities (a quarter of the bond slots active) this beats the predicated code
#pragma unroll
            for (int dir = 0; dir < 2; ++dir) {
                uint32_t todo = work[dir];
                work[dir] = 0u;
                while (__any_sync(FULL, todo != 0u)) {
                    if (todo) {
                        const uint32_t k = 31u - (uint32_t)__clz((int)(todo & (0u - todo)));
                        todo &= todo - 1u;
                        const uint32_t a = (uint32_t)tid * 4u + (k >> 2) * (uint32_t)(NT * 4) + (k & 3u);
                        const uint32_t pa = lab_s[a], pb = lab_s[a + (dir ? TX * TY : TX)];
                        const uint32_t hi = max(pa, pb), lo = min(pa, pb);
                        if (hi != lo) {
                            const uint32_t old = atomicCAS(&lab_s[hi], hi, lo);
                            if (old != hi && old != lo) work[dir] |= 1u << k;  // old == lo: a twin bond did it already
                        }
                    }
                }
            }
        } else {
#pragma unroll
        for (int j = 0; j < QPT; ++j) {
            const int li = (tid + j * NT) * 4;
            const uint4 la = *reinterpret_cast<const uint4 *>(lab_s + li);
            const uint32_t av[4] = {la.x, la.y, la.z, la.w};
#pragma unroll
            for (int dir = 0; dir < (DIM == 3 ? 2 : 1); ++dir) {
                const uint32_t nib = (work[dir] >> (4 * j)) & 0xfu;
                const uint4 lb = *reinterpret_cast<const uint4 *>(lab_s + ((li + (dir ? TX * TY : TX)) & (NS - 1)));
                const uint32_t bv[4] = {lb.x, lb.y, lb.z, lb.w};
                uint32_t left = 0u;
#pragma unroll
                for (int sidx = 0; sidx < 4; ++sidx) {
                    const uint32_t hi = max(av[sidx], bv[sidx]), lo = min(av[sidx], bv[sidx]);
                    const uint32_t need = ((nib >> sidx) & 1u) & (uint32_t)(hi != lo);
                    uint32_t old = hi;
                    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %4, 0;\n\t"
                                 "@p atom.shared.cas.b32 %0, [%1], %2, %3;\n\t}"
                                 : "+r"(old) : "r"(lab_sa + 4u * hi), "r"(hi), "r"(lo), "r"(need) : "memory");
                    left |= (uint32_t)(old != hi && old != lo) << sidx;  // old == lo: a twin bond did it already
                }
                work[dir] = (work[dir] & ~(0xfu << (4 * j))) | (left << (4 * j));
            }
        }
        }
        __syncthreads();
        volatile uint32_t *vl = lab_s;
#pragma unroll
        for (int j = 0; j < QPT; ++j) {
            const int li = (tid + j * NT) * 4;
            uint4 r = *reinterpret_cast<const uint4 *>(lab_s + li);
            uint4 prev = make_uint4(li, li + 1, li + 2, li + 3);
#pragma unroll
            for (int k = 0; k < SW_BL_MIDJUMPS; ++k) jump4(vl, r, prev);
            *reinterpret_cast<uint4 *>(lab_s + li) = r;
        }
        __syncthreads();
    }
    // phase 2b: whatever is left (roots that several bonds wanted to hook at once, deep trees) goes
    // through the general union-find.  The leftovers of all threads are first compacted into one list
    // so that every lane of every warp has a union to do (a warp whose entries do not fit keeps them).
    if (SW_BL_ROUNDS > 0) {
        const uint32_t cnt = __popc(work[0]) + __popc(work[1]);
        uint32_t inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += u;
        }
        const uint32_t tot = __shfl_sync(FULL, inc, 31);
        uint32_t base = 0u;
        if (lane == 31 && tot) base = atomicAdd(&fpre_s[G::NFWP + 1], tot);
        base = __shfl_sync(FULL, base, 31);
        if (tot && base + tot <= (uint32_t)G::LEFT_CAP) {
            uint32_t pos = base + inc - cnt;
#pragma unroll
            for (int dir = 0; dir < (DIM == 3 ? 2 : 1); ++dir) {
                uint32_t w = work[dir];
                while (w) {
                    const uint32_t k = 31u - (uint32_t)__clz((int)(w & (0u - w)));
                    w &= w - 1u;
                    left_s[pos++] = (uint16_t)(((uint32_t)tid * 4u + (k >> 2) * (uint32_t)(NT * 4) + (k & 3u)) | (dir ? 0x8000u : 0u));
                }
                work[dir] = 0u;
            }
        } else if (tot && lane == 31) {
            atomicMin(&fpre_s[G::NFWP + 2], base);  // the list is valid below the first range that did not fit
        }
        __syncthreads();
        const int nleft = min(fpre_s[G::NFWP + 1], fpre_s[G::NFWP + 2]);
        // warps whose entries did not fit still hold their bits and run the loop below
        for (int e0 = (tid & ~31); e0 < nleft; e0 += NT) {
            const int e = e0 + lane;
            if (e < nleft) {
                const uint32_t v = left_s[e];
                const uint32_t a = v & 0x7fffu;
                union_s(lab_s, a, a + ((v & 0x8000u) ? (uint32_t)(TX * TY) : (uint32_t)TX));
            }
            __syncwarp();
        }
    }
    // warp-uniform trip count + __syncwarp: lanes whose union ends early wait for the others instead
    // of drifting into later iterations on their own (that would serialise the warp)
#pragma unroll
    for (int dir = 0; dir < (DIM == 3 ? 2 : 1); ++dir) {
        uint32_t w = work[dir];
        while (__any_sync(FULL, w != 0u)) {
            if (w) {
                const uint32_t k = 31u - (uint32_t)__clz((int)(w & (0u - w)));
                w &= w - 1u;
                const uint32_t a = (uint32_t)tid * 4u + (k >> 2) * (uint32_t)(NT * 4) + (k & 3u);
                union_s(lab_s, a, a + (dir ? (uint32_t)(TX * TY) : (uint32_t)TX));
            }
            __syncwarp();
        }
    }
    __syncthreads();

    // active face bonds -> (address of i, address of j) in the global pair list (k_merge's work)
    {
        const uint32_t ntx = p.ntx, nty = p.nty;
        const uint32_t tjx = (bx + 1 == ntx) ? tile - (ntx - 1) : tile + 1;
        const uint32_t tjy = (by + 1 == nty) ? tile - ntx * (nty - 1) : tile + ntx;
        const uint32_t tjz = (DIM == 3) ? ((bz + 1 == p.ntz) ? tile - ntx * nty * (p.ntz - 1) : tile + ntx * nty) : 0u;
        const uint32_t fbase = fpre_s[G::NFWP];
        for (int sl = tid; sl < 32 * G::NFW; sl += NT) {
            const uint32_t fw = face_s[sl >> 5];
            if ((fw >> (sl & 31)) & 1u) {
                const uint32_t pos = fbase + fpre_s[sl >> 5] + __popc(fw & ((1u << (sl & 31)) - 1u));
                uint32_t li_i, li_j, tj;
                if (sl < 32 * G::FXW) {                      // slot = ly + TY lz
                    li_j = TX * sl; li_i = li_j + (TX - 1); tj = tjx;
                } else if (sl < 32 * (G::FXW + G::FYW)) {    // slot = lx + TX lz
                    const uint32_t b = sl - 32 * G::FXW;
                    li_j = (b % TX) + (TX * TY) * (b / TX); li_i = li_j + TX * (TY - 1); tj = tjy;
                } else {                                     // slot = lx + TX ly
                    li_j = sl - 32 * (G::FXW + G::FYW); li_i = li_j + TX * TY * (TZ - 1); tj = tjz;
                }
                p.pairs[pos] = make_uint2(tile_base + li_i, (tj << G::LOG2NS) + li_j);
            }
        }
    }
    // phase 3: no unions any more, the forest is static.  JUMPS rounds of pointer jumping (uniform
    // work, no divergence; a thread only rewrites the entries of its own sites, and whatever another
    // thread reads is a valid ancestor), then the parent is stored as it stands: k_merge and k_flip
    // follow whatever is left of the chain through L1/L2.
    volatile uint32_t *vlab = lab_s;
#pragma unroll
    for (int j = 0; j < QPT; ++j) {
        const int li = (tid + j * NT) * 4;
        uint4 r = *reinterpret_cast<const uint4 *>(lab_s + li);
        uint4 prev = make_uint4(li, li + 1, li + 2, li + 3);
#pragma unroll
        for (int k = 0; k < SW_BL_JUMPS; ++k) {
            jump4(vlab, r, prev);
            if (k + 1 < SW_BL_JUMPS) *reinterpret_cast<uint4 *>(lab_s + li) = r;
        }
        const uint32_t dm = (1u << db) - 1u, d = bnd[j] >> 12;
        uint4 o;
        o.x = ((tile_base + r.x) << db) | (d & dm);
        o.y = ((tile_base + r.y) << db) | ((d >> db) & dm);
        o.z = ((tile_base + r.z) << db) | ((d >> (2 * db)) & dm);
        o.w = ((tile_base + r.w) << db) | ((d >> (3 * db)) & dm);
        *reinterpret_cast<uint4 *>(p.labels + tile_base + li) = o;
        if (p.bonds) {
            const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
            const uint32_t g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
            *reinterpret_cast<uint32_t *>(p.bonds + g) =
                spread4(bnd[j] & 0xfu) | (spread4((bnd[j] >> 4) & 0xfu) << 1) | (spread4((bnd[j] >> 8) & 0xfu) << 2);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Global union-find over the packed label words.  A root is only ever changed by the atomicCAS that
// hooks it; path splitting rewrites non-roots with (valid) ancestors, keeping their draw field.
// ------------------------------------------------------------------------------------------------
// Label words are read and path-split by many threads while others hook roots with atomicCAS: these
// accesses are relaxed device-scope atomics (a word is only ever replaced by a valid word: same draw field,
// parent = an ancestor), not plain loads and stores.
__device__ __forceinline__ uint32_t ld_relaxed(const uint32_t *ptr)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(uint32_t *ptr, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" :: "l"(ptr), "r"(v) : "memory");
}

template <int LOG2NS, int TX, int TY>
__device__ __forceinline__ uint32_t linear_of(const Params &p, uint32_t a)
{
    const uint32_t li = a & ((1u << LOG2NS) - 1u);
    return p.tile_origin[a >> LOG2NS] + (li % TX) + p.L * (((li / TX) % TY) + p.L * (li / (TX * TY)));
}

// ------------------------------------------------------------------------------------------------
// k_merge: grid-stride loop over the compact pair list (grid: 96 CTAs per SM, i.e. one or two pairs per
// thread, so that the list - which is in tile order - is walked in order and label blocks stay in L2).  Union of (a, b): both chains are followed in
// one loop (two loads in flight), path splitting on the way (non-roots are re-pointed to their
// grandparent with relaxed atomic stores, keeping their draw field); then the root with the larger linear
// index is hooked under the other with atomicCAS(root word -> parent word); a lost race starts
// over from the roots found.  Thread 0 also clears the magnetisation accumulators k_flip adds to.
// ------------------------------------------------------------------------------------------------
template <int DIM, int TX, int TY, int TZ>
__global__ void __launch_bounds__(256) k_merge(const Params p)
{
    using G = TileGeom<DIM, TX, TY, TZ>;
    const uint32_t gid = blockIdx.x * 256u + threadIdx.x;
    if (gid == 0) { p.acc->M_int = 0ull; p.acc->mx = 0.0; p.acc->my = 0.0; }
    if (gid < (uint32_t)p.nk_clear) p.acc->nk[gid] = 0ull;   // Potts: the accumulators k_flip adds to
    const uint32_t n = *p.npairs;
    const int db = p.db;
    const uint32_t dm = (1u << db) - 1u;
    uint32_t *lab = p.labels;
    for (uint32_t i = gid; i < n; i += gridDim.x * 256u) {
        const uint2 ab = p.pairs[i];
        uint32_t a = ab.x, b = ab.y;
        unsigned hops = 0, retries = 0, linked = 0;
        uint32_t wa = ld_relaxed(lab + a), wb = ld_relaxed(lab + b);
        for (;;) {
            for (;;) {
                const uint32_t pa = wa >> db, pb = wb >> db;
                const bool ra = pa == a, rb = pb == b;
                if (ra && rb) break;
                uint32_t wpa = 0u, wpb = 0u;
                if (!ra) wpa = ld_relaxed(lab + pa);
                if (!rb) wpb = ld_relaxed(lab + pb);
                if (!ra) {
                    const uint32_t gp = wpa >> db;
                    if (gp != pa) st_relaxed(lab + a, (gp << db) | (wa & dm));
                    a = pa; wa = wpa; ++hops;
                }
                if (!rb) {
                    const uint32_t gp = wpb >> db;
                    if (gp != pb) st_relaxed(lab + b, (gp << db) | (wb & dm));
                    b = pb; wb = wpb; ++hops;
                }
            }
            if (a == b) break;
            if (linear_of<G::LOG2NS, TX, TY>(p, a) < linear_of<G::LOG2NS, TX, TY>(p, b)) {
                const uint32_t t = a; a = b; b = t;
                const uint32_t tw = wa; wa = wb; wb = tw;
            }
            // a is the root with the larger linear index: hook it under b (keeping a's draw field)
            const uint32_t old = atomicCAS(&p.labels[a], wa, (b << db) | (wa & dm));
            if (old == wa) { linked = 1; break; }
            wa = old;  // a was hooked by another thread meanwhile: go on from its new word
            ++retries;
        }
        if (p.counting) {
            atomicAdd(&p.acc->stats[1], 1ull);
            atomicAdd(&p.acc->stats[2], (unsigned long long)linked);
            atomicAdd(&p.acc->stats[3], (unsigned long long)retries);
            atomicAdd(&p.acc->stats[4], (unsigned long long)hops);
            atomicMax(&p.acc->stats[5], (unsigned long long)hops);
        }
    }
}

__device__ __forceinline__ uint4 ldg_stream(const uint32_t *ptr)
{
    uint4 v;
    asm volatile("ld.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(ptr) : "memory");
    return v;
}

// ------------------------------------------------------------------------------------------------
// k_flip: one CTA per tile, QPT quads per thread.  Every site follows its parent words to the root
// (first hop: the tile-local root, whose word sits in this tile's 4*NS-byte block and is served by
// L1; further hops only for clusters that cross tile faces), takes the root's draw field as the
// cluster's new value and writes its spin; magnetisation sums per CTA.
// ------------------------------------------------------------------------------------------------
#ifndef SW_FLIP_FIRST_HOP_ALWAYS
#define SW_FLIP_FIRST_HOP_ALWAYS 1
#endif
#ifndef SW_FLIP_PREFETCH
#define SW_FLIP_PREFETCH 1   // quads whose label words are in flight ahead of the chase
#endif
#ifndef SW_FLIP_THREADS_PER_SM
#define SW_FLIP_THREADS_PER_SM 2048  // resident threads per SM k_flip is compiled for (register cap)
#endif
template <int DIM, int MODEL, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT, (SW_FLIP_THREADS_PER_SM / NT > 0 ? SW_FLIP_THREADS_PER_SM / NT : 1)) k_flip(const Params p)
{
    using G = TileGeom<DIM, TX, TY, TZ>;
    constexpr int NS = G::NS, NQ = NS / 4, QPT = NQ / NT;
    __shared__ uint32_t hist_s[256];  // Potts: n_k of this tile (<= NS, fits 32 bits)
    __shared__ int red_s[32];

    const uint32_t L = p.L;
    const uint32_t x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = (DIM == 3) ? blockIdx.z * TZ : 0u;
    const uint32_t tile = blockIdx.x + p.ntx * (blockIdx.y + p.nty * blockIdx.z);
    const uint32_t tile_base = tile << G::LOG2NS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int db = (MODEL == POTTS) ? p.db : 1;
    const uint32_t dm = (1u << db) - 1u;
    const uint32_t *__restrict__ lab = p.labels;
    asm volatile("" : "+l"(lab));  // keep the base address in registers (else it is re-read from the constant bank per load)
    const unsigned counting = p.counting ? 1u : 0u;

    if (MODEL == POTTS) {
        for (int k = tid; k < 256; k += NT) hist_s[k] = 0u;
        __syncthreads();
    }
    if (tile == 0 && tid == 0) {
        *p.npairs = 0u;   // k_merge of this step is done: empty list for the next one
        p.acc->t += 1ull; // and the next k_bond_label works on the next step
    }
    int m_loc = 0;
    uint32_t cnt_lo = 0u, cnt_hi = 0u;  // Potts, q <= 8: per-thread counts of states 0-3 / 4-7, one byte each
    unsigned chase_hops = 0;
    constexpr int STEP = NT * 4;                                                     // sites between two quads of a thread
    constexpr int STEP_PLANES = (DIM == 3 && STEP % (TX * TY) == 0) ? STEP / (TX * TY) : 0;
    constexpr int STEP_ROWS = (DIM == 2 && STEP % TX == 0) ? STEP / TX : 0;
    uint32_t g_first, g_step;
    {
        const int li0 = tid * 4, lx = li0 % TX, ly = (li0 / TX) % TY, lz = li0 / (TX * TY);
        g_first = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
        g_step = STEP_PLANES > 0 ? (uint32_t)STEP_PLANES * L * L : (uint32_t)STEP_ROWS * L;
    }
    asm volatile("" : "+r"(g_first));   // (kept in a register: otherwise it is rebuilt from threadIdx / blockIdx for every quad)
    // the label words of the NEXT quad are requested before the parents of this one are followed: the
    // kernel is bound by the latency of these reads (DRAM), not by instruction issue
#if SW_FLIP_PREFETCH == 2
    uint4 w4n = ldg_stream(lab + tile_base + tid * 4), w4m = w4n;
    if (QPT > 1) w4m = ldg_stream(lab + tile_base + (tid + NT) * 4);
#else
    uint4 w4n = ldg_stream(lab + tile_base + tid * 4);
#endif
#pragma unroll
    for (int j = 0; j < QPT; ++j) {
        const int li = (tid + j * NT) * 4;
        const uint32_t a0 = tile_base + li;
        const uint4 w4 = w4n;
#if SW_FLIP_PREFETCH == 2
        w4n = w4m;
        if (j + 2 < QPT) w4m = ldg_stream(lab + a0 + 2 * NT * 4);
#else
        if (j + 1 < QPT) w4n = ldg_stream(lab + a0 + NT * 4);
#endif
        // follow the parent words to the root: the node whose parent field is its own address; that word's
        // draw field is the cluster's new value.  First hop in straight-line code, four loads in flight: a
        // site that is no root loads the word of its parent (the tile-local ancestor k_bond_label stored;
        // this tile's block, usually in L1).  If that node is a root (most sites: clusters inside one
        // tile, or whose tile-local root is the global one) the site is done; the rest goes on in a loop.
        uint32_t pw[4] = {w4.x, w4.y, w4.z, w4.w};
        uint32_t at[4];
#pragma unroll
        for (int s = 0; s < 4; ++s) {
            at[s] = pw[s] >> db;
#if SW_FLIP_FIRST_HOP_ALWAYS
            pw[s] = __ldg(lab + at[s]);     // (a site that is its own ancestor reads its own word again: an L1 hit, no predicate)
#else
            if (at[s] != a0 + (uint32_t)s) pw[s] = __ldg(lab + at[s]);
#endif
        }
        for (;;) {
            const uint32_t q0 = pw[0] >> db, q1 = pw[1] >> db, q2 = pw[2] >> db, q3 = pw[3] >> db;
            const bool m0 = q0 != at[0], m1 = q1 != at[1], m2 = q2 != at[2], m3 = q3 != at[3];
            chase_hops += counting;
            if (!(m0 | m1 | m2 | m3)) break;
            if (m0) { at[0] = q0; pw[0] = __ldg(lab + q0); }
            if (m1) { at[1] = q1; pw[1] = __ldg(lab + q1); }
            if (m2) { at[2] = q2; pw[2] = __ldg(lab + q2); }
            if (m3) { at[3] = q3; pw[3] = __ldg(lab + q3); }
        }
        __syncwarp();

        // linear index of the quad's first site: the quads of a thread are a whole number of planes (3D) or rows (2D)
        // apart, so one multiply-add per quad replaces the decomposition of li
        uint32_t g;
        if (STEP_PLANES > 0 || STEP_ROWS > 0) g = g_first + (uint32_t)j * g_step;
        else {
            const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
            g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
        }
        if (MODEL == ISING) {
            // "All spins in each cluster are set randomly to +1 or -1"
            const uint32_t dn = (pw[0] & 1u) | ((pw[1] & 1u) << 1) | ((pw[2] & 1u) << 2) | ((pw[3] & 1u) << 3);
            *reinterpret_cast<uint32_t *>((uint8_t *)p.spins + g) = 0xffffffffu ^ (spread4(dn) * 0xfeu);
            m_loc += 2 * __popc(dn) - 4;
        } else if (MODEL == POTTS) {
            const uint32_t d0 = pw[0] & dm, d1 = pw[1] & dm, d2 = pw[2] & dm, d3 = pw[3] & dm;
            *reinterpret_cast<uint32_t *>((uint8_t *)p.spins + g) = d0 | (d1 << 8) | (d2 << 16) | (d3 << 24);
            if (p.q <= 8) {
                const uint32_t dv[4] = {d0, d1, d2, d3};
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const uint32_t inc = 1u << ((dv[s] & 3u) * 8u);
                    if (dv[s] & 4u) cnt_hi += inc; else cnt_lo += inc;
                }
            } else {
                atomicAdd(&hist_s[d0], 1u);
                atomicAdd(&hist_s[d1], 1u);
                atomicAdd(&hist_s[d2], 1u);
                atomicAdd(&hist_s[d3], 1u);
            }
        } else if (MODEL == CLOCK) {
            // PAPER.md:159 mirror projection of the cluster: p -> (m - p) mod q
            if ((pw[0] | pw[1] | pw[2] | pw[3]) & 1u) {
                uint2 v = *reinterpret_cast<uint2 *>((uint16_t *)p.spins + g);
                uint32_t st[4] = {v.x & 0xffffu, v.x >> 16, v.y & 0xffffu, v.y >> 16};
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    if (pw[s] & 1u) {
                        int n = p.mirror - (int)st[s];
                        if (n < 0) n += p.q;
                        st[s] = (uint32_t)n;
                    }
                }
                *reinterpret_cast<uint2 *>((uint16_t *)p.spins + g) = make_uint2(st[0] | (st[1] << 16), st[2] | (st[3] << 16));
            }
        } else {
            // PAPER.md:159 mirror projection: theta' = c - theta, wrapped into [0, 2 pi]
            if ((pw[0] | pw[1] | pw[2] | pw[3]) & 1u) {
                float4 t4 = *reinterpret_cast<float4 *>((float *)p.spins + g);
                float th[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    if (pw[s] & 1u) {
                        float v = p.crefl - th[s];
                        if (v < 0.0f) v = v + 6.283185307179586476925286766559f;
                        th[s] = v;
                    }
                }
                *reinterpret_cast<float4 *>((float *)p.spins + g) = make_float4(th[0], th[1], th[2], th[3]);
            }
        }
    }

    if (MODEL == ISING) {
        m_loc = __reduce_add_sync(FULL, m_loc);
        if (lane == 0) red_s[warp] = m_loc;
        __syncthreads();
        if (warp == 0) {
            int v = lane < NT / 32 ? red_s[lane] : 0;
            v = __reduce_add_sync(FULL, v);
            if (lane == 0) atomicAdd(&p.acc->M_int, (unsigned long long)(long long)v);
        }
    } else if (MODEL == POTTS) {
        if (p.q <= 8) {
            // a thread counted at most 4 QPT <= 255 sites per state: bytes cannot overflow
            for (int k = 0; k < p.q; ++k) {
                const uint32_t c = ((k < 4 ? cnt_lo : cnt_hi) >> ((k & 3) * 8)) & 0xffu;
                const uint32_t w = __reduce_add_sync(FULL, c);
                if (lane == 0 && w) atomicAdd(&hist_s[k], w);
            }
        }
        __syncthreads();
        for (int k = tid; k < p.q; k += NT)
            if (hist_s[k]) atomicAdd(&p.acc->nk[k], (unsigned long long)hist_s[k]);
    }
    if (p.counting) {
        atomicAdd(&p.acc->stats[6], (unsigned long long)chase_hops);
        atomicMax(&p.acc->stats[7], (unsigned long long)chase_hops);
    }
}

// ------------------------------------------------------------------------------------------------
// k_export_labels: canonical labels on request (sw_get_labels): labels_out[i] = minimum linear site
// index of the cluster of site i, linear order.  Not on the hot path.
// ------------------------------------------------------------------------------------------------
template <int DIM, int TX, int TY, int TZ>
__global__ void __launch_bounds__(256) k_export_labels(const Params p)
{
    using G = TileGeom<DIM, TX, TY, TZ>;
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= p.N) return;
    uint32_t x, y, z;
    decode(p, i, x, y, z);
    const uint32_t tile = x / TX + p.ntx * (y / TY + p.nty * (z / TZ));
    uint32_t a = (tile << G::LOG2NS) + (x % TX) + TX * ((y % TY) + TY * (z % TZ));
    const int db = p.db;
    for (;;) {
        const uint32_t n = p.labels[a] >> db;
        if (n == a) break;
        a = n;
    }
    p.labels_out[i] = linear_of<G::LOG2NS, TX, TY>(p, a);
}

// ------------------------------------------------------------------------------------------------
// k_measure_xy: E = -sum cos(theta_i - theta_j) (Eq. 3) and, if WITH_M, (sum cos, sum sin), four consecutive
// sites per thread.  The 12 (8) cosines of a thread and the sums of a warp are accumulated in fp32 (a few
// hundred terms of magnitude <= 1: rounding error ~1e-5 per warp sum, random in sign), the warp sums in
// fp64: the fp64 pipe of this GPU is slow, and one thread per site with fp64 shuffles made this pass cost
// as much as the whole SW step.
// ------------------------------------------------------------------------------------------------
template <int DIM, bool WITH_M>
__global__ void __launch_bounds__(256) k_measure_xy(const Params p)
{
    __shared__ double red_s[3][8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t L = p.L, LL = L * L;
    const uint32_t g = (blockIdx.x * 256u + tid) * 4u;  // N is a multiple of 1024
    uint32_t x, y, z;
    decode(p, g, x, y, z);
    const float *s = (const float *)p.spins;
    const float4 a = *reinterpret_cast<const float4 *>(s + g);
    const float ax = s[(x + 4 == L) ? g + 4 - L : g + 4];
    const float4 b = *reinterpret_cast<const float4 *>(s + ((y + 1 == L) ? g - L * (L - 1) : g + L));
    float e = cosf(a.x - a.y) + cosf(a.y - a.z) + cosf(a.z - a.w) + cosf(a.w - ax)
            + cosf(a.x - b.x) + cosf(a.y - b.y) + cosf(a.z - b.z) + cosf(a.w - b.w);
    if (DIM == 3) {
        const float4 c = *reinterpret_cast<const float4 *>(s + ((z + 1 == L) ? g - LL * (L - 1) : g + LL));
        e += cosf(a.x - c.x) + cosf(a.y - c.y) + cosf(a.z - c.z) + cosf(a.w - c.w);
    }
    e = -e;
    float cx = 0.f, cy = 0.f;
    if (WITH_M) {
        float sn, cs;
        sincosf(a.x, &sn, &cs); cx += cs; cy += sn;
        sincosf(a.y, &sn, &cs); cx += cs; cy += sn;
        sincosf(a.z, &sn, &cs); cx += cs; cy += sn;
        sincosf(a.w, &sn, &cs); cx += cs; cy += sn;
    }
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_down_sync(FULL, e, o);
        if (WITH_M) { cx += __shfl_down_sync(FULL, cx, o); cy += __shfl_down_sync(FULL, cy, o); }
    }
    if (lane == 0) { red_s[0][warp] = (double)e; red_s[1][warp] = (double)cx; red_s[2][warp] = (double)cy; }
    __syncthreads();
    if (tid == 0) {
        double es = 0.0, xs = 0.0, ys = 0.0;
        for (int w = 0; w < 8; ++w) { es += red_s[0][w]; xs += red_s[1][w]; ys += red_s[2][w]; }
        atomicAdd(&p.acc->E_xy, es);
        if (WITH_M) { atomicAdd(&p.acc->mx, xs); atomicAdd(&p.acc->my, ys); }
    }
}

// ------------------------------------------------------------------------------------------------
// k_measure4 (Ising, Potts): E (Eq. 1, 2) and, if WITH_M, the magnetisation sums (Eq. 4, 5).  Grid-stride over
// groups of 16 consecutive sites (L is a multiple of 32), 16-byte loads; the spin words of the group and of its
// +x / +y / +z neighbours give byte-equality masks, and with spins in the model's range the energy is a popcount:
// Ising -sum s_i s_j = (#pairs - 2 #equal), Potts #unequal pairs.  A CTA adds to the global sums once, at its
// end (one atomic per 1024 sites on a single address was what bounded the first version of this kernel).
// ------------------------------------------------------------------------------------------------
template <int DIM, int MODEL, bool WITH_M>
__global__ void __launch_bounds__(256) k_measure4(const Params p)
{
    __shared__ uint32_t hist_s[256];
    __shared__ long long red_s[2][8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t L = p.L, LL = L * L;
    if (MODEL == POTTS && WITH_M) {
        hist_s[tid] = 0u;
        __syncthreads();
    }
    const uint8_t *sp = (const uint8_t *)p.spins;
    const uint32_t ngroups = p.N >> 4;
    long long e_acc = 0, m_acc = 0;
    for (uint32_t q = blockIdx.x * 256u + (uint32_t)tid; q < ngroups; q += gridDim.x * 256u) {
        const uint32_t g = q << 4;
        uint32_t x, y, z;
        decode(p, g, x, y, z);
        const uint4 own = *reinterpret_cast<const uint4 *>(sp + g);
        const uint32_t nb = sp[(x + 16 == L) ? g + 16 - L : g + 16];
        const uint4 up = *reinterpret_cast<const uint4 *>(sp + ((y + 1 == L) ? g - L * (L - 1) : g + L));
        int equal = __popc(eq4(own.x, __funnelshift_r(own.x, own.y, 8))) + __popc(eq4(own.y, __funnelshift_r(own.y, own.z, 8))) +
                    __popc(eq4(own.z, __funnelshift_r(own.z, own.w, 8))) + __popc(eq4(own.w, __funnelshift_r(own.w, nb, 8))) +
                    __popc(eq4(own.x, up.x)) + __popc(eq4(own.y, up.y)) + __popc(eq4(own.z, up.z)) + __popc(eq4(own.w, up.w));
        if (DIM == 3) {
            const uint4 fr = *reinterpret_cast<const uint4 *>(sp + ((z + 1 == L) ? g - LL * (L - 1) : g + LL));
            equal += __popc(eq4(own.x, fr.x)) + __popc(eq4(own.y, fr.y)) + __popc(eq4(own.z, fr.z)) + __popc(eq4(own.w, fr.w));
        }
        e_acc += (MODEL == ISING) ? 16 * DIM - 2 * equal : 16 * DIM - equal;
        if (WITH_M) {
            const uint32_t ow[4] = {own.x, own.y, own.z, own.w};
            if (MODEL == ISING) {
                m_acc += 16 - 2 * (__popc(own.x & 0x80808080u) + __popc(own.y & 0x80808080u) + __popc(own.z & 0x80808080u) +
                                   __popc(own.w & 0x80808080u));  // +1 = 0x01, -1 = 0xff
            } else if (p.q <= 8) {
                // (every thread of the warp is in the loop or none: ngroups is a multiple of 64)
                uint32_t lo = 0u, hi = 0u;   // per-thread counts of states 0-3 / 4-7, one byte each (16 sites: no overflow)
#pragma unroll
                for (int w = 0; w < 4; ++w) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const uint32_t v = (ow[w] >> (8 * b)) & 0xffu, inc = 1u << ((v & 3u) * 8u);
                        if (v & 4u) hi += inc; else lo += inc;
                    }
                }
                for (int k = 0; k < p.q; ++k) {
                    const uint32_t c = ((k < 4 ? lo : hi) >> ((k & 3) * 8)) & 0xffu;
                    const uint32_t w = __reduce_add_sync(FULL, c);
                    if (lane == 0 && w) atomicAdd(&hist_s[k], w);
                }
            } else {
#pragma unroll
                for (int w = 0; w < 4; ++w) {
#pragma unroll
                    for (int b = 0; b < 4; ++b) atomicAdd(&hist_s[(ow[w] >> (8 * b)) & 0xffu], 1u);
                }
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e_acc += __shfl_down_sync(FULL, e_acc, o);
        m_acc += __shfl_down_sync(FULL, m_acc, o);
    }
    if (lane == 0) { red_s[0][warp] = e_acc; red_s[1][warp] = m_acc; }
    __syncthreads();
    if (tid == 0) {
        long long es = 0, ms = 0;
        for (int w = 0; w < 8; ++w) { es += red_s[0][w]; ms += red_s[1][w]; }
        atomicAdd(&p.acc->E_int, (unsigned long long)es);
        if (WITH_M && MODEL == ISING) atomicAdd(&p.acc->M_int, (unsigned long long)ms);
    }
    if (MODEL == POTTS && WITH_M) {
        if (tid < p.q && hist_s[tid]) atomicAdd(&p.acc->nk[tid], (unsigned long long)hist_s[tid]);
    }
}

// ------------------------------------------------------------------------------------------------
// k_measure_clock: the exact integer histograms of the clock model -- n[p] (sites per state, the
// paper's fmy[] table gives M from it) and D[d] (nearest-neighbour pairs per state difference, the
// paper's rule[] table gives E from it).  Shared histograms per CTA, grid-stride over the sites.
// ------------------------------------------------------------------------------------------------
template <int DIM>
__global__ void __launch_bounds__(256) k_measure_clock(const Params p)
{
    __shared__ uint32_t n_s[512], d_s[512];
    const int tid = threadIdx.x;
    for (int k = tid; k < 512; k += 256) { n_s[k] = 0u; d_s[k] = 0u; }
    __syncthreads();
    // grid-stride over the sites: a CTA keeps its shared histograms for many sites and adds them to the
    // global ones once (one CTA per 256 sites made the 2 q global atomics of every CTA the whole cost)
    const uint32_t L = p.L;
    const uint16_t *s = (const uint16_t *)p.spins;
    const int q = p.q;
    for (uint32_t i = blockIdx.x * 256u + tid; i < p.N; i += gridDim.x * 256u) {  // N is a multiple of 1024
        uint32_t x, y, z;
        decode(p, i, x, y, z);
        const int v = s[i];
        atomicAdd(&n_s[v], 1u);
        const uint32_t jx = (x + 1 == L) ? i - (L - 1) : i + 1;
        const uint32_t jy = (y + 1 == L) ? i - L * (L - 1) : i + L;
        int dx = v - (int)s[jx], dy = v - (int)s[jy];
        if (dx < 0) dx += q;
        if (dy < 0) dy += q;
        atomicAdd(&d_s[dx], 1u);
        atomicAdd(&d_s[dy], 1u);
        if (DIM == 3) {
            const uint32_t jz = (z + 1 == L) ? i - L * L * (L - 1) : i + L * L;
            int dz = v - (int)s[jz];
            if (dz < 0) dz += q;
            atomicAdd(&d_s[dz], 1u);
        }
    }
    __syncthreads();
    for (int k = tid; k < q; k += 256) {
        if (n_s[k]) atomicAdd(&p.acc->nk[k], (unsigned long long)n_s[k]);
        if (d_s[k]) atomicAdd(&p.acc->dk[k], (unsigned long long)d_s[k]);
    }
}

// ------------------------------------------------------------------------------------------------
// Cluster statistics of the last step's labelling, on request (sw_get_cluster_stats): the improved
// estimator <M^2> = <sum_c n_c^2> of the FK representation ("easy to
// extend").  k_cluster_sizes: every site adds 1 to the counter of its root; k_cluster_moments: number
// of clusters and sum of squared sizes over the non-empty counters.  Not on the hot path.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_cluster_sizes(const Params p, uint32_t *sizes)
{
    const uint32_t a0 = blockIdx.x * 256u + threadIdx.x;  // tile-major address; N is a multiple of 1024
    uint32_t a = a0;
    const int db = p.db;
    for (;;) {
        const uint32_t n = p.labels[a] >> db;
        if (n == a) break;
        a = n;
    }
    atomicAdd(&sizes[a], 1u);
}

__global__ void __launch_bounds__(256) k_cluster_moments(const Params p, const uint32_t *sizes, unsigned long long *out)
{
    const uint32_t a = blockIdx.x * 256u + threadIdx.x;
    const unsigned long long n = sizes[a];
    unsigned long long cnt = n ? 1ull : 0ull, sq = n * n;
    for (int o = 16; o > 0; o >>= 1) {
        cnt += __shfl_down_sync(FULL, cnt, o);
        sq += __shfl_down_sync(FULL, sq, o);
    }
    if ((threadIdx.x & 31) == 0 && cnt) { atomicAdd(&out[0], cnt); atomicAdd(&out[1], sq); }
}

// k_snapshot: copy the head of the accumulators (one record of a per-step series) -- sw_run_series:
// w1 words from the start, then w2 words from word offset off2 (the clock model's D[d]).
__global__ void __launch_bounds__(1024) k_snapshot(const Acc *acc, unsigned long long *dst, int w1, int off2, int w2)
{
    const unsigned long long *src = reinterpret_cast<const unsigned long long *>(acc);
    for (int k = threadIdx.x; k < w1 + w2; k += 1024) dst[k] = k < w1 ? src[k] : src[off2 + (k - w1)];
}

__global__ void k_philox_selftest(const uint32_t *ctr, const uint32_t *key, uint32_t *out, int count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

// ------------------------------------------------------------------------------------------------
// Micro-benchmarks (sw_micro_bench): the ALU cost of the random numbers alone and the rate of independent
// random 4-byte reads, the two bounds DESIGN.md section 6 quotes next to the HBM roofline.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_micro_philox_site(uint8_t *out, uint32_t n, uint32_t P32, uint32_t k0, uint32_t k1)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= n) return;
    const uint4 w = philox4x32_10(i, 7u, 0u, DOM_SITE, k0, k1);
    out[i] = (uint8_t)((w.x < P32) | ((w.y < P32) << 1) | ((w.z < P32) << 2) | ((w.w >> 31) << 3));
}

__global__ void __launch_bounds__(256) k_micro_gather(const uint32_t *table, uint32_t mask, uint32_t *out, uint32_t n)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= n) return;
    uint32_t h = i * 2654435761u;   // a cheap hash: the addresses are spread over the whole table
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
    out[i] = __ldg(table + (h & mask));
}

}  // namespace swk
