// sw_kernels.cuh -- CUDA kernels (sm_100a) of one Swendsen-Wang step, arXiv 1403.7560 section 2
// (PAPER.md:94-98).  Independent of oracle/: nothing here is shared with or derived from it.
//
// Kernels of one step t:
//   k_bond_label  (1) bond activation fused with (2a) tile-local cluster labelling in
//                 shared memory: warp-ballot run detection along x + atomicMin union-find;
//   k_merge       (2b) global atomicMin union-find over the active bonds that cross tile faces
//                 (incl. the periodic wrap), PAPER.md:97, 100-104;
//   k_flip        (2c) root chase (flatten) fused with (3) the per-cluster draw / XY reflection
//                  and the magnetisation sums of PAPER.md:142-157;
//   k_measure     energy (Eq. 1-3) and magnetisation (Eq. 4, 5) of the current configuration.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace swk {

enum { ISING = 0, POTTS = 1, XY = 2 };
constexpr uint32_t DOM_SITE = 0u, DOM_INIT = 2u, DOM_XYDIR = 3u;
constexpr uint32_t FULL = 0xffffffffu;

// Device accumulators of the observables and the labelling counters.
struct Acc {
    unsigned long long E_int;    // Ising: -sum s_i s_j (two's complement); Potts: #unequal pairs
    double E_xy;                 // XY: -sum cos(theta_i - theta_j)
    unsigned long long M_int;    // Ising: sum s_i (two's complement)
    double mx, my;               // XY: sum cos, sum sin
    unsigned long long nk[256];  // Potts: n_k
    unsigned long long stats[8]; // see sw_get_label_stats
};

struct Params {
    void *spins;       // int8 (Ising) | uint8 (Potts) | float (XY angle), N elements
    uint8_t *bonds;    // N bytes, bit k = bond i -> i + e_k
    uint32_t *labels;  // N parent pointers, label[i] <= i, roots have label[i] == i
    Acc *acc;
    uint32_t L, N;
    int log2L;         // >= 0 if L is a power of two, else -1
    uint32_t k0, k1;   // Philox key = (seed low, seed high)
    uint32_t t_lo, t_hi;
    uint32_t P32;      // Ising/Potts: bond active iff word < P32
    int q;
    float rx, ry, crefl, m2beta;  // XY: direction, reflection constant, -2 beta
    int counting;
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

__device__ __forceinline__ void decode(const Params &p, uint32_t i, uint32_t &x, uint32_t &y, uint32_t &z)
{
    if (p.log2L >= 0) {
        x = i & (p.L - 1u);
        y = (i >> p.log2L) & (p.L - 1u);
        z = i >> (2 * p.log2L);
    } else {
        x = i % p.L;
        const uint32_t r = i / p.L;
        y = r % p.L;
        z = r / p.L;
    }
}

template <int MODEL> struct ValT { using type = uint8_t; };
template <> struct ValT<XY> { using type = float; };

// ------------------------------------------------------------------------------------------------
// Shared-memory union-find (min-index roots).  Every link hangs the larger root under the smaller
// one, so the root of a finished tree is the minimum index of its set whatever the order in which
// concurrent unions land (the paper's analogue: atomicMin on labels initialised to the site index,
// PAPER.md:102).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t find_s(volatile uint32_t *lab, uint32_t x)
{
    uint32_t n;
    while ((n = lab[x]) != x) x = n;
    return x;
}

__device__ __forceinline__ void union_s(uint32_t *lab, uint32_t a, uint32_t b)
{
    for (;;) {
        a = find_s(lab, a);
        b = find_s(lab, b);
        if (a == b) return;
        if (a < b) { const uint32_t t = a; a = b; b = t; }
        const uint32_t old = atomicMin(&lab[a], b);
        if (old == a) return;  // a was a root and now hangs under b
        a = old;               // a had been linked meanwhile: go on with (old parent, b)
    }
}

// Global union-find over the label array.  Loads bypass L1 (volatile) because other CTAs update
// parents concurrently; every update is an atomicMin, so parents only ever decrease.
__device__ __forceinline__ uint32_t find_g(uint32_t *lab, uint32_t x, unsigned &hops)
{
    volatile uint32_t *vl = lab;
    for (;;) {
        const uint32_t p = vl[x];
        if (p == x) return x;
        const uint32_t gp = vl[p];
        ++hops;
        if (gp == p) return p;
        atomicMin(&lab[x], gp);  // path halving; result unused -> RED
        x = gp;
        ++hops;
    }
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
    else ((float *)p.spins)[i] = (float)(w >> 8) * (float)(6.283185307179586476925286766559 / 16777216.0);
}

// ------------------------------------------------------------------------------------------------
// k_bond_label: one CTA per TX x TY x TZ tile.
//   (XY only) stage the projections a_i = r . s_i of the tile and its +x/+y/+z faces in smem
//   rows    one warp per row of 32 sites along x: Philox(site, t) -> bond bits; the ballot of the
//           x-bond bits gives every lane the start of its run, so x-connectivity costs no union;
//           active y/z bonds inside the tile are compacted into a work list (ballot + popc)
//   unions  the work list is processed densely, one bond per thread: atomicMin union-find in smem
//   flatten label[i] = global index of the tile-local root
// Local index order (lx fastest, then ly, lz) is monotone in the global index inside a tile, so the
// tile-local minimum is the global minimum over the tile's part of the cluster.
// ------------------------------------------------------------------------------------------------
template <int DIM, int MODEL, int TX, int TY, int TZ>
struct TileGeom {
    static constexpr int SX = TX + 1, SY = TY + 1, SZ = (DIM == 3) ? TZ + 1 : 1;
    static constexpr int NS = TX * TY * TZ;
    static_assert(NS <= 8192, "work-list entries keep the local index in 13 bits");
    static constexpr int NSTAGE = (MODEL == XY) ? SX * SY * SZ : 0;
    static constexpr int NWORK = 2 * NS + NS / 32;  // every y/z bond of the tile + the x seams
    static constexpr size_t VAL_BYTES = ((size_t)NSTAGE * 4 + 15) / 16 * 16;
    static constexpr size_t OFF_LAB = VAL_BYTES;
    static constexpr size_t OFF_WORK = OFF_LAB + (size_t)NS * 4;
    static constexpr size_t SMEM_BOND_LABEL = OFF_WORK + (size_t)NWORK * 2;
    static constexpr size_t SMEM_FLIP = (size_t)NS * 4 + (size_t)NS + (size_t)NS * 2;
};

template <int DIM, int MODEL, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT) k_bond_label(const Params p)
{
    static_assert(TX % 32 == 0, "rows are warps");
    using G = TileGeom<DIM, MODEL, TX, TY, TZ>;
    constexpr int SX = G::SX, SY = G::SY, SZ = G::SZ, NS = G::NS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float *val_s = reinterpret_cast<float *>(smem_raw);
    uint32_t *lab_s = reinterpret_cast<uint32_t *>(smem_raw + G::OFF_LAB);
    uint16_t *work_s = reinterpret_cast<uint16_t *>(smem_raw + G::OFF_WORK);
    __shared__ int count_s;

    const uint32_t L = p.L;
    const uint32_t x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = (DIM == 3) ? blockIdx.z * TZ : 0u;
    const int tid = threadIdx.x;
    constexpr int ROWS = NS / 32, NW = NT / 32;
    const int lane = tid & 31, warp = tid >> 5;

    if (tid == 0) count_s = 0;
    if (MODEL == XY) {
        // a_i = r . s_i for the tile and its three plus-faces, one staged row per warp
        for (int r = warp; r < SY * SZ; r += NW) {
            const int ly = r % SY, lz = r / SY;
            const bool face = (ly == TY) || (DIM == 3 && lz == TZ);
            if (ly == TY && DIM == 3 && lz == TZ) continue;
            uint32_t gy = y0 + ly, gz = z0 + lz;
            if (gy == L) gy = 0;
            if (DIM == 3 && gz == L) gz = 0;
            const uint32_t rowbase = L * (gy + L * gz);
            for (int lx = lane; lx < SX; lx += 32) {
                if (face && lx == TX) continue;
                uint32_t gx = x0 + lx;
                if (gx == L) gx = 0;
                float sn, cs;
                sincosf(((const float *)p.spins)[rowbase + gx], &sn, &cs);
                val_s[(lz * SY + ly) * SX + lx] = p.rx * cs + p.ry * sn;
            }
        }
    }
    __syncthreads();

    for (int row = warp; row < ROWS; row += NW) {
        const int li = row * 32 + lane;
        const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
        const uint32_t gx = x0 + lx, gy = y0 + ly, gz = z0 + lz;
        const uint32_t g = gx + L * (gy + L * gz);
        const uint4 w = philox4x32_10(g, p.t_lo, p.t_hi, DOM_SITE, p.k0, p.k1);
        uint32_t b = 0;
        if (MODEL == XY) {
            // Wolff embedding: aligned iff a_i a_j > 0, p = 1 - exp(-2 beta a_i a_j)
            const int si = (lz * SY + ly) * SX + lx;
            const float scale = 5.9604644775390625e-8f;  // 2^-24
            const float v = val_s[si];
            const float px = v * val_s[si + 1];
            const float py = v * val_s[si + SX];
            if (px > 0.f && (float)(w.x >> 8) * scale < -expm1f(p.m2beta * px)) b |= 1u;
            if (py > 0.f && (float)(w.y >> 8) * scale < -expm1f(p.m2beta * py)) b |= 2u;
            if (DIM == 3) {
                const float pz = v * val_s[si + SX * SY];
                if (pz > 0.f && (float)(w.z >> 8) * scale < -expm1f(p.m2beta * pz)) b |= 4u;
            }
        } else {
            // a bond between equal neighbours is active with probability p.
            // Spins straight from global memory (the +y/+z rows hit L1: other warps load them as theirs).
            const uint8_t *sp = (const uint8_t *)p.spins;
            const uint32_t v = sp[g];
            uint32_t vx = __shfl_down_sync(FULL, v, 1);
            if (lane == 31) vx = sp[(gx + 1 == L) ? g - (L - 1) : g + 1];
            const uint32_t vy = sp[(gy + 1 == L) ? g - L * (L - 1) : g + L];
            if (v == vx && w.x < p.P32) b |= 1u;
            if (v == vy && w.y < p.P32) b |= 2u;
            if (DIM == 3) {
                const uint32_t LL = L * L;
                const uint32_t vz = sp[(gz + 1 == L) ? g - LL * (L - 1) : g + LL];
                if (v == vz && w.z < p.P32) b |= 4u;
            }
        }
        p.bonds[g] = (uint8_t)b;
        const uint32_t xm = __ballot_sync(FULL, b & 1u);
        const uint32_t below = (1u << lane) - 1u;
        const uint32_t zeros = ~xm & below;  // lanes below me whose +x bond is off
        const int start = zeros ? 32 - __clz(zeros) : 0;
        lab_s[li] = (uint32_t)(row * 32 + start);
        // compact the bonds that need a union: +y / +z inside the tile, +x across a 32-lane seam
        const bool wy = (b & 2u) && ly < TY - 1;
        const bool wz = DIM == 3 && (b & 4u) && lz < TZ - 1;
        const bool wx = TX > 32 && (b & 1u) && lane == 31 && lx < TX - 1;
        const uint32_t my = __ballot_sync(FULL, wy), mz = __ballot_sync(FULL, wz);
        const int nx = (TX > 32) ? (int)((__ballot_sync(FULL, wx) >> 31) & 1u) : 0;
        const int ny = __popc(my), nz = __popc(mz);
        int base = 0;
        if (lane == 0 && ny + nz + nx > 0) base = atomicAdd(&count_s, ny + nz + nx);
        base = __shfl_sync(FULL, base, 0);
        if (wy) work_s[base + __popc(my & below)] = (uint16_t)(li | (1u << 13));
        if (wz) work_s[base + ny + __popc(mz & below)] = (uint16_t)(li | (2u << 13));
        if (wx) work_s[base + ny + nz] = (uint16_t)li;
    }
    __syncthreads();

    const int nwork = count_s;
    for (int e0 = 0; e0 < nwork; e0 += NT) {
        const int e = e0 + tid;
        if (e < nwork) {
            const uint32_t wk = work_s[e];
            const uint32_t a = wk & 0x1fffu, d = wk >> 13;
            union_s(lab_s, a, a + (d == 0 ? 1u : (d == 1 ? (uint32_t)TX : (uint32_t)(TX * TY))));
        }
        __syncwarp();
    }
    __syncthreads();

    for (int row = warp; row < ROWS; row += NW) {
        const int li = row * 32 + lane;
        const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
        const uint32_t g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
        const uint32_t r = find_s(lab_s, li);
        __syncwarp();
        const int rx = r % TX, ry = (r / TX) % TY, rz = r / (TX * TY);
        p.labels[g] = (x0 + rx) + L * ((y0 + ry) + L * (z0 + rz));
    }
}

// ------------------------------------------------------------------------------------------------
// k_merge: one thread per bond slot that crosses a tile face (family k: sites whose coordinate k is
// the last of its tile; includes the periodic wrap faces).  Lock-free min-root union with retry.
// Thread 0 also clears the magnetisation accumulators that k_flip adds to.
// ------------------------------------------------------------------------------------------------
template <int DIM, int TX, int TY, int TZ>
__global__ void __launch_bounds__(256) k_merge(const Params p)
{
    const uint32_t L = p.L;
    const uint32_t n0 = p.N / TX, n1 = p.N / TY, n2 = (DIM == 3) ? p.N / TZ : 0u;
    uint32_t s = blockIdx.x * 256u + threadIdx.x;
    if (s == 0) {
        p.acc->M_int = 0ull; p.acc->mx = 0.0; p.acc->my = 0.0;
        for (int k = 0; k < p.q; ++k) p.acc->nk[k] = 0ull;
    }
    uint32_t i, j;
    int k;
    if (s < n0) {
        k = 0;
        const uint32_t ntx = L / TX;
        const uint32_t xt = s % ntx, rest = s / ntx;
        const uint32_t x = xt * TX + (TX - 1);
        i = x + L * rest;
        j = (x + 1 == L) ? i - (L - 1) : i + 1;
    } else if (s < n0 + n1) {
        k = 1;
        s -= n0;
        const uint32_t nty = L / TY;
        const uint32_t x = s % L, rest = s / L;
        const uint32_t yt = rest % nty, z = rest / nty;
        const uint32_t y = yt * TY + (TY - 1);
        i = x + L * (y + L * z);
        j = (y + 1 == L) ? i - L * (L - 1) : i + L;
    } else if (s < n0 + n1 + n2) {
        k = 2;
        s -= n0 + n1;
        const uint32_t LL = L * L;
        const uint32_t xy = s % LL, zt = s / LL;
        const uint32_t z = zt * TZ + (TZ - 1);
        i = xy + LL * z;
        j = (z + 1 == L) ? xy : i + LL;
    } else {
        return;
    }
    const bool active = (p.bonds[i] >> k) & 1u;
    if (p.counting) {
        atomicAdd(&p.acc->stats[0], 1ull);
        if (active) atomicAdd(&p.acc->stats[1], 1ull);
    }
    if (!active) return;
    uint32_t a = p.labels[i], b = p.labels[j];
    unsigned hops = 0, retries = 0, linked = 0, maxhops = 0;
    for (;;) {
        unsigned h = 0;
        a = find_g(p.labels, a, h);
        b = find_g(p.labels, b, h);
        hops += h;
        maxhops = h > maxhops ? h : maxhops;
        if (a == b) break;
        if (a < b) { const uint32_t t = a; a = b; b = t; }
        const uint32_t old = atomicMin(&p.labels[a], b);
        if (old == a) { linked = 1; break; }
        a = old;
        ++retries;
    }
    if (p.counting) {
        atomicAdd(&p.acc->stats[2], (unsigned long long)linked);
        atomicAdd(&p.acc->stats[3], (unsigned long long)retries);
        atomicAdd(&p.acc->stats[4], (unsigned long long)hops);
        atomicMax(&p.acc->stats[5], (unsigned long long)maxhops);
    }
}

// ------------------------------------------------------------------------------------------------
// k_flip: one CTA per tile.
//   phase A   every site reads its parent; sites whose parent is themselves or lies outside the tile
//             (the former tile-local roots) are compacted into a list, the others park a tile-local
//             pointer in smem
//   phase A2  the list is processed densely, one root per thread: chase the global root r, draw the
//             cluster's new value from word 3 of Philox(r, t), park (r, draw) in smem
//   phase B   the other sites follow the tile-local pointers in smem to a parked entry
//   then      new spin / XY reflection written in place, magnetisation sums reduced per CTA
// ------------------------------------------------------------------------------------------------
constexpr uint32_t LOCAL_PTR = 0x80000000u;

template <int DIM, int MODEL, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT) k_flip(const Params p)
{
    using G = TileGeom<DIM, MODEL, TX, TY, TZ>;
    constexpr int NS = G::NS;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint32_t *res_s = reinterpret_cast<uint32_t *>(smem_raw);
    uint16_t *root_s = reinterpret_cast<uint16_t *>(smem_raw + (size_t)NS * 4);
    uint8_t *draw_s = reinterpret_cast<uint8_t *>(smem_raw + (size_t)NS * 6);
    __shared__ unsigned long long hist_s[256];
    __shared__ double red_s[2][32];
    __shared__ int count_s;

    const uint32_t L = p.L;
    const uint32_t x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = (DIM == 3) ? blockIdx.z * TZ : 0u;
    const int tid = threadIdx.x;
    constexpr int ROWS = NS / 32, NW = NT / 32;
    const int lane = tid & 31, warp = tid >> 5;
    const uint32_t below = (1u << lane) - 1u;

    if (tid == 0) count_s = 0;
    if (MODEL == POTTS) {
        for (int k = tid; k < 256; k += NT) hist_s[k] = 0ull;
    }
    __syncthreads();

    for (int row = warp; row < ROWS; row += NW) {
        const int li = row * 32 + lane;
        const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
        const uint32_t g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
        const uint32_t par = p.labels[g];
        uint32_t px, py, pz;
        decode(p, par, px, py, pz);
        const uint32_t dx = px - x0, dy = py - y0, dz = pz - z0;
        const bool in_tile = dx < (uint32_t)TX && dy < (uint32_t)TY && dz < (uint32_t)TZ;
        const bool is_root = (par == g) || !in_tile;
        res_s[li] = is_root ? par : (LOCAL_PTR | (dx + TX * (dy + TY * dz)));
        const uint32_t m = __ballot_sync(FULL, is_root);
        int base = 0;
        if (lane == 0 && m) base = atomicAdd(&count_s, __popc(m));
        base = __shfl_sync(FULL, base, 0);
        if (is_root) root_s[base + __popc(m & below)] = (uint16_t)li;
    }
    __syncthreads();

    const int nroots = count_s;
    unsigned chase_hops = 0, chase_max = 0;
    for (int e0 = 0; e0 < nroots; e0 += NT) {
        const int e = e0 + tid;
        if (e < nroots) {
            const int li = root_s[e];
            uint32_t r = res_s[li], n;
            unsigned h = 0;
            while ((n = p.labels[r]) != r) { r = n; ++h; }
            chase_hops += h;
            chase_max = h > chase_max ? h : chase_max;
            const uint32_t w = philox4x32_10(r, p.t_lo, p.t_hi, DOM_SITE, p.k0, p.k1).w;
            res_s[li] = r;
            draw_s[li] = (MODEL == POTTS) ? (uint8_t)(((unsigned long long)w * (unsigned)p.q) >> 32)
                                          : (uint8_t)(w >> 31);
        }
        __syncwarp();
    }
    __syncthreads();

    long long m_loc = 0;
    double cx = 0.0, cy = 0.0;
    for (int row = warp; row < ROWS; row += NW) {
        const int li = row * 32 + lane;
        const int lx = li % TX, ly = (li / TX) % TY, lz = li / (TX * TY);
        const uint32_t g = (x0 + lx) + L * ((y0 + ly) + L * (z0 + lz));
        uint32_t at = li, v = res_s[li];
        while (v & LOCAL_PTR) { at = v & ~LOCAL_PTR; v = res_s[at]; }
        __syncwarp();
        const uint32_t d = draw_s[at];
        if (MODEL == ISING) {
            // "All spins in each cluster are set randomly to +1 or -1"
            const int s = d ? 1 : -1;
            ((int8_t *)p.spins)[g] = (int8_t)s;
            m_loc += s;
        } else if (MODEL == POTTS) {
            ((uint8_t *)p.spins)[g] = (uint8_t)d;
            if (p.q <= 8) {
                for (int k = 0; k < p.q; ++k) {
                    const unsigned c = __popc(__ballot_sync(FULL, d == (uint32_t)k));
                    if (lane == 0) atomicAdd(&hist_s[k], (unsigned long long)c);
                }
            } else {
                atomicAdd(&hist_s[d], 1ull);
            }
        } else {
            // PAPER.md:159 mirror projection: theta' = c - theta, wrapped into [0, 2 pi]
            float th = ((float *)p.spins)[g];
            if (d) {
                th = p.crefl - th;
                if (th < 0.0f) th = th + 6.283185307179586476925286766559f;
                ((float *)p.spins)[g] = th;
            }
            float sn, cs;
            sincosf(th, &sn, &cs);
            cx += (double)cs;
            cy += (double)sn;
        }
    }

    if (MODEL == ISING) {
        int m = (int)m_loc;
        m = __reduce_add_sync(FULL, m);
        if (lane == 0) atomicAdd(&p.acc->M_int, (unsigned long long)(long long)m);
    } else if (MODEL == POTTS) {
        __syncthreads();
        for (int k = tid; k < p.q; k += NT)
            if (hist_s[k]) atomicAdd(&p.acc->nk[k], hist_s[k]);
    } else {
        for (int o = 16; o > 0; o >>= 1) {
            cx += __shfl_down_sync(FULL, cx, o);
            cy += __shfl_down_sync(FULL, cy, o);
        }
        if (lane == 0) { red_s[0][warp] = cx; red_s[1][warp] = cy; }
        __syncthreads();
        if (warp == 0) {
            cx = lane < NW ? red_s[0][lane] : 0.0;
            cy = lane < NW ? red_s[1][lane] : 0.0;
            for (int o = 16; o > 0; o >>= 1) {
                cx += __shfl_down_sync(FULL, cx, o);
                cy += __shfl_down_sync(FULL, cy, o);
            }
            if (lane == 0) { atomicAdd(&p.acc->mx, cx); atomicAdd(&p.acc->my, cy); }
        }
    }
    if (p.counting) {
        atomicAdd(&p.acc->stats[6], (unsigned long long)chase_hops);
        atomicMax(&p.acc->stats[7], (unsigned long long)chase_max);
    }
}

// ------------------------------------------------------------------------------------------------
// k_flatten: label[i] <- root of i, in place (parents only decrease, so concurrent readers are safe).
// Only run on request (sw_get_labels): the step itself never needs the flat array.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_flatten(const Params p)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= p.N) return;
    uint32_t r = p.labels[i], n;
    while ((n = p.labels[r]) != r) r = n;
    p.labels[i] = r;
}

// ------------------------------------------------------------------------------------------------
// k_measure: E (Eq. 1-3) and, if WITH_M, the magnetisation sums (Eq. 4, 5) of the configuration.
// One thread per site, its d owned bonds; block reduction, one atomic per CTA and quantity.
// ------------------------------------------------------------------------------------------------
template <int DIM, int MODEL, bool WITH_M>
__global__ void __launch_bounds__(256) k_measure(const Params p)
{
    __shared__ unsigned long long hist_s[256];
    __shared__ double red_s[3][8];
    __shared__ long long redi_s[2][8];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t i = blockIdx.x * 256u + tid;  // N is a multiple of 1024
    const uint32_t L = p.L;
    if (MODEL == POTTS && WITH_M) {
        hist_s[tid] = 0ull;
        __syncthreads();
    }
    uint32_t x, y, z;
    decode(p, i, x, y, z);
    const uint32_t jx = (x + 1 == L) ? i - (L - 1) : i + 1;
    const uint32_t jy = (y + 1 == L) ? i - L * (L - 1) : i + L;
    const uint32_t jz = (DIM == 3) ? ((z + 1 == L) ? i - L * L * (L - 1) : i + L * L) : 0u;
    long long e = 0, m = 0;
    double ex = 0.0, cx = 0.0, cy = 0.0;
    if (MODEL == ISING) {
        const int8_t *s = (const int8_t *)p.spins;
        const int v = s[i];
        e = -(v * s[jx] + v * s[jy] + (DIM == 3 ? v * s[jz] : 0));
        m = v;
    } else if (MODEL == POTTS) {
        const uint8_t *s = (const uint8_t *)p.spins;
        const uint32_t v = s[i];
        e = (v != s[jx]) + (v != s[jy]) + (DIM == 3 ? (v != s[jz]) : 0);
        if (WITH_M) atomicAdd(&hist_s[v], 1ull);
    } else {
        const float *s = (const float *)p.spins;
        const float v = s[i];
        ex = -((double)cosf(v - s[jx]) + (double)cosf(v - s[jy]) + (DIM == 3 ? (double)cosf(v - s[jz]) : 0.0));
        if (WITH_M) {
            float sn, cs;
            sincosf(v, &sn, &cs);
            cx = cs; cy = sn;
        }
    }
    if (MODEL == XY) {
        for (int o = 16; o > 0; o >>= 1) {
            ex += __shfl_down_sync(FULL, ex, o);
            cx += __shfl_down_sync(FULL, cx, o);
            cy += __shfl_down_sync(FULL, cy, o);
        }
        if (lane == 0) { red_s[0][warp] = ex; red_s[1][warp] = cx; red_s[2][warp] = cy; }
        __syncthreads();
        if (tid == 0) {
            for (int w = 1; w < 8; ++w) { ex += red_s[0][w]; cx += red_s[1][w]; cy += red_s[2][w]; }
            atomicAdd(&p.acc->E_xy, ex);
            if (WITH_M) { atomicAdd(&p.acc->mx, cx); atomicAdd(&p.acc->my, cy); }
        }
    } else {
        int ei = __reduce_add_sync(FULL, (int)e), mi = __reduce_add_sync(FULL, (int)m);
        if (lane == 0) { redi_s[0][warp] = ei; redi_s[1][warp] = mi; }
        __syncthreads();
        if (tid == 0) {
            long long es = 0, ms = 0;
            for (int w = 0; w < 8; ++w) { es += redi_s[0][w]; ms += redi_s[1][w]; }
            atomicAdd(&p.acc->E_int, (unsigned long long)es);
            if (WITH_M && MODEL == ISING) atomicAdd(&p.acc->M_int, (unsigned long long)ms);
        }
        if (MODEL == POTTS && WITH_M) {
            if (tid < p.q && hist_s[tid]) atomicAdd(&p.acc->nk[tid], hist_s[tid]);
        }
    }
}

__global__ void k_philox_selftest(const uint32_t *ctr, const uint32_t *key, uint32_t *out, int count)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= count) return;
    const uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

}  // namespace swk
