// sw_rows.cuh -- k_bond_label_rows: bond activation fused with the tile-local part
// of the cluster labelling.  Ising, q-state Potts and the q-state clock model by
// default, XY on request (sw_api.cu use_rows).  Independent of oracle/.
//
// The unit of work is a ROW: 32 consecutive sites along x, held as 32-bit masks (bit x = site x of the
// row; tiles are 32 sites wide, "nx ... multiple of 32").
//   phase 1a  [thread = row] (Ising) spins of the thread's R rows -> sign masks in shared memory (+ halo rows)
//   phase 1b  [thread = row] Ising / Potts: the random decisions of the row's 32 x DIM bonds from the
//             transposed uniform integers of DESIGN.md reading 6 (13 binary digits = 10 Philox calls per row
//             in 3D settle every bond of the row in 99.6 % of the cases, further digits are drawn only when
//             some site is still undecided), AND-ed with the equality masks -> bond masks Bx, By, Bz.
//             [warp = 32 rows, lane = x] XY / clock: per-site decisions (the probability depends on the two
//             spins), three ballots per row give the same masks.
//             Bx gives the x-runs of the row with no union at all.  Bonds through the tile faces go to face
//             words (-> global pair list, k_merge).  Nodes of the tile-local union-find are the RUN STARTS;
//             the run start of a site is one bfind on the row's Bx mask.  16-bit parent entries that hold the
//             shared-window address of the parent's entry (a chain is followed with no address arithmetic).
//   phase 2a  [thread = row] "pull": every run looks back at the bonds that reach it from the row below
//             (y - 1) and the row behind (z - 1); the first such bond of the run makes the run start it
//             comes from the parent of this run start -- a plain store, no atomic, no retry, because only
//             the owner of a row writes the row's entries in this phase.  Which bond of a run is the first
//             is settled for all 32 sites at once by a carry trick on the masks.  Further bonds into the
//             same run (minus twins joining the same two runs) are appended to a list.
//   phase 2b  [all threads] the listed bonds go through a lock-free union-find (CAS: larger root under
//             smaller, so that the root of a tree is its minimum index; path halving on the
//             way up).  Lanes take the next bond of their warp's share as soon as they are free.
//   phase 3   [lane = x] per site: run start, a few dependent parent loads, label word =
//             (address of the ancestor reached << DB) | own draw, coalesced stores.  Whatever is left of a
//             longer chain is followed by k_merge / k_flip.  The pair list hands k_merge the same ancestor
//             for this tile's end of every face bond.
// Label words, pair list and bond bytes are the ones of sw_kernels.cuh (k_merge / k_flip read them).
#pragma once
#include "sw_kernels.cuh"

namespace swk {

// reading 6, domain GROUP: W_G[n] = word n % 4 of the call with counter word 3 = DOM_GROUP + 256 (n / 4)
constexpr uint32_t GROUP_DRAW_BASE = 128u;

#ifndef SW_ROW_UF_MERGED
#define SW_ROW_UF_MERGED 1   // phase 2b: a climb that ends at two roots hooks them in the same round
#endif
#ifndef SW_ROW_EARLY_RANDOM
#define SW_ROW_EARLY_RANDOM 1   // 2D Ising / Potts, R = 1: the row's random decisions before the spins arrive
#endif
#ifndef SW_ROW_P3_UNROLL
#define SW_ROW_P3_UNROLL 4   // rows of phase 3 in flight per warp (1 / 2 / 4: C2 kernel 0.0632 / 0.0614 / 0.0600 ms, C4 0.447 / 0.439 / 0.439)
#endif
#ifndef SW_ROW_JUMPS
#define SW_ROW_JUMPS 3   // parent loads per site in phase 3 after the one of its run start
#endif

template <int DIM, int MODEL, int TY, int TZ>
struct RowGeom {
    static_assert(DIM == 3 || TZ == 1, "2D tiles have TZ = 1");
    static_assert(DIM == 2 || TY == 32, "3D: the 32 lanes of a warp are the 32 rows of one z-plane of the tile");
    static constexpr int NROWS = TY * TZ, NS = 32 * NROWS;
    static constexpr int LOG2NS = ilog2(NS);
    static_assert((1 << LOG2NS) == NS && NS <= 16384, "tile sizes are powers of two; the shared-window address of a parent entry fits 16 bits");
    static constexpr int NDIR = DIM - 1;                         // pending directions: y (and z)
    // face words: +x face one bit per row; +y face one word per z (the row y = TY-1); +z face one word per y
    static constexpr int FXW = NROWS / 32, FYW = TZ, FZW = (DIM == 3) ? TY : 0;
    static constexpr int NFW = FXW + FYW + FZW;
    static constexpr int NFWP = (NFW + 3) / 4 * 4;
    static_assert(NFW <= 64, "two face words per lane of warp 0");
    // sign masks of the tile's rows and of the halo rows at y = TY and z = TZ
    static constexpr int SGY = TY + 1;
    static constexpr int NSG = (DIM == 3) ? SGY * (TZ + 1) : SGY;
    // shared memory, 32-bit words
    static constexpr int OFF_BX = NS / 2;                   // after the 16-bit parent entries: Bx of every row (face bit cleared)
    static constexpr int OFF_PM = OFF_BX + NROWS;           // pending masks [dir][row]
    static constexpr int OFF_DR = OFF_PM + NDIR * NROWS;    // Ising: draw mask of every row; Potts: one draw byte per site
    static constexpr int OFF_SG = OFF_DR + (MODEL != POTTS ? NROWS : NS / 4);
    static constexpr int OFF_FACE = OFF_SG + (NSG + 3) / 4 * 4;
    static constexpr int OFF_FPRE = OFF_FACE + NFWP;     // NFW prefix counts, [NFWP] = base in the pair list, [NFWP+1] = list length, [NFWP+2] = its valid part
    static constexpr int OFF_LIST = OFF_FPRE + NFWP + 4; // bonds left for the union-find: (node a << 16) | node b
    // (the 3D Ising and XY tiles of 16 planes keep a sixth: 54.7 KB per CTA, so that four CTAs of 512 threads fit one SM)
    static constexpr int LIST_CAP = (DIM == 3 && TZ == 16 && (MODEL == ISING || MODEL == XY)) ? NS / 6 : NS / 4;
    static constexpr int WORDS = OFF_LIST + LIST_CAP;
    static constexpr size_t smem_bytes = (size_t)WORDS * 4;
};

// 16 spin bytes (+1 = 0x01, -1 = 0xff) -> 16 sign bits
__device__ __forceinline__ uint32_t sign16(const uint4 v)
{
    const uint32_t n0 = ((v.x & 0x80808080u) * 0x00204081u) >> 28;
    const uint32_t n1 = ((v.y & 0x80808080u) * 0x00204081u) >> 28;
    const uint32_t n2 = ((v.z & 0x80808080u) * 0x00204081u) >> 28;
    const uint32_t n3 = ((v.w & 0x80808080u) * 0x00204081u) >> 28;
    return n0 | (n1 << 4) | (n2 << 8) | (n3 << 12);
}
__device__ __forceinline__ uint32_t sign32(const uint4 *row)
{
    const uint4 a = row[0], b = row[1];
    return sign16(a) | (sign16(b) << 16);
}

// 4-bit equality nibble of two words of 4 bytes, at bit position sh
__device__ __forceinline__ uint32_t eqnib(uint32_t a, uint32_t b) { return eq4(a, b); }

// 32 bytes against 32 bytes -> 32 equality bits
__device__ __forceinline__ uint32_t eq32(const uint32_t (&a)[8], const uint32_t (&b)[8])
{
    uint32_t m = 0u;
#pragma unroll
    for (int j = 0; j < 8; ++j) m |= eq4(a[j], b[j]) << (4 * j);
    return m;
}

__device__ __forceinline__ uint32_t lds_u32(uint32_t saddr)
{
    uint32_t v;
    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t saddr)
{
    uint32_t v;   // (a 32-bit destination: the load zero-extends, no conversion instruction follows)
    asm volatile("ld.volatile.shared.u16 %0, [%1];" : "=r"(v) : "r"(saddr) : "memory");
    return v;
}
// v <- 16-bit shared[saddr] if flag != 0 (predicated: no branch, no shared-memory wavefront when off)
__device__ __forceinline__ void lds_u16_if(uint32_t &v, uint32_t flag, uint32_t saddr)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %1, 0;\n\t@p ld.shared.u16 %0, [%2];\n\t}"
                 : "+r"(v) : "r"(flag), "r"(saddr) : "memory");
}
__device__ __forceinline__ void sts_u16(uint32_t saddr, uint32_t v)
{
    asm volatile("st.volatile.shared.u16 [%0], %1;" :: "r"(saddr), "r"(v) : "memory");   // (the low 16 bits of v)
}
__device__ __forceinline__ uint32_t cas_shared(uint32_t saddr, uint32_t cmp, uint32_t val)
{
    uint32_t old;
    asm volatile("atom.shared.cas.b32 %0, [%1], %2, %3;" : "=r"(old) : "r"(saddr), "r"(cmp), "r"(val) : "memory");
    return old;
}
// Compare-and-swap of one 16-bit parent entry through the 32-bit word that holds it (there is no native
// 16-bit shared-memory CAS): returns the entry's old value (== cmp on success).
__device__ __forceinline__ uint32_t cas_u16(uint32_t saddr, uint32_t cmp, uint32_t val)
{
    const uint32_t wa = saddr & ~3u, sh = (saddr & 2u) << 3;
    uint32_t old = lds_u32(wa);
    for (;;) {
        const uint32_t cur = (old >> sh) & 0xffffu;
        if (cur != cmp) return cur;
        const uint32_t got = cas_shared(wa, old, (old & ~(0xffffu << sh)) | (val << sh));
        if (got == old) return cmp;
        old = got;
    }
}
// Lock-free union of the trees of nodes a and b.  A node is 2 x the local index of a run start (k_sw_small; lab = the
// shared-window address of the entries) or the shared-window address of its entry itself (k_bond_label_rows; lab = 0); its
// 16-bit parent entry sits at lab + node; a root points to itself; every link hangs the larger root under
// a smaller node, so the root of a tree is its minimum index.
__device__ __forceinline__ void union_nodes(uint32_t lab, uint32_t a, uint32_t b)
{
    for (;;) {
        uint32_t pa = lds_u16(lab + a), pb = lds_u16(lab + b);
        while (pa != a || pb != b) { a = pa; b = pb; pa = lds_u16(lab + a); pb = lds_u16(lab + b); }
        if (a == b) return;
        const uint32_t hi = max(a, b), lo = min(a, b);
        const uint32_t old = cas_u16(lab + hi, hi, lo);
        if (old == hi) return;
        a = old; b = lo;
    }
}
// The same with path halving on the way up (every node visited is re-pointed to its grandparent: a non-root is never
// the target of a hook, and any ancestor is a valid parent) -- for the bonds that found no room in the list (ordered
// phase), which a thread works off one after the other.
__device__ __forceinline__ void union_nodes_halving(uint32_t a, uint32_t b)
{
    for (;;) {
        for (;;) {
            const uint32_t pa = lds_u16(a), pb = lds_u16(b);
            if (pa == a && pb == b) break;
            const uint32_t ga = lds_u16(pa), gb = lds_u16(pb);
            if (ga != pa) sts_u16(a, ga);
            if (gb != pb) sts_u16(b, gb);
            a = ga; b = gb;
        }
        if (a == b) return;
        const uint32_t hi = max(a, b), lo = min(a, b);
        const uint32_t old = cas_u16(hi, hi, lo);
        if (old == hi) return;
        a = old; b = lo;
    }
}
// start of the x-run of site x (below = mask of the bits under x): one past the highest inactive x-bond under it
__device__ __forceinline__ uint32_t run_start(uint32_t bx, uint32_t below)
{
    uint32_t f;   // bfind: position of the highest set bit, 0xffffffff if there is none (one instruction; 32 - clz takes three)
    asm("bfind.u32 %0, %1;" : "=r"(f) : "r"(~bx & below));
    return f + 1u;
}

// The random decisions "u < P32" of the 32 x DIM bonds of group G (reading 6): X[k] bit b = decision
// of bond k of site b; D = W_G[0] (Ising draw bits).  Digits are compared most significant first:
// und[k] holds the sites whose digits so far equal those of P32.
template <int DIM>
__device__ __forceinline__ void group_decisions(const Params &p, uint32_t G, uint32_t t_lo, uint32_t t_hi,
                                                uint32_t (&X)[3], uint32_t &D)
{
    constexpr int NC = (DIM == 3) ? 10 : 7;                 // eager calls: 13 digits per direction
    constexpr int NCMAX = (1 + 32 * DIM + 3) / 4;           // all 32 digits
    const uint32_t P = p.P32;
    uint32_t U[3] = {FULL, FULL, FULL};
    X[0] = X[1] = X[2] = 0u;
    D = 0u;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const uint4 w4 = philox4x32_10(G, t_lo, t_hi, DOM_GROUP + 256u * (uint32_t)c, p.k0, p.k1);
        const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = 4 * c + j;
            if (n == 0) { D = w[0]; continue; }
            const int s = (n - 1) / DIM, k = (n - 1) % DIM;
            // digit 31 - s of P32 (warp-uniform): 1 -> sites whose digit is 0 are decided "u < P32", the others
            // stay undecided; 0 -> sites whose digit is 1 are decided "u > P32", the others stay undecided
            if ((P >> (31 - s)) & 1u) { X[k] |= U[k] & ~w[j]; U[k] &= w[j]; }
            else U[k] &= ~w[j];
        }
    }
    uint32_t und = U[0] | U[1] | (DIM == 3 ? U[2] : 0u);
    for (int c = NC; c < NCMAX && __any_sync(FULL, und != 0u); ++c) {
        const uint4 w4 = philox4x32_10(G, t_lo, t_hi, DOM_GROUP + 256u * (uint32_t)c, p.k0, p.k1);
        const uint32_t w[4] = {w4.x, w4.y, w4.z, w4.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int n = 4 * c + j;
            const int s = (n - 1) / DIM, k = (n - 1) - s * DIM;
            if (s < 32) {
                const uint32_t pm = (uint32_t)((int32_t)(P << s) >> 31);
#pragma unroll
                for (int kk = 0; kk < DIM; ++kk) {
                    if (kk == k) {
                        X[kk] |= U[kk] & ~w[j] & pm;
                        U[kk] &= ~(w[j] ^ pm);
                    }
                }
            }
        }
        und = U[0] | U[1] | (DIM == 3 ? U[2] : 0u);
    }
}

// sw_micro_bench: group_decisions alone, one group of 32 sites per thread
__global__ void __launch_bounds__(256) k_micro_philox_group(uint32_t *out, uint32_t ngroups, const Params p)
{
    const uint32_t G = blockIdx.x * 256u + threadIdx.x;   // ngroups is a multiple of 256 (whole warps: __any_sync)
    uint32_t X[3], D;
    group_decisions<3>(p, G, 7u, 0u, X, D);
    if (G < ngroups) { out[3u * G] = X[0] ^ D; out[3u * G + 1u] = X[1]; out[3u * G + 2u] = X[2]; }
}

template <int DIM, int MODEL, int TY, int TZ, int R>
struct RowKernelTraits {
    static constexpr int NT = (DIM == 3) ? 32 * TZ / R : TY / R;
    static_assert(NT % 32 == 0 && NT >= 32 && NT <= 1024, "whole warps");
    static_assert(DIM == 2 || TZ % R == 0, "R rows along z per thread");
};

template <int DIM, int MODEL, int TY, int TZ, int R, int MINB>
__global__ void __launch_bounds__((RowKernelTraits<DIM, MODEL, TY, TZ, R>::NT), MINB) k_bond_label_rows(const Params p)
{
    using G = RowGeom<DIM, MODEL, TY, TZ>;
    constexpr int NT = RowKernelTraits<DIM, MODEL, TY, TZ, R>::NT;
    constexpr int NROWS = G::NROWS, NW = NT / 32;
    static_assert(R == 1 || MODEL == ISING || MODEL == POTTS, "XY / clock: the 32 threads of a warp make the masks of their 32 rows together");
    extern __shared__ __align__(16) uint32_t smem_u32[];
    uint32_t *lab_s = smem_u32;                       // 16-bit parent entries, one per site: node of the parent
    uint32_t *bx_s = smem_u32 + G::OFF_BX;
    uint32_t *pm_s = smem_u32 + G::OFF_PM;
    uint32_t *dr_s = smem_u32 + G::OFF_DR;
    uint32_t *sg_s = smem_u32 + G::OFF_SG;
    uint32_t *face_s = smem_u32 + G::OFF_FACE;
    uint32_t *fpre_s = smem_u32 + G::OFF_FPRE;        // NFW prefix counts, [NFWP] = base in the global pair list, [NFWP+1] = list length
    uint32_t *list_s = smem_u32 + G::OFF_LIST;
    // A node of the tile-local forest is the shared-window ADDRESS of its 16-bit parent entry (lab_sa + 2 x local index;
    // the entries are the first thing in dynamic shared memory, so the address fits 16 bits): an entry is followed with a
    // load from the value just read, no base address is added in the loops.
    const uint32_t lab_sa = (uint32_t)__cvta_generic_to_shared(lab_s);
    if (lab_sa + 2u * (uint32_t)G::NS > 65536u) __trap();

    const uint32_t L = p.L, LL = L * L;
    const uint32_t bx = blockIdx.x, by = blockIdx.y, bz = (DIM == 3) ? blockIdx.z : 0u;
    const uint32_t x0 = bx * 32u, y0 = by * TY, z0 = bz * TZ;
    const uint32_t tile = bx + p.ntx * (by + p.nty * bz);
    const uint32_t tile_base = tile << G::LOG2NS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned long long t_step = p.acc->t;
    const uint32_t t_lo = (uint32_t)t_step, t_hi = (uint32_t)(t_step >> 32);
    const uint8_t *sp = (const uint8_t *)p.spins;
    const uint32_t xh = (x0 + 32u == L) ? 0u : x0 + 32u;   // x of the +x halo column

    // rows of this thread: r = 0 .. R-1 -> (ly, lz); local row index = ly + TY lz; site = x + 32 row
    auto row_y = [&](int r) -> int { return (DIM == 3) ? lane : tid * R + r; };
    auto row_z = [&](int r) -> int { return (DIM == 3) ? warp * R + r : 0; };
    auto grow = [&](int ly, int lz) -> uint32_t {            // linear index of the first site of a row (periodic)
        uint32_t gy = y0 + (uint32_t)ly, gz = z0 + (uint32_t)lz;
        if (gy >= L) gy -= L;
        if (DIM == 3 && gz >= L) gz -= L;
        return L * gy + (DIM == 3 ? LL * gz : 0u);
    };

    // 2D Ising / Potts, one row per thread: the spins are requested (L2 prefetch) and the random decisions of the row, which need
    // no spin, are made while they are on their way -- the DRAM latency at the start of the CTA is hidden behind the
    // ten Philox calls instead of being waited for at the first barrier.
    constexpr bool EARLY_RANDOM = SW_ROW_EARLY_RANDOM && (MODEL == ISING || MODEL == POTTS) && R == 1 && DIM == 2;   // (3D: Ising spills at 32 registers, Potts 0.096 vs 0.090 ms)
    uint32_t Xe[3] = {0u, 0u, 0u}, De = 0u;
    if (EARLY_RANDOM) {
        const int ly = row_y(0), lz = row_z(0);
        const uint32_t g0 = grow(ly, lz);
        asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + g0));
        asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + xh + g0));
        if (MODEL == POTTS) {   // (Potts reads the +y / +z rows itself: no halo masks in shared memory)
            asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + grow(ly + 1, lz)));
            if (DIM == 3) asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + grow(ly, lz + 1)));
        } else if (DIM == 3) {
            if (warp == NW - 1 && lane < TZ) asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + grow(TY, lane)));
            if (warp == 0) asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + grow(lane, TZ)));
        } else if (tid == NT - 1) asm volatile("prefetch.global.L2 [%0];" :: "l"(sp + x0 + grow(TY, 0)));
        group_decisions<DIM>(p, (x0 + g0) >> 5, t_lo, t_hi, Xe, De);
    }

    if (MODEL == ISING) {
        // phase 1a: sign masks of the own rows and of the halo rows (+y halo: one row per z, taken by the
        // first lanes of the last warp; +z halo: one row per y, taken by warp 0)
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int ly = row_y(r), lz = row_z(r);
            sg_s[ly + G::SGY * lz] = sign32(reinterpret_cast<const uint4 *>(sp + x0 + grow(ly, lz)));
        }
        if (DIM == 3) {
            if (warp == NW - 1 && lane < TZ)
                sg_s[TY + G::SGY * lane] = sign32(reinterpret_cast<const uint4 *>(sp + x0 + grow(TY, lane)));
            if (warp == 0)
                sg_s[lane + G::SGY * TZ] = sign32(reinterpret_cast<const uint4 *>(sp + x0 + grow(lane, TZ)));
        } else {
            if (tid == NT - 1) sg_s[TY] = sign32(reinterpret_cast<const uint4 *>(sp + x0 + grow(TY, 0)));
        }
    }
    if (tid == 0) { fpre_s[G::NFWP + 1] = 0u; fpre_s[G::NFWP + 2] = (uint32_t)G::LIST_CAP; }
    __syncthreads();

    // phase 1b: bond masks of the own rows
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const int ly = row_y(r), lz = row_z(r);
        const int row = ly + TY * lz;
        const uint32_t g0 = grow(ly, lz);
        uint32_t Bx, By, Bz = 0u, D = 0u;
        if (MODEL == XY || MODEL == CLOCK) {
            // XY (Wolff embedding) and the q-state clock model (readings 23-25): the bond
            // probability depends on the two spins, so the decisions are made per site with the per-site
            // keying (domain SITE: word k decides bond k, the top bit of word 3 is the cluster draw).  The 32
            // threads of a warp own 32 rows that follow each other in y; they take these rows one at a time
            // with lane = x, from the last to the first, so that the row done before is the +y neighbour
            // (its projections are still in registers); +x comes by shuffle, +z is computed again from the
            // neighbour's spin.  Three ballots turn the decisions of a row into its bond masks, which the
            // thread that owns the row keeps.
            Bx = By = 0u;
            const uint32_t gxl = x0 + (uint32_t)lane;
            const uint32_t rowbase0 = g0 - L * (uint32_t)lane - (DIM == 2 ? 0u : 0u);   // row of lane 0 of this warp (same z)
            auto proj = [&](uint32_t gsite) -> float {           // XY: a = r . s;  clock: class word (u | sign << 16) as float bits
                if (MODEL == XY) {
                    float sn, cs;
                    SW_SINCOSF(((const float *)p.spins)[gsite], &sn, &cs);
                    return p.rx * cs + p.ry * sn;
                } else {
                    int k = 2 * (int)((const uint16_t *)p.spins)[gsite] - p.mirror;
                    if (k < 0) k += 2 * p.q;
                    const int u = k >= p.q ? k - p.q : k;
                    return __uint_as_float((uint32_t)u | (u == 0 ? 0u : (k >= p.q ? 2u : 1u) << 16));
                }
            };
            auto decide = [&](float a, float b, uint32_t word) -> bool {
                if (MODEL == XY) {
                    // (no short-circuit: for pr <= 0 the right-hand side is <= 0 and the comparison false anyway; a warp
                    // has a site with pr > 0 in practically every row, so the branch saved nothing)
                    const float pr = a * b;
                    const bool below = (float)(word >> 8) * 5.9604644775390625e-8f < SW_NEG_EXPM1F(p.m2beta * pr);
                    return (pr > 0.f) & below;
                } else {
                    const uint32_t ca = __float_as_uint(a), cb = __float_as_uint(b);
                    if (((ca & cb) >> 16) == 0u) return false;        // different sign, or one component is zero
                    return word < __ldg(p.clock_T + (ca & 0xffffu) * (uint32_t)p.q + (cb & 0xffffu));
                }
            };
            // the row above the warp's last row (periodic; 2D: the next rows of the tile or its +y halo)
            uint32_t gup = rowbase0 + 32u * L;
            {
                const uint32_t gy = y0 + (uint32_t)(ly - lane) + 32u;      // y of that row
                if (gy >= L) gup -= L * L;                                  // wrapped: back by L rows
            }
            float aprev = proj(gxl + gup);
            // the +z neighbour of a site of this plane is a fixed distance away (periodic wrap: back by L - 1 planes)
            uint32_t dzoff = (z0 + (uint32_t)lz + 1u == L) ? 0u - LL * (L - 1u) : LL;
            asm volatile("" : "+r"(dzoff));   // (kept in a register: otherwise it is recomputed from blockIdx in every iteration)
#pragma unroll 1
            for (int yy = 31; yy >= 0; --yy) {
                const uint32_t grow_ = rowbase0 + L * (uint32_t)yy;
                const uint32_t site = gxl + grow_;
                const float a = proj(site);
                float ax = __shfl_down_sync(FULL, a, 1);
                if (lane == 31) ax = proj(xh + grow_);
                const uint4 w = philox4x32_10_rk(site, t_lo, t_hi, DOM_SITE, p);
                const uint32_t mx = __ballot_sync(FULL, decide(a, ax, w.x));
                const uint32_t my = __ballot_sync(FULL, decide(a, aprev, w.y));
                uint32_t mz = 0u;
                if (DIM == 3) {
                    mz = __ballot_sync(FULL, decide(a, proj(site + dzoff), w.z));
                }
                const uint32_t md = __ballot_sync(FULL, (w.w >> 31) != 0u);
                if (lane == yy) { Bx = mx; By = my; Bz = mz; D = md; }
                aprev = a;
            }
        } else {
        uint32_t ex, ey, ez = 0u;
        if (MODEL == ISING) {
            const uint32_t nxb = sp[xh + g0] >> 7;             // sign of the +x neighbour of site 31
            const uint32_t S = sg_s[ly + G::SGY * lz];
            ex = ~(S ^ ((S >> 1) | (nxb << 31)));
            ey = ~(S ^ sg_s[ly + 1 + G::SGY * lz]);
            if (DIM == 3) ez = ~(S ^ sg_s[ly + G::SGY * (lz + 1)]);
        } else {
            // Potts: byte equality of the row with itself shifted by one site, with the +y and the +z row
            uint32_t own[8], oth[8];
            {
                const uint4 a = reinterpret_cast<const uint4 *>(sp + x0 + g0)[0], b = reinterpret_cast<const uint4 *>(sp + x0 + g0)[1];
                own[0] = a.x; own[1] = a.y; own[2] = a.z; own[3] = a.w; own[4] = b.x; own[5] = b.y; own[6] = b.z; own[7] = b.w;
            }
            const uint32_t nxb = sp[xh + g0];
#pragma unroll
            for (int j = 0; j < 8; ++j) oth[j] = __funnelshift_r(own[j], j < 7 ? own[j + 1] : nxb, 8);
            ex = eq32(own, oth);
            {
                const uint32_t gy = grow(ly + 1, lz);
                const uint4 a = reinterpret_cast<const uint4 *>(sp + x0 + gy)[0], b = reinterpret_cast<const uint4 *>(sp + x0 + gy)[1];
                oth[0] = a.x; oth[1] = a.y; oth[2] = a.z; oth[3] = a.w; oth[4] = b.x; oth[5] = b.y; oth[6] = b.z; oth[7] = b.w;
                ey = eq32(own, oth);
            }
            if (DIM == 3) {
                const uint32_t gz = grow(ly, lz + 1);
                const uint4 a = reinterpret_cast<const uint4 *>(sp + x0 + gz)[0], b = reinterpret_cast<const uint4 *>(sp + x0 + gz)[1];
                oth[0] = a.x; oth[1] = a.y; oth[2] = a.z; oth[3] = a.w; oth[4] = b.x; oth[5] = b.y; oth[6] = b.z; oth[7] = b.w;
                ez = eq32(own, oth);
            }
        }
        uint32_t X[3];
        if (EARLY_RANDOM) { X[0] = Xe[0]; X[1] = Xe[1]; X[2] = Xe[2]; D = De; }
        else group_decisions<DIM>(p, (x0 + g0) >> 5, t_lo, t_hi, X, D);
        Bx = ex & X[0]; By = ey & X[1]; Bz = (DIM == 3) ? (ez & X[2]) : 0u;
        }
        if (p.bonds) {   // canonical bond bytes on request (parity tests): bit k = bond in direction k
#pragma unroll
            for (int j = 0; j < 8; ++j)
                *reinterpret_cast<uint32_t *>(p.bonds + x0 + g0 + 4 * j) =
                    spread4((Bx >> (4 * j)) & 0xfu) | (spread4((By >> (4 * j)) & 0xfu) << 1) | (spread4((Bz >> (4 * j)) & 0xfu) << 2);
        }
        // bonds through the tile faces (incl. the periodic wrap) go to the global merge
        const uint32_t fx = __ballot_sync(FULL, Bx >> 31);
        Bx &= 0x7fffffffu;
        if (DIM == 3) {
            if (lane == 0) face_s[lz] = fx;                                // bit y of word z
            if (lane == 31) { face_s[G::FXW + lz] = By; By = 0u; }         // word z: row (TY-1, z), bit x
            if (lz == TZ - 1) { face_s[G::FXW + G::FYW + ly] = Bz; Bz = 0u; }  // word y: row (y, TZ-1), bit x
        } else {
            if (lane == 0) face_s[warp * R + r] = fx;                      // bit l of word (warp, r): row (32 warp + l) R + r
            if (ly == TY - 1) { face_s[G::FXW] = By; By = 0u; }
        }
        bx_s[row] = Bx;
        pm_s[row] = By;
        if (DIM == 3) pm_s[NROWS + row] = Bz;
        if (MODEL != POTTS) {
            dr_s[row] = D;
        } else {
            // Potts: the draw word of site b of the group is W_G[128 + b] (reading 6): call 32 + b / 4, word
            // b % 4; new state (w q) >> 32, one byte per site
            const unsigned qq = (unsigned)p.q;
            const uint32_t G0 = (x0 + g0) >> 5;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint4 dw = philox4x32_10(G0, t_lo, t_hi, DOM_GROUP + 256u * (GROUP_DRAW_BASE / 4u + (uint32_t)j), p.k0, p.k1);
                const uint32_t d = (uint32_t)(((unsigned long long)dw.x * qq) >> 32) | ((uint32_t)(((unsigned long long)dw.y * qq) >> 32) << 8) |
                                   ((uint32_t)(((unsigned long long)dw.z * qq) >> 32) << 16) | ((uint32_t)(((unsigned long long)dw.w * qq) >> 32) << 24);
                dr_s[row * 8 + j] = d;
            }
        }
        // every site starts as its own root: its 16-bit parent entry = own node = the address of that entry.  Lanes
        // take the 16-byte pieces of their rows (64 bytes apart) in rotated order so that they spread
        // over all banks
        const uint32_t o = lab_sa + (uint32_t)row * 64u;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t jj = (uint32_t)(j + (lane >> 1)) & 3u;
            const uint32_t v = o + 16u * jj;
            const uint32_t w0 = v | ((v + 2u) << 16);
            *reinterpret_cast<uint4 *>(lab_s + row * 16 + 4 * jj) = make_uint4(w0, w0 + 0x00040004u, w0 + 0x00080008u, w0 + 0x000c000cu);
        }
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

    // phase 2a: pull.  For the row B of this thread: sy / sz = bonds that reach it from the row below /
    // behind (inside the tile), T = its x-links.  A site with such a bond is the FIRST of its run iff no
    // lower site of the run has one: adding the bonds that sit on a link to T lets a carry run up every
    // run from its lowest such site (V marks what the carries touched).
    struct Back { uint32_t T, sz, bxY, bxZ, first, restY, restZ, rowB; };
    auto back_bonds = [&](int r) -> Back {
        const int ly = row_y(r), lz = row_z(r);
        const int row = ly + TY * lz;
        Back k;
        k.T = bx_s[row];
        const uint32_t sy = (ly > 0) ? pm_s[row - 1] : 0u;
        k.sz = (DIM == 3 && lz > 0) ? pm_s[NROWS + row - TY] : 0u;
        k.bxY = (ly > 0) ? bx_s[row - 1] : 0u;
        k.bxZ = (DIM == 3 && lz > 0) ? bx_s[row - TY] : 0u;
        const uint32_t sa = sy | k.sz;
        const uint32_t s1 = sa & k.T;
        const uint32_t V = (k.T + s1) ^ k.T;
        k.first = (s1 & V) | (sa & ~k.T & ~V);
        // a further bond joins the same two runs as the bond one site to the left (a twin) if both rows link
        // the two sites: nothing to do for it
        k.restY = sy & ~(k.first & ~k.sz) & ~((sy << 1) & (k.T << 1) & (k.bxY << 1));
        k.restZ = k.sz & ~k.first & ~((k.sz << 1) & (k.T << 1) & (k.bxZ << 1));
        k.rowB = lab_sa + (uint32_t)row * 64u;
        return k;
    };
    uint32_t unfit = 0u;   // rows of this thread whose further bonds did not fit into the list
#pragma unroll 1
    for (int r = 0; r < R; ++r) {
        const Back k = back_bonds(r);
        const uint32_t rowY = k.rowB - 64u, rowZ = k.rowB - 64u * TY;
        uint32_t f = k.first;
        while (f) {
            const uint32_t low = f & (0u - f), below = low - 1u;
            f ^= low;
            const bool isz = (DIM == 3) && (k.sz & low);   // a site reached from both rows takes the z bond
            const uint32_t b = k.rowB + 2u * run_start(k.T, below);
            const uint32_t a = (isz ? rowZ : rowY) + 2u * run_start(isz ? k.bxZ : k.bxY, below);
            sts_u16(b, a);
        }
        // the other bonds: (a, b) pairs for phase 2b, warp-aggregated reservation in the list
        const uint32_t cnt = __popc(k.restY) + __popc(k.restZ);
        uint32_t inc = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(FULL, inc, o);
            if (lane >= o) inc += u;
        }
        const uint32_t tot = __shfl_sync(FULL, inc, 31);
        if (tot) {
            uint32_t base = 0u;
            if (lane == 31) base = atomicAdd(&fpre_s[G::NFWP + 1], tot);
            base = __shfl_sync(FULL, base, 31);
            if (base + tot <= (uint32_t)G::LIST_CAP) {
                uint32_t pos = base + inc - cnt;
#pragma unroll
                for (int dir = 0; dir < G::NDIR; ++dir) {
                    uint32_t w = dir ? k.restZ : k.restY;
                    const uint32_t rowP = dir ? rowZ : rowY, bxP = dir ? k.bxZ : k.bxY;
                    while (w) {
                        const uint32_t low = w & (0u - w), below = low - 1u;
                        w ^= low;
                        const uint32_t b = k.rowB + 2u * run_start(k.T, below);
                        const uint32_t a = rowP + 2u * run_start(bxP, below);
                        // b has just been given a parent by this thread (a run with a further bond has a first
                        // one): the union starts from that parent, one level up
                        list_s[pos++] = (a << 16) | lds_u16(b);
                    }
                }
            } else {
                // list full (ordered phase with many domain walls): these bonds are done after phase 2b, and
                // the list is valid only below the first reservation that did not fit
                unfit |= 1u << r;
                if (lane == 31) atomicMin(&fpre_s[G::NFWP + 2], base);
            }
        }
    }
    __syncthreads();

    // phase 2b: union-find over the listed bonds.  Every warp takes a contiguous share of the list; a lane
    // holds the two nodes (a, b) of the union it is working on (a == b: none) and, per round, either
    // fetches the next bond of the warp's share, or climbs one level, or hooks -- lanes whose union needs
    // several rounds do not hold up lanes that are ready for their next bond.
    {
        const uint32_t n = min(fpre_s[G::NFWP + 1], fpre_s[G::NFWP + 2]);
        uint32_t nxt = (n * (uint32_t)warp) / NW;
        const uint32_t end = (n * (uint32_t)(warp + 1)) / NW;
        const uint32_t lt = (1u << lane) - 1u;
        uint32_t a = 0u, b = 0u;
        for (;;) {
            const uint32_t need = __ballot_sync(FULL, a == b);
            if (need && nxt < end) {
                const uint32_t idx = nxt + __popc(need & lt);
                if (a == b && idx < end) {
                    const uint32_t ent = list_s[idx];
                    a = ent >> 16;
                    b = ent & 0xffffu;
                }
                nxt += __popc(need);
            }
            if (!__any_sync(FULL, a != b)) {
                if (nxt >= end) break;
                continue;   // every bond just fetched joins a run with its own parent: fetch again
            }
            if (a != b) {
#if SW_ROW_UF_MERGED
                // climb (two levels, path halving: a non-root is never the target of a hook, and any ancestor is
                // a valid parent); if the parents turn out to be roots the hook follows in the same round
                const uint32_t pa = lds_u16(a), pb = lds_u16(b);
                bool roots = pa == a && pb == b;
                if (!roots) {
                    const uint32_t ga = lds_u16(pa), gb = lds_u16(pb);
                    if (ga != pa) sts_u16(a, ga);
                    if (gb != pb) sts_u16(b, gb);
                    roots = ga == pa && gb == pb;
                    a = roots ? pa : ga;
                    b = roots ? pb : gb;                  // (a == b afterwards: same tree already)
                }
                if (roots && a != b) {
                    const uint32_t hi = max(a, b), lo = min(a, b);
                    const uint32_t old = cas_u16(hi, hi, lo);
                    if (old == hi) a = b;                 // done
                    else { a = old; b = lo; }             // hi was hooked meanwhile: go on from its new parent
                }
#else
                const uint32_t pa = lds_u16(a), pb = lds_u16(b);
                if (pa == a && pb == b) {
                    const uint32_t hi = max(a, b), lo = min(a, b);
                    const uint32_t old = cas_u16(hi, hi, lo);
                    if (old == hi) a = b;                 // done
                    else { a = old; b = lo; }             // hi was hooked meanwhile: go on from its new parent
                } else {
                    // climb two levels and make both nodes skip their parents (path halving: a non-root is
                    // never the target of a hook, and any ancestor is a valid parent)
                    const uint32_t ga = lds_u16(pa), gb = lds_u16(pb);
                    if (ga != pa) sts_u16(a, ga);
                    if (gb != pb) sts_u16(b, gb);
                    a = ga; b = gb;                       // (a == b afterwards: same tree already)
                }
#endif
            }
        }
    
    }
    if (fpre_s[G::NFWP + 1] > (uint32_t)G::LIST_CAP) {   // block-uniform; rare
#pragma unroll 1
        for (int r = 0; r < R; ++r) {
            if (!((unfit >> r) & 1u)) continue;
            const Back k = back_bonds(r);
            const uint32_t rowY = k.rowB - 64u, rowZ = k.rowB - 64u * TY;
#pragma unroll
            for (int dir = 0; dir < G::NDIR; ++dir) {
                uint32_t w = dir ? k.restZ : k.restY;
                const uint32_t rowP = dir ? rowZ : rowY, bxP = dir ? k.bxZ : k.bxY;
                while (w) {
                    const uint32_t low = w & (0u - w), below = low - 1u;
                    w ^= low;
                    union_nodes_halving(rowP + 2u * run_start(bxP, below), k.rowB + 2u * run_start(k.T, below));
                }
            }
        }
    }
    __syncthreads();

    // active face bonds -> (address of i, address of j) in the global pair list (k_merge's work): a warp
    // takes one face word at a time, lane = bit
    {
        const uint32_t ntx = p.ntx, nty = p.nty;
        const uint32_t tjx = (bx + 1 == ntx) ? tile - (ntx - 1) : tile + 1;
        const uint32_t tjy = (by + 1 == nty) ? tile - ntx * (nty - 1) : tile + ntx;
        const uint32_t tjz = (DIM == 3) ? ((bz + 1 == p.ntz) ? tile - ntx * nty * (p.ntz - 1) : tile + ntx * nty) : 0u;
        const uint32_t fbase = fpre_s[G::NFWP];
        for (int wd = warp; wd < G::NFW; wd += NW) {
            const uint32_t fw = face_s[wd];
            if ((fw >> lane) & 1u) {
                const uint32_t pos = fbase + fpre_s[wd] + __popc(fw & ((1u << lane) - 1u));
                uint32_t li_i, li_j, tj;
                if (wd < G::FXW) {
                    const int row = (DIM == 3) ? lane + TY * wd : (32 * (wd / R) + lane) * R + (wd % R);
                    li_j = 32u * (uint32_t)row; li_i = li_j + 31u; tj = tjx;
                } else if (wd < G::FXW + G::FYW) {
                    const int lz = wd - G::FXW;
                    li_j = (uint32_t)lane + 32u * (uint32_t)(TY * lz); li_i = li_j + 32u * (TY - 1); tj = tjy;
                } else {
                    const int ly = wd - G::FXW - G::FYW;
                    li_j = (uint32_t)lane + 32u * (uint32_t)ly; li_i = li_j + 32u * TY * (TZ - 1); tj = tjz;
                }
                // this tile's end of the bond is handed over as the ancestor the tile-local forest gives for
                // it (k_merge then starts its find there instead of walking the chain through L2)
                const uint32_t ri = li_i >> 5;
                uint32_t v = lds_u16(lab_sa + ri * 64u + 2u * run_start(bx_s[ri], (1u << (li_i & 31u)) - 1u));
#pragma unroll
                for (int k = 0; k < SW_ROW_JUMPS; ++k) v = lds_u16(v);
                p.pairs[pos] = make_uint2(tile_base + ((v - lab_sa) >> 1), (tj << G::LOG2NS) + li_j);
            }
        }
    }

    // phase 3: the forest is static now.  A warp takes one row at a time, lane = x: the site's run start,
    // its parent and SW_ROW_JUMPS further ancestors (a root points to itself); label word =
    // (address of the ancestor reached << DB) | own draw.
    {
        const int db = (MODEL == POTTS) ? p.db : 1;
        const uint32_t below = (1u << lane) - 1u;
#if SW_ROW_P3_UNROLL == 4
#pragma unroll 4
#elif SW_ROW_P3_UNROLL == 1
#pragma unroll 1
#else
#pragma unroll 2
#endif
        for (int row = warp; row < NROWS; row += NW) {
            const uint32_t st = run_start(bx_s[row], below);
            uint32_t v = lds_u16(lab_sa + (uint32_t)row * 64u + 2u * st);
            if (SW_ROW_JUMPS > 0) {
                // first ancestor; if it is the run start itself the run start is a root and the site is done
                // (no further loads: fewer shared-memory wavefronts; 45 % of the run starts are roots)
                const uint32_t v0 = v;
                v = lds_u16(v);
                const uint32_t more = (v != v0) ? 1u : 0u;
#pragma unroll
                for (int k = 1; k < SW_ROW_JUMPS; ++k) lds_u16_if(v, more, v);
            }
            uint32_t word;
            if (MODEL != POTTS) word = ((tile_base << 1) - lab_sa) + v + ((dr_s[row] >> lane) & 1u);   // v - lab_sa = 2 x local index
            else word = ((tile_base + ((v - lab_sa) >> 1)) << db) | reinterpret_cast<const uint8_t *>(dr_s)[row * 32 + lane];
            p.labels[tile_base + (uint32_t)row * 32u + (uint32_t)lane] = word;
        }
    }
}

}  // namespace swk
