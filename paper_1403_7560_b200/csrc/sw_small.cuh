// sw_small.cuh -- k_sw_small: the whole Swendsen-Wang step (bonds, clusters, new values,
// observables) for lattices that fit one CTA, n steps per launch.  PAPER.md:174: "for smaller lattices the
// parallelization is not so effective" -- with one tile per lattice the three-kernel path is bound by
// launch and dependency latency (config C1, 2D L = 64: 4096 sites), so here spins, bond masks and the
// union-find stay in shared memory from step to step and nothing but the barrier separates the phases.
// Ising and Potts, N <= 32768 sites (2D L <= 160, 3D L = 32); 1024 threads, of which the first N / 32 own one row of 32 consecutive sites each
// (rows are 32 consecutive LINEAR indices, so a node = 2 x linear index and no merge across tiles exists;
// periodic-wrap bonds are ordinary entries of the union list).  Independent of oracle/.
#pragma once
#include "sw_rows.cuh"

#ifndef SW_SMALL_PREJUMPS
#define SW_SMALL_PREJUMPS 0   // pointer-jumping passes between the pull and the union-find (measured: no gain)
#endif
#ifndef SW_SMALL_JUMPS
#define SW_SMALL_JUMPS 3      // pointer-jumping passes before the root chase
#endif

#ifdef SW_SMALL_PROFILE   // developer build: cycles per phase, summed over the steps, in acc->stats[0..5]
#define SW_SMALL_MARK(k) do { if (tid == 0) { const long long now_ = clock64(); p.acc->stats[k] += (unsigned long long)(now_ - mark_); mark_ = now_; } } while (0)
#else
#define SW_SMALL_MARK(k) do { } while (0)
#endif

namespace swk {

struct SmallArgs {
    int nsteps;
    int write_labels;               // label words (root << DB | draw, address = linear index) of the LAST step
    unsigned long long *series;     // per step: E_int, (E_xy), M_int, (mx), (my), n_k[q]  (the head of Acc) or NULL
    int series_words;
};

template <int DIM, int MODEL>
struct SmallGeom {
    // shared memory, 32-bit words, for N sites (NR = N / 32 rows)
    static __host__ __device__ constexpr size_t off_bx(size_t N) { return N / 2; }              // after the 16-bit parent entries
    static __host__ __device__ constexpr size_t off_by(size_t N) { return off_bx(N) + N / 32; }
    static __host__ __device__ constexpr size_t off_bz(size_t N) { return off_by(N) + N / 32; }
    static __host__ __device__ constexpr size_t off_dr(size_t N) { return off_bz(N) + N / 32; }   // Ising: draw masks; Potts: draw bytes
    static __host__ __device__ constexpr size_t off_st(size_t N) { return off_dr(N) + (MODEL == ISING ? N / 32 : N / 4); }  // state: sign masks / spin bytes
    static __host__ __device__ constexpr size_t off_lk(size_t N) { return off_st(N) + (MODEL == ISING ? N / 32 : N / 4); }   // x-link of a row into the next row of its line
    static __host__ __device__ constexpr size_t off_misc(size_t N) { return off_lk(N) + N / 32; } // counters, histogram
    static __host__ __device__ constexpr size_t off_list(size_t N) { return off_misc(N) + 8 + 256; }
    static __host__ __device__ constexpr size_t list_cap(size_t N) { return N / 4; }
    static __host__ __device__ constexpr size_t words(size_t N) { return off_list(N) + list_cap(N); }
};

template <int DIM, int MODEL>
__global__ void __launch_bounds__(1024, 1) k_sw_small(const Params p, const SmallArgs args)
{
    static_assert(MODEL == ISING || MODEL == POTTS, "constant bond probability");
    using G = SmallGeom<DIM, MODEL>;
    extern __shared__ __align__(16) uint32_t smem_u32[];
    const uint32_t N = p.N, L = p.L, NR = N >> 5, BX = L >> 5;       // rows, rows per lattice line
    uint32_t *lab_s = smem_u32;
    uint32_t *bx_s = smem_u32 + G::off_bx(N);    // x-links inside the row (bit 31 cleared)
    uint32_t *by_s = smem_u32 + G::off_by(N);
    uint32_t *bz_s = smem_u32 + G::off_bz(N);
    uint32_t *dr_s = smem_u32 + G::off_dr(N);
    uint32_t *st_s = smem_u32 + G::off_st(N);
    uint32_t *lk_s = smem_u32 + G::off_lk(N);     // 1: site 31 of the row is bonded to site 0 of row rxp
    uint32_t *misc_s = smem_u32 + G::off_misc(N);   // [0] list length, [1] valid part, [2..3] E, [4..5] M (64-bit), [8..] Potts histogram
    uint32_t *list_s = smem_u32 + G::off_list(N);
    const uint32_t LIST_CAP = (uint32_t)G::list_cap(N);
    const uint32_t lab_sa = (uint32_t)__cvta_generic_to_shared(lab_s);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, NW = blockDim.x >> 5;
    const uint32_t r = (uint32_t)tid;                                 // my row: sites 32 r .. 32 r + 31 ...
    const bool rowthread = r < NR;                                    // ... if there is one: the other warps only help in the dense phases
    const int db = (MODEL == POTTS) ? p.db : 1;
    const unsigned qq = (unsigned)p.q;

    // neighbour rows (periodic)
    const uint32_t line = r / BX, yy = line % L, zz = (DIM == 3) ? line / L : 0u;
    const uint32_t rxp = ((r % BX) == BX - 1u) ? r - (BX - 1u) : r + 1u;
    const uint32_t ryp = (yy == L - 1u) ? r - (L - 1u) * BX : r + BX;
    const uint32_t rzp = (DIM == 3) ? ((zz == L - 1u) ? r - (L - 1u) * L * BX : r + L * BX) : r;
    const bool has_xm = (r % BX) != 0u, has_ym = yy > 0u, has_zm = (DIM == 3) && zz > 0u;   // back neighbours with smaller index
    const uint32_t rxm = r - 1u, rym = r - BX, rzm = r - L * BX;

    // state: global spins -> shared (Ising: sign masks; Potts: the spin bytes)
    const uint8_t *sp = (const uint8_t *)p.spins;
    if (rowthread) {
        if (MODEL == ISING) st_s[r] = sign32(reinterpret_cast<const uint4 *>(sp + 32u * r));
        else {
            const uint4 a = reinterpret_cast<const uint4 *>(sp + 32u * r)[0], b = reinterpret_cast<const uint4 *>(sp + 32u * r)[1];
            *reinterpret_cast<uint4 *>(st_s + 8u * r) = a;
            *reinterpret_cast<uint4 *>(st_s + 8u * r + 4u) = b;
        }
    }
    unsigned long long t_step = p.acc->t;
    __syncthreads();

    // equality masks of my row with its +x / +y / +z neighbours (bit 31 of ex: site 31 against site 0 of row rxp)
    auto equal_masks = [&](uint32_t &ex, uint32_t &ey, uint32_t &ez) {
        ez = 0u;
        if (MODEL == ISING) {
            const uint32_t S = st_s[r];
            ex = ~(S ^ ((S >> 1) | (st_s[rxp] << 31)));
            ey = ~(S ^ st_s[ryp]);
            if (DIM == 3) ez = ~(S ^ st_s[rzp]);
        } else {
            uint32_t own[8], oth[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) own[j] = st_s[8u * r + j];
            const uint32_t nxb = st_s[8u * rxp];
#pragma unroll
            for (int j = 0; j < 8; ++j) oth[j] = __funnelshift_r(own[j], j < 7 ? own[j + 1] : nxb, 8);
            ex = eq32(own, oth);
#pragma unroll
            for (int j = 0; j < 8; ++j) oth[j] = st_s[8u * ryp + j];
            ey = eq32(own, oth);
            if (DIM == 3) {
#pragma unroll
                for (int j = 0; j < 8; ++j) oth[j] = st_s[8u * rzp + j];
                ez = eq32(own, oth);
            }
        }
    };
    // energy of the configuration in shared memory from the equality masks: Ising E = -(2 #equal - #pairs)
    // (Eq. 1), Potts E = #unequal pairs (Eq. 2); block sum into misc_s[2..3]
    auto add_energy = [&](uint32_t ex, uint32_t ey, uint32_t ez) {
        const int eq = __popc(ex) + __popc(ey) + (DIM == 3 ? __popc(ez) : 0);
        int e = (MODEL == ISING) ? 32 * DIM - 2 * eq : 32 * DIM - eq;
        e = __reduce_add_sync(FULL, e);
        if (lane == 0) atomicAdd(reinterpret_cast<unsigned long long *>(misc_s + 2), (unsigned long long)(long long)e);
    };

    // pointer jumping: every parent entry is replaced by the entry of the parent (8 entries = 16 bytes per
    // thread and step).  The pull leaves chains as long as a cluster is wide in y + z (at T_c: the lattice
    // size); each pass halves them before the root chase of the flip phase.
    auto jump_pass = [&]() {
        // (four entries per thread: all 1024 threads work on a 4096-site lattice)
        for (uint32_t v = (uint32_t)tid; v < N / 4u; v += blockDim.x) {
            const uint2 w = *reinterpret_cast<const uint2 *>(lab_s + 2u * v);
            uint2 o;
            o.x = lds_u16(lab_sa + (w.x & 0xffffu)) | (lds_u16(lab_sa + (w.x >> 16)) << 16);
            o.y = lds_u16(lab_sa + (w.y & 0xffffu)) | (lds_u16(lab_sa + (w.y >> 16)) << 16);
            *reinterpret_cast<uint2 *>(lab_s + 2u * v) = o;
        }
        __syncthreads();
    };
#ifdef SW_SMALL_PROFILE
    long long mark_ = clock64();
#endif
#pragma unroll 1
    for (int step = 0; step < args.nsteps; ++step, ++t_step) {
        const uint32_t t_lo = (uint32_t)t_step, t_hi = (uint32_t)(t_step >> 32);
        const bool last = step + 1 == args.nsteps;
        // ---- bonds: equality AND the random decision u < P32 (reading 6: group = row) ----
        uint32_t BxF = 0u, By = 0u, Bz = 0u, Bx = 0u;
        if (rowthread) {
        uint32_t ex, ey, ez;
        equal_masks(ex, ey, ez);
        uint32_t X[3], D;
        group_decisions<DIM>(p, r, t_lo, t_hi, X, D);
        BxF = ex & X[0]; By = ey & X[1]; Bz = (DIM == 3) ? (ez & X[2]) : 0u;
        if (p.bonds && last) {
#pragma unroll
            for (int j = 0; j < 8; ++j)
                *reinterpret_cast<uint32_t *>(p.bonds + 32u * r + 4 * j) =
                    spread4((BxF >> (4 * j)) & 0xfu) | (spread4((By >> (4 * j)) & 0xfu) << 1) | (spread4((Bz >> (4 * j)) & 0xfu) << 2);
        }
        Bx = BxF & 0x7fffffffu;
        bx_s[r] = Bx;
        by_s[r] = By;
        if (DIM == 3) bz_s[r] = Bz;
        lk_s[r] = BxF >> 31;
        if (MODEL == ISING) dr_s[r] = D;
        else {
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint4 dw = philox4x32_10(r, t_lo, t_hi, DOM_GROUP + 256u * (GROUP_DRAW_BASE / 4u + (uint32_t)j), p.k0, p.k1);
                dr_s[8u * r + j] = (uint32_t)(((unsigned long long)dw.x * qq) >> 32) | ((uint32_t)(((unsigned long long)dw.y * qq) >> 32) << 8) |
                                   ((uint32_t)(((unsigned long long)dw.z * qq) >> 32) << 16) | ((uint32_t)(((unsigned long long)dw.w * qq) >> 32) << 24);
            }
        }
        {   // every site starts as its own root: 16-bit parent entry = own node = 2 x linear index
            const uint32_t o = r * 64u;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t jj = (uint32_t)(j + (lane >> 1)) & 3u;
                const uint32_t v = o + 16u * jj;
                const uint32_t w0 = v | ((v + 2u) << 16);
                *reinterpret_cast<uint4 *>(lab_s + r * 16u + 4u * jj) = make_uint4(w0, w0 + 0x00040004u, w0 + 0x00080008u, w0 + 0x000c000cu);
            }
        }
        }
        if (tid == 0) { misc_s[0] = 0u; misc_s[1] = LIST_CAP; misc_s[4] = 0u; misc_s[5] = 0u; }
        if (MODEL == POTTS) for (int k = tid; k < 256; k += blockDim.x) misc_s[8 + k] = 0u;
        __syncthreads();
        SW_SMALL_MARK(0);

        // ---- pull (see sw_rows.cuh phase 2a): back bonds from the rows with smaller index ----
        {
            const uint32_t T = Bx;
            bool fits = true;
            uint32_t tot = 0u, restY = 0u, restZ = 0u, restX = 0u, wyr = 0u, wzr = 0u, wx = 0u, bxY = 0u, bxZ = 0u, bxWY = 0u, bxWZ = 0u;
            const uint32_t rowB = r * 64u, rowY = rym * 64u, rowZ = rzm * 64u;
            if (rowthread) {
            const uint32_t sy = has_ym ? by_s[rym] : 0u;
            const uint32_t sz = has_zm ? bz_s[rzm] : 0u;
            const uint32_t sx = has_xm ? lk_s[rxm] : 0u;     // bit 0: link into my site 0
            bxY = has_ym ? bx_s[rym] : 0u; bxZ = has_zm ? bx_s[rzm] : 0u;
            const uint32_t sa = sy | sz | sx;
            const uint32_t s1 = sa & T;
            const uint32_t V = (T + s1) ^ T;
            const uint32_t first = (s1 & V) | (sa & ~T & ~V);
            restY = sy & ~(first & ~sz) & ~((sy << 1) & (T << 1) & (bxY << 1));
            restZ = sz & ~first & ~((sz << 1) & (T << 1) & (bxZ << 1));
            restX = sx & ~(first & ~sz & ~sy);
            uint32_t f = first;
            while (f) {
                const uint32_t low = f & (0u - f), below = low - 1u;
                f ^= low;
                const uint32_t b = rowB + 2u * run_start(T, below);
                uint32_t a;
                if (sz & low) a = rowZ + 2u * run_start(bxZ, below);
                else if (sy & low) a = rowY + 2u * run_start(bxY, below);
                else a = rxm * 64u + 2u * run_start(bx_s[rxm], 0x7fffffffu);   // the run of site 31 of the row before
                sts_u16(lab_sa + b, a);
            }
            // everything else goes through the union-find: further back bonds, and the periodic-wrap bonds
            // (owned by the row with the LARGER index: y = L-1, z = L-1, last row of a line)
            const uint32_t wy = (yy == L - 1u) ? By : 0u, wz = (DIM == 3 && zz == L - 1u) ? Bz : 0u;
            wx = ((r % BX) == BX - 1u) ? (BxF >> 31) : 0u;
            bxWY = bx_s[ryp]; bxWZ = bx_s[rzp];
            wyr = wy & ~((wy << 1) & (T << 1) & (bxWY << 1)); wzr = wz & ~((wz << 1) & (T << 1) & (bxWZ << 1));
            const uint32_t cnt = __popc(restY) + __popc(restZ) + restX + __popc(wyr) + __popc(wzr) + wx;
            uint32_t inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(FULL, inc, o);
                if (lane >= o) inc += u;
            }
            tot = __shfl_sync(FULL, inc, 31);
            uint32_t base = 0u;
            if (lane == 31 && tot) base = atomicAdd(&misc_s[0], tot);
            base = __shfl_sync(FULL, base, 31);
            fits = base + tot <= LIST_CAP;
            if (tot && !fits && lane == 31) atomicMin(&misc_s[1], base);
            uint32_t pos = base + inc - cnt;
            auto emit = [&](uint32_t a, uint32_t b) { list_s[pos++] = (a << 16) | b; };
            // (a warp whose bonds find no room in the list keeps them until the pulls of all rows are done)
            if (fits) {
                uint32_t w = restY;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; emit(rowY + 2u * run_start(bxY, below), rowB + 2u * run_start(T, below)); }
                w = restZ;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; emit(rowZ + 2u * run_start(bxZ, below), rowB + 2u * run_start(T, below)); }
                if (restX) emit(rxm * 64u + 2u * run_start(bx_s[rxm], 0x7fffffffu), rowB);
                w = wyr;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; emit(ryp * 64u + 2u * run_start(bxWY, below), rowB + 2u * run_start(T, below)); }
                w = wzr;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; emit(rzp * 64u + 2u * run_start(bxWZ, below), rowB + 2u * run_start(T, below)); }
                if (wx) emit(rxp * 64u, rowB + 2u * run_start(T, 0x7fffffffu));
            }
            }
            __syncthreads();
        SW_SMALL_MARK(1);
#pragma unroll 1
            for (int pass = 0; pass < SW_SMALL_PREJUMPS; ++pass) jump_pass();
            // ---- union-find over the list (sw_rows.cuh phase 2b) ----
            {
                const uint32_t n = min(misc_s[0], misc_s[1]);
                uint32_t nxt = (n * (uint32_t)warp) / (uint32_t)NW;
                const uint32_t end = (n * (uint32_t)(warp + 1)) / (uint32_t)NW;
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
                        continue;
                    }
                    if (a != b) {
                        // climb two levels (path halving); if the parents turn out to be roots, hook in the same round
                        const uint32_t pa = lds_u16(lab_sa + a), pb = lds_u16(lab_sa + b);
                        bool roots = pa == a && pb == b;
                        if (!roots) {
                            const uint32_t ga = lds_u16(lab_sa + pa), gb = lds_u16(lab_sa + pb);
                            if (ga != pa) sts_u16(lab_sa + a, ga);
                            if (gb != pb) sts_u16(lab_sa + b, gb);
                            roots = ga == pa && gb == pb;
                            a = roots ? pa : ga;
                            b = roots ? pb : gb;
                        }
                        if (roots && a != b) {
                            const uint32_t hi = max(a, b), lo = min(a, b);
                            const uint32_t old = cas_u16(lab_sa + hi, hi, lo);
                            if (old == hi) a = b;
                            else { a = old; b = lo; }
                        }
                    }
                }
            }
            if (rowthread && !fits && tot) {   // bonds that found no room in the list: now that all pulls are done
                uint32_t w = restY;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; union_nodes(lab_sa, rowY + 2u * run_start(bxY, below), rowB + 2u * run_start(T, below)); }
                w = restZ;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; union_nodes(lab_sa, rowZ + 2u * run_start(bxZ, below), rowB + 2u * run_start(T, below)); }
                if (restX) union_nodes(lab_sa, rxm * 64u + 2u * run_start(bx_s[rxm], 0x7fffffffu), rowB);
                w = wyr;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; union_nodes(lab_sa, ryp * 64u + 2u * run_start(bxWY, below), rowB + 2u * run_start(T, below)); }
                w = wzr;
                while (w) { const uint32_t low = w & (0u - w), below = low - 1u; w ^= low; union_nodes(lab_sa, rzp * 64u + 2u * run_start(bxWZ, below), rowB + 2u * run_start(T, below)); }
                if (wx) union_nodes(lab_sa, rxp * 64u, rowB + 2u * run_start(T, 0x7fffffffu));
            }
        }
        __syncthreads();
        SW_SMALL_MARK(2);

#pragma unroll 1
        for (int pass = 0; pass < SW_SMALL_JUMPS; ++pass) jump_pass();
        SW_SMALL_MARK(3);

        // ---- new value per cluster and magnetisation: a warp takes one row at a time, lane = x;
        //      the root (minimum linear index) is followed to the end: no later kernel does it ----
        {
            const uint32_t below = (1u << lane) - 1u;
            int m_loc = 0;
            // four rows of a warp in flight: the chases are chains of dependent shared-memory loads
#pragma unroll 1
            for (uint32_t row0 = (uint32_t)warp; row0 < NR; row0 += 4u * (uint32_t)NW) {
                uint32_t v[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t row = row0 + (uint32_t)j * (uint32_t)NW;
                    v[j] = row < NR ? lds_u16(lab_sa + row * 64u + 2u * run_start(bx_s[row], below)) : 0u;   // (node 0 is a root)
                }
                for (;;) {
                    uint32_t nn[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) nn[j] = lds_u16(lab_sa + v[j]);
                    const bool done = nn[0] == v[0] && nn[1] == v[1] && nn[2] == v[2] && nn[3] == v[3];
#pragma unroll
                    for (int j = 0; j < 4; ++j) v[j] = nn[j];
                    if (done) break;
                }
                __syncwarp();
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t row = row0 + (uint32_t)j * (uint32_t)NW;
                    if (row >= NR) break;                            // (uniform in the warp)
                    const uint32_t root = v[j] >> 1;                 // linear index of the root
                    if (MODEL == ISING) {
                        const uint32_t d = (dr_s[root >> 5] >> (root & 31u)) & 1u;   // 1: the cluster becomes +1
                        const uint32_t plus = __ballot_sync(FULL, d);
                        if (lane == 0) st_s[row] = ~plus;                // sign masks: bit set = spin -1
                        m_loc += 2 * __popc(plus) - 32;
                        if (last && args.write_labels) {
                            const uint32_t own = (dr_s[row] >> lane) & 1u;
                            p.labels[row * 32u + (uint32_t)lane] = (root << 1) | own;
                        }
                    } else {
                        const uint32_t d = reinterpret_cast<const uint8_t *>(dr_s)[root];
                        reinterpret_cast<uint8_t *>(st_s)[row * 32u + (uint32_t)lane] = (uint8_t)d;
                        atomicAdd(&misc_s[8 + d], 1u);
                        if (last && args.write_labels)
                            p.labels[row * 32u + (uint32_t)lane] = (root << db) | reinterpret_cast<const uint8_t *>(dr_s)[row * 32u + (uint32_t)lane];
                    }
                }
            }
            if (MODEL == ISING && lane == 0) atomicAdd(reinterpret_cast<unsigned long long *>(misc_s + 4), (unsigned long long)(long long)m_loc);
        }
        if (tid == 0) { misc_s[2] = 0u; misc_s[3] = 0u; }
        __syncthreads();
        SW_SMALL_MARK(4);

        if (args.series || last) {
            // observables of the new configuration
            if (rowthread) {
                uint32_t fx, fy, fz;
                equal_masks(fx, fy, fz);
                add_energy(fx, fy, fz);
            }
            __syncthreads();
            unsigned long long *dst = last ? reinterpret_cast<unsigned long long *>(p.acc) : nullptr;
            if (tid == 0) {
                const unsigned long long e = *reinterpret_cast<unsigned long long *>(misc_s + 2);
                const unsigned long long m = *reinterpret_cast<unsigned long long *>(misc_s + 4);
                if (dst) { dst[0] = e; dst[2] = m; }
                if (args.series) { unsigned long long *rec = args.series + (size_t)step * args.series_words; rec[0] = e; rec[1] = 0ull; rec[2] = m; rec[3] = 0ull; rec[4] = 0ull; }
            }
            if (MODEL == POTTS) {
                for (int k = tid; k < p.q; k += blockDim.x) {
                    if (dst) dst[5 + k] = (unsigned long long)misc_s[8 + k];
                    if (args.series) args.series[(size_t)step * args.series_words + 5 + k] = (unsigned long long)misc_s[8 + k];
                }
            }
            __syncthreads();
        SW_SMALL_MARK(5);
        }
    }

    // state back to global memory
    if (!rowthread) return;
    if (MODEL == ISING) {
        const uint32_t S = st_s[r];
#pragma unroll
        for (int j = 0; j < 8; ++j)
            *reinterpret_cast<uint32_t *>((uint8_t *)p.spins + 32u * r + 4 * j) = 0x01010101u + spread4((S >> (4 * j)) & 0xfu) * 0xfeu;
    } else {
        reinterpret_cast<uint4 *>((uint8_t *)p.spins + 32u * r)[0] = *reinterpret_cast<const uint4 *>(st_s + 8u * r);
        reinterpret_cast<uint4 *>((uint8_t *)p.spins + 32u * r)[1] = *reinterpret_cast<const uint4 *>(st_s + 8u * r + 4u);
    }
    if (tid == 0) p.acc->t = t_step;
}

// canonical labels for the one-CTA path: label words are addressed by the linear site index
__global__ void __launch_bounds__(256) k_export_labels_linear(const Params p)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= p.N) return;
    uint32_t a = i;
    const int db = p.db;
    for (;;) {
        const uint32_t n = p.labels[a] >> db;
        if (n == a) break;
        a = n;
    }
    p.labels_out[i] = a;
}

}  // namespace swk
