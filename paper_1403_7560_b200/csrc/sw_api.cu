// sw_api.cu -- host driver and C ABI (include/sw.h) of libsw_b200.
// Launch sequencing of one Swendsen-Wang step: k_bond_label -> k_merge -> k_flip,
// all asynchronous on the context's stream (plain launches, or CUDA-graph replay for Ising / Potts on
// any lattice size); no host synchronisation inside sw_step.
#include "../../include/sw.h"
#include "sw_kernels.cuh"
#include "sw_rows.cuh"
#include "sw_small.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace swk;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}

// One tile configuration = the tiled kernels instantiated for it.
struct TileOps {
    int tx, ty, tz, nt, nt_bl, rows;   // nt: threads of k_flip, nt_bl: threads of the bond / label kernel
    size_t smem_bond_label;
    void (*bond_label)(const Params);
    void (*merge)(const Params);
    void (*flip)(const Params);
    void (*export_labels)(const Params);
    void (*tile_origin)(const Params);
};

// XY, clock: k_bond_label (a thread owns QPT quads of 4 sites).
template <int DIM, int MODEL, int TX, int TY, int TZ, int QPT = 4>
TileOps make_ops()
{
    using G = TileGeom<DIM, TX, TY, TZ>;
    constexpr int NS = G::NS;
    constexpr int NT = NS / (4 * QPT);  // QPT quads = 4 QPT sites per thread
    TileOps o;
    o.tx = TX; o.ty = TY; o.tz = TZ; o.nt = NT; o.nt_bl = NT; o.rows = 0;
    o.smem_bond_label = G::template smem_bond_label<MODEL>();
    o.bond_label = k_bond_label<DIM, MODEL, TX, TY, TZ, NT>;
    o.merge = k_merge<DIM, TX, TY, TZ>;
    o.flip = k_flip<DIM, MODEL, TX, TY, TZ, NT>;
    o.export_labels = k_export_labels<DIM, TX, TY, TZ>;
    o.tile_origin = k_tile_origin<TX, TY, TZ>;
    return o;
}

// Ising, Potts: k_bond_label_rows (a thread owns R rows of 32 sites); k_flip with QPT quads per thread.
template <int DIM, int MODEL, int TY, int TZ, int R, int QPT, int MINB>
TileOps make_ops_rows()
{
    using G = RowGeom<DIM, MODEL, TY, TZ>;
    constexpr int NT = G::NS / (4 * QPT);
    TileOps o;
    o.tx = 32; o.ty = TY; o.tz = TZ; o.nt = NT; o.nt_bl = RowKernelTraits<DIM, MODEL, TY, TZ, R>::NT; o.rows = R;
    o.smem_bond_label = G::smem_bytes;
    o.bond_label = k_bond_label_rows<DIM, MODEL, TY, TZ, R, MINB>;
    o.merge = k_merge<DIM, 32, TY, TZ>;
    o.flip = k_flip<DIM, MODEL, 32, TY, TZ, NT>;
    o.export_labels = k_export_labels<DIM, 32, TY, TZ>;
    o.tile_origin = k_tile_origin<32, TY, TZ>;
    return o;
}

// Tile menu of the row kernel (Ising, Potts): 32 x TY (x TZ) sites, R rows per thread.  rows = 0 picks the
// default R of the tile.
template <int MODEL>
bool pick_ops_rows(int dim, int tx, int ty, int tz, int rows, TileOps &o)
{
    if (tx != 32) return false;
#ifdef SW_MENU_MIN   // developer builds: few instantiations (fast to compile)
#ifndef SW_EXP_FLIP_QPT
#define SW_EXP_FLIP_QPT 8
#endif
    if (MODEL != ISING) return false;
    if (dim == 3 && ty == 32 && tz == 16) { o = make_ops_rows<3, ISING, 32, 16, 1, SW_EXP_FLIP_QPT, 4>(); return true; }
    if (dim == 2 && ty == 128) { o = make_ops_rows<2, ISING, 128, 1, 1, 4, 12>(); return true; }
    return false;
#else
#define SW_ROWS2(Y, RR, Q, B) if (dim == 2 && ty == Y && (rows == RR || rows == 0)) { o = make_ops_rows<2, MODEL, Y, 1, RR, Q, B>(); return true; }
#define SW_ROWS3(Z, RR, Q, B) if (dim == 3 && ty == 32 && tz == Z && (rows == RR || rows == 0)) { o = make_ops_rows<3, MODEL, 32, Z, RR, Q, B>(); return true; }
    SW_ROWS2(32, 1, 1, 16)
    SW_ROWS2(128, 1, 4, 12)
    SW_ROWS2(128, 2, 4, 8)
    SW_ROWS2(256, 1, 4, 6)
    SW_ROWS2(256, 2, 4, 6)
    SW_ROWS2(512, 1, 8, 3)
    SW_ROWS2(512, 2, 8, 3)
    SW_ROWS3(4, 1, 4, 12)
    SW_ROWS3(8, 1, 4, 6)
    SW_ROWS3(8, 2, 4, 6)
    SW_ROWS3(16, 1, 8, (MODEL == ISING ? 4 : 3))   // Ising: 32 registers and 54.8 KB per CTA, four CTAs per SM
    SW_ROWS3(16, 2, 8, 3)
#undef SW_ROWS2
#undef SW_ROWS3
    return false;
#endif
}

// XY, clock on the row kernel: one row per thread only (the warp makes the masks of its 32 rows together).
template <int MODEL>
bool pick_ops_rows1(int dim, int tx, int ty, int tz, TileOps &o)
{
    if (tx != 32) return false;
#ifdef SW_MENU_MIN
    return false;
#else
    if (dim == 2 && ty == 32) { o = make_ops_rows<2, MODEL, 32, 1, 1, 1, 16>(); return true; }
    if (dim == 2 && ty == 128) { o = make_ops_rows<2, MODEL, 128, 1, 1, 4, 12>(); return true; }
    if (dim == 2 && ty == 256) { o = make_ops_rows<2, MODEL, 256, 1, 1, 4, 6>(); return true; }
    if (dim == 3 && ty == 32 && tz == 4) { o = make_ops_rows<3, MODEL, 32, 4, 1, 4, 12>(); return true; }
    if (dim == 3 && ty == 32 && tz == 8) { o = make_ops_rows<3, MODEL, 32, 8, 1, 4, 6>(); return true; }
    if (dim == 3 && ty == 32 && tz == 16) { o = make_ops_rows<3, MODEL, 32, 16, 1, 8, (MODEL == XY ? 4 : 3)>(); return true; }
    return false;
#endif
}

// Tile menu of the quad kernel (XY, clock; round-1 kernel, kept selectable with SW_B200_KERNEL=quad).  Tile sides are powers of two, TX in {32, 64, 128}; every side
// must divide L.
template <int MODEL>
bool pick_ops(int dim, int tx, int ty, int tz, TileOps &o)
{
#ifdef SW_MENU_MIN
    return false;
#endif
#define SW_TILE2(X, Y) if (dim == 2 && tx == X && ty == Y) { o = make_ops<2, MODEL, X, Y, 1>(); return true; }
#define SW_TILE3(X, Y, Z) if (dim == 3 && tx == X && ty == Y && tz == Z) { o = make_ops<3, MODEL, X, Y, Z>(); return true; }
    SW_TILE2(32, 32)
    SW_TILE2(64, 64)
    SW_TILE2(128, 32)
    SW_TILE2(128, 64)
    SW_TILE3(32, 8, 8)
    SW_TILE3(32, 16, 8)
    SW_TILE3(32, 16, 16)
    SW_TILE3(64, 8, 8)
#undef SW_TILE2
#undef SW_TILE3
    return false;
}

// Which bond / label kernel a model runs: the row kernel (sw_rows.cuh) for every model; the quad kernel of
// round 1 (sw_kernels.cuh k_bond_label) stays selectable for XY and the clock model with SW_B200_KERNEL=quad.
// Measured (ms per step, rows vs quad): clock X3 0.249 vs 0.260; XY with the SFU intrinsics C5 0.245 vs
// 0.247, X2 0.080 vs 0.084 (with full-precision sincosf the row kernel lost on XY, 0.341 vs 0.286: it computes
// the projection of the +z neighbour a second time).
bool use_rows(int model)
{
    if (model == SW_ISING || model == SW_POTTS) return true;
    const char *kern = std::getenv("SW_B200_KERNEL");
    return !(kern && std::strcmp(kern, "quad") == 0);
}

// Small lattices (fewer tiles than the GPU has room for): what counts is the critical path of one CTA,
// so the smallest tile of the menu with the fewest sites per thread.
bool pick_ops_small_model(int model, int dim, TileOps &o)
{
#ifdef SW_MENU_MIN
    return false;
#endif
    if (model == SW_ISING) return pick_ops_rows<ISING>(dim, 32, 32, dim == 3 ? 4 : 1, 1, o);
    if (model == SW_POTTS) return pick_ops_rows<POTTS>(dim, 32, 32, dim == 3 ? 4 : 1, 1, o);
    if (!use_rows(model)) {
        if (model == SW_CLOCK) { if (dim == 2) o = make_ops<2, CLOCK, 32, 32, 1, 1>(); else o = make_ops<3, CLOCK, 32, 8, 8, 1>(); return true; }
        if (dim == 2) o = make_ops<2, XY, 32, 32, 1, 1>(); else o = make_ops<3, XY, 32, 8, 8, 1>();
        return true;
    }
    if (model == SW_CLOCK) return pick_ops_rows1<CLOCK>(dim, 32, 32, dim == 3 ? 4 : 1, o);
    return pick_ops_rows1<XY>(dim, 32, 32, dim == 3 ? 4 : 1, o);
}

bool pick_ops_model(int model, int dim, int tx, int ty, int tz, int rows, TileOps &o)
{
    if (model == SW_ISING) return pick_ops_rows<ISING>(dim, tx, ty, tz, rows, o);
    if (model == SW_POTTS) return pick_ops_rows<POTTS>(dim, tx, ty, tz, rows, o);
    const bool quad = !use_rows(model);
    if (model == SW_CLOCK) return quad ? pick_ops<CLOCK>(dim, tx, ty, tz, o) : pick_ops_rows1<CLOCK>(dim, tx, ty, tz, o);
    return quad ? pick_ops<XY>(dim, tx, ty, tz, o) : pick_ops_rows1<XY>(dim, tx, ty, tz, o);
}

// Default tile of a lattice (SW_B200_TILE=TXxTYxTZ and SW_B200_ROWS=R override it: tuning knobs).
void default_tile(int dim, int L, int model, int &tx, int &ty, int &tz)
{
    const bool rows = use_rows(model);
    if (dim == 2) {
        tz = 1;
        if (rows) { tx = 32; ty = (L % 128 == 0) ? 128 : 32; }   // measured on C2 / C3: 32 x 128, one row per thread
        else if (L % 64 == 0) { tx = 64; ty = 64; }   // measured on C2 / C3 (round 1): 64x64 3 % ahead of 128x64
        else { tx = 32; ty = 32; }
    } else {
        tx = 32;
        if (rows) { ty = 32; tz = (L % 16 == 0) ? 16 : (L % 8 == 0 ? 8 : 4); }
        else { ty = 16; tz = 16; }  // XY: 75 KB of shared memory per CTA (projections + labels)
    }
}

int draw_bits(int model, int q)
{
    if (model != SW_POTTS) return 1;
    int b = 1;
    while ((1 << b) < q) ++b;
    return b;
}

size_t align256(size_t v) { return (v + 255) / 256 * 256; }

bool valid_args(int dim, int L, int model, int q, double beta, bool check_beta)
{
    if (dim != 2 && dim != 3) return false;
    if (L < 32 || L % 32 != 0) return false;
    if (model != SW_ISING && model != SW_POTTS && model != SW_XY && model != SW_CLOCK) return false;
    if (model == SW_POTTS && (q < 2 || q > 255)) return false;
    if (model == SW_CLOCK && (q < 2 || q > 512)) return false;  // q <= 512
    if (check_beta && !(std::isfinite(beta) && beta >= 0.0)) return false;
    double n = std::pow((double)L, dim);
    if (n > 2147483648.0) return false;
    // a label word holds (site address << draw bits) | draw
    if (n * (double)(1u << draw_bits(model, q)) > 4294967296.0) return false;
    return true;
}

struct Layout { size_t spins, bonds, labels, pairs, origin, table, acc, total; };

size_t spin_bytes(int model) { return model == SW_XY ? 4 : (model == SW_CLOCK ? 2 : 1); }

Layout layout(int dim, int L, int model, int q)
{
    size_t N = 1;
    for (int a = 0; a < dim; ++a) N *= (size_t)L;
    Layout l;
    size_t off = 0;
    l.spins = off; off += align256(N * spin_bytes(model));
    l.bonds = off; off += align256(N);
    l.labels = off; off += align256(N * 4);
    // pair list: one (i, j) address pair per bond through a tile face, sized for the tile of the menu
    // with the largest face area (3D 32x32x4: (1/32 + 1/32 + 1/4) N bonds; 2D 32x32: N/16); then the
    // tile origins (smallest tile: 1024 sites)
    l.pairs = off; off += align256((dim == 3 ? N / 32 * 10 : N / 16) * 8);
    l.origin = off; off += align256((N / 1024) * 4);
    l.table = off; off += align256(model == SW_CLOCK ? (size_t)q * q * 4 : 0);  // clock: bond thresholds
    l.acc = off; off += align256(sizeof(Acc));
    l.total = off;
    return l;
}

}  // namespace

struct sw_ctx {
    int dim, L, model, q;
    double beta;
    uint64_t seed, t;
    size_t N;
    Params p;
    TileOps ops;
    cudaStream_t stream;
    void *workspace;
    uint8_t *bonds_mem;
    unsigned merge_blocks;
    // lattices of at most 32768 sites (Ising, Potts): the whole step in one CTA, n steps per launch (sw_small.cuh)
    bool small;
    size_t small_smem;
    void (*small_kernel)(const Params, const SmallArgs);
    // CUDA graphs of 1 and GRAPH_STEPS consecutive steps (3 kernel nodes per step); built lazily for
    // Ising / Potts, rebuilt when the bond-recording flag changes.  XY passes a new direction with
    // every step and keeps plain launches.
    unsigned long long *series_dev;   // sw_run_series: device records, kept and grown on demand
    size_t series_cap;                // in 64-bit words
    cudaGraphExec_t graph1, graphK;
    int graph_record;   // record_bonds state the graphs were built for (-1: none)
    bool own_workspace, own_stream;
    bool stepped;      // labels of a step are available
    bool bonds_valid;  // the last step recorded its bond bytes
    int record_bonds;
    bool M_fresh;      // acc holds the magnetisation sums of the current configuration
    bool E_fresh;
    int force_phi;
    double forced_phi;
    float rx, ry, crefl;
    int mirror;
    int sticky;
    int timing;            // per-kernel event timing mode
    cudaEvent_t ev[4];
    double kernel_ms[3];
    uint64_t timed_steps;
};

namespace {

int cuda_fail(sw_ctx *c, cudaError_t e, const char *what)
{
    if (c) c->sticky = 1;
    return fail(SW_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define SW_CUDA(c, call)                                         \
    do {                                                         \
        cudaError_t e_ = (call);                                 \
        if (e_ != cudaSuccess) return cuda_fail(c, e_, #call);   \
    } while (0)

int check_ctx(sw_ctx *c)
{
    if (!c) return fail(SW_EINVAL, "null context");
    if (c->sticky) return fail(SW_ECUDA, "context is in a sticky CUDA error state");
    return SW_OK;
}

dim3 tile_grid(const sw_ctx *c)
{
    return dim3(c->p.ntx, c->p.nty, c->p.ntz);
}

uint32_t threshold32(double prob)
{
    double v = std::floor(prob * 4294967296.0);
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

template <int MODEL>
void launch_init(sw_ctx *c)
{
    k_init<MODEL><<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(c->p);
}

template <int DIM, int MODEL>
void launch_measure_dm(sw_ctx *c, bool with_m)
{
    if (MODEL == XY) {
        const unsigned g = (unsigned)(c->N / 1024);  // four sites per thread
        if (with_m) k_measure_xy<DIM, true><<<g, 256, 0, c->stream>>>(c->p);
        else k_measure_xy<DIM, false><<<g, 256, 0, c->stream>>>(c->p);
    } else {
        unsigned g = (unsigned)(c->N / 4096);        // 16 sites per thread and iteration, grid-stride
        if (g < 1u) g = 1u;
        if (g > 148u * 8u) g = 148u * 8u;            // a CTA adds to the global sums once
        if (with_m) k_measure4<DIM, MODEL, true><<<g, 256, 0, c->stream>>>(c->p);
        else k_measure4<DIM, MODEL, false><<<g, 256, 0, c->stream>>>(c->p);
    }
}

void launch_measure(sw_ctx *c, bool with_m)
{
    if (c->model == SW_CLOCK) {
        unsigned g = (unsigned)(c->N / 256);
        if (g > 148u * 8u) g = 148u * 8u;   // a CTA flushes its histograms once: few CTAs, many sites each
        if (c->dim == 2) k_measure_clock<2><<<g, 256, 0, c->stream>>>(c->p);
        else k_measure_clock<3><<<g, 256, 0, c->stream>>>(c->p);
        return;
    }
    if (c->dim == 2) {
        if (c->model == SW_ISING) launch_measure_dm<2, ISING>(c, with_m);
        else if (c->model == SW_POTTS) launch_measure_dm<2, POTTS>(c, with_m);
        else launch_measure_dm<2, XY>(c, with_m);
    } else {
        if (c->model == SW_ISING) launch_measure_dm<3, ISING>(c, with_m);
        else if (c->model == SW_POTTS) launch_measure_dm<3, POTTS>(c, with_m);
        else launch_measure_dm<3, XY>(c, with_m);
    }
}

// Make acc hold E (and M) of the current configuration.
int refresh_observables(sw_ctx *c)
{
    if (c->E_fresh && c->M_fresh) return SW_OK;
    const bool with_m = !c->M_fresh || c->model == SW_CLOCK;  // clock: both histograms in one pass
    // E_int and E_xy are the first 16 bytes of Acc; the magnetisation sums follow.
    const size_t clear = with_m ? offsetof(Acc, stats) : offsetof(Acc, M_int);
    SW_CUDA(c, cudaMemsetAsync(c->p.acc, 0, clear, c->stream));
    launch_measure(c, with_m);
    SW_CUDA(c, cudaGetLastError());
    c->E_fresh = c->M_fresh = true;
    return SW_OK;
}

// Extensive observables from the accumulator head (E_int, E_xy, M_int, mx, my, n_k[q]).
void sums_to_observables(const sw_ctx *c, const unsigned long long *w, const unsigned long long *nk,
                         const unsigned long long *dk, double &e, double &m, double &m2)
{
    double dv[5];
    std::memcpy(dv, w, sizeof(dv));
    if (c->model == SW_CLOCK) {
        // Eq. (3) with theta = 2 pi p / q from the exact histograms (the paper's tables rule[] and
        // fmy[]), summed in increasing d and p
        const double two_pi = 6.283185307179586476925286766559;
        const int q = c->q;
        double mx = 0.0, my = 0.0;
        e = 0.0;
        for (int d = 0; d < q; ++d) e -= (double)(long long)dk[d] * std::cos(two_pi * (double)d / (double)q);
        for (int pp = 0; pp < q; ++pp) {
            mx += (double)(long long)nk[pp] * std::cos(two_pi * (double)pp / (double)q);
            my += (double)(long long)nk[pp] * std::sin(two_pi * (double)pp / (double)q);
        }
        m2 = mx * mx + my * my;
        m = std::sqrt(m2);
        return;
    }
    if (c->model == SW_ISING) {
        e = (double)(long long)w[0];
        m = (double)(long long)w[2];
        m2 = m * m;
    } else if (c->model == SW_POTTS) {
        // Eq. (5): M^2 = (q sum_k n_k^2 - N^2) / (q - 1)
        double s2 = 0.0;
        for (int k = 0; k < c->q; ++k) s2 += (double)nk[k] * (double)nk[k];
        const double Nd = (double)c->N;
        e = (double)(long long)w[0];
        m2 = ((double)c->q * s2 - Nd * Nd) / (double)(c->q - 1);
        m = std::sqrt(m2);
    } else {
        e = dv[1];
        m2 = dv[3] * dv[3] + dv[4] * dv[4];
        m = std::sqrt(m2);
    }
}

int create_common(sw_ctx **out, int dim, int L, int model, int q, double beta, uint64_t seed,
                  void *workspace, size_t workspace_bytes, void *stream, bool external)
{
    if (!out) return fail(SW_EINVAL, "out is NULL");
    *out = nullptr;
    if (!valid_args(dim, L, model, q, beta, true))
        return fail(SW_EINVAL, "invalid arguments (dim 2|3, L multiple of 32 with L^dim <= 2^31 and L^dim 2^ceil(log2 q) <= 2^32, model, Potts 2<=q<=255 / clock 2<=q<=512, beta>=0)");
    const Layout lay = layout(dim, L, model, q);
    if (external) {
        if (!workspace || workspace_bytes < lay.total || ((uintptr_t)workspace & 255u))
            return fail(SW_EINVAL, "device workspace missing, too small or not 256-byte aligned");
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(SW_ECUDA, "no usable CUDA device (this library has no CPU fallback)");
    }
    sw_ctx *c = new (std::nothrow) sw_ctx();
    if (!c) return fail(SW_ENOMEM, "host allocation failed");
    c->dim = dim; c->L = L; c->model = model; c->q = (model == SW_POTTS || model == SW_CLOCK) ? q : 0;
    c->beta = beta; c->seed = seed; c->t = 0;
    c->N = lay.total ? 1 : 0;
    for (int a = 0; a < dim; ++a) c->N *= (size_t)L;
    c->own_workspace = !external; c->own_stream = !external;
    c->stream = external ? (cudaStream_t)stream : nullptr;
    c->workspace = workspace;
    if (!external) {
        e = cudaMalloc(&c->workspace, lay.total);
        if (e != cudaSuccess) { cudaGetLastError(); delete c; return fail(SW_ENOMEM, "cudaMalloc failed"); }
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { cudaFree(c->workspace); delete c; return fail(SW_ECUDA, "cudaStreamCreate failed"); }
    }
    // tile choice: default per dimension and model, SW_B200_TILE=TXxTYxTZ / SW_B200_ROWS=R override (tuning knobs)
    int tx, ty, tz, rows = 0;
    default_tile(dim, L, model, tx, ty, tz);
    const char *env_tile = std::getenv("SW_B200_TILE");
    if (env_tile) {
        int ex = 0, ey = 0, ez = 1;
        if (std::sscanf(env_tile, "%dx%dx%d", &ex, &ey, &ez) >= 2) { tx = ex; ty = ey; tz = (dim == 2) ? 1 : ez; }
    }
    if (const char *env = std::getenv("SW_B200_ROWS")) rows = std::atoi(env);
    bool ok = tx > 0 && ty > 0 && tz > 0 && (L % tx == 0) && (L % ty == 0) && (L % tz == 0) &&
              pick_ops_model(model, dim, tx, ty, tz, rows, c->ops);
    if (!ok) ok = pick_ops_small_model(model, dim, c->ops);
    if (!env_tile) {
        // fewer default tiles than 2 per SM: latency variant (smallest tile, fewest sites per thread)
        int sms = 148, dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const size_t ntiles_default = c->N / ((size_t)c->ops.tx * c->ops.ty * c->ops.tz);
        if (ntiles_default < (size_t)2 * sms) pick_ops_small_model(model, dim, c->ops);
    }
    c->small = false; c->small_smem = 0; c->small_kernel = nullptr;
#ifndef SW_MENU_MIN
    if ((model == SW_ISING || model == SW_POTTS) && c->N <= 32768 && !std::getenv("SW_B200_NO_SMALL")) {
        c->small = true;
        if (model == SW_ISING) {
            c->small_kernel = (dim == 2) ? k_sw_small<2, ISING> : k_sw_small<3, ISING>;
            c->small_smem = 4 * ((dim == 2) ? SmallGeom<2, ISING>::words(c->N) : SmallGeom<3, ISING>::words(c->N));
        } else {
            c->small_kernel = (dim == 2) ? k_sw_small<2, POTTS> : k_sw_small<3, POTTS>;
            c->small_smem = 4 * ((dim == 2) ? SmallGeom<2, POTTS>::words(c->N) : SmallGeom<3, POTTS>::words(c->N));
        }
    }
#endif
    char *base = (char *)c->workspace;
    Params &p = c->p;
    p.spins = base + lay.spins;
    p.bonds = nullptr;
    c->bonds_mem = (uint8_t *)(base + lay.bonds);
    p.labels = (uint32_t *)(base + lay.labels);
    p.pairs = (uint2 *)(base + lay.pairs);
    p.npairs = &((Acc *)(base + lay.acc))->npairs;
    p.tile_origin = (uint32_t *)(base + lay.origin);
    p.labels_out = nullptr;
    p.acc = (Acc *)(base + lay.acc);
    p.ntx = (uint32_t)(L / c->ops.tx); p.nty = (uint32_t)(L / c->ops.ty);
    p.ntz = (dim == 3) ? (uint32_t)(L / c->ops.tz) : 1u;
    p.ntiles = p.ntx * p.nty * p.ntz;
    p.db = draw_bits(model, q);
    {   // k_merge: grid-stride loop over the pair list.  The grid is fixed at create time (graph replay) from
        // the capacity of the list; 96 CTAs per SM leave about one pair per thread at T_c, so that CTAs
        // run through the list in order (the list is in tile order: neighbouring pairs touch neighbouring
        // label blocks, which stay in L2).  A resident grid (8 CTAs per SM, 13 pairs per thread) sweeps the
        // whole label array 13 times instead: C4 k_merge 0.264 ms vs 0.138 ms.
        int dev = 0, sms = 148;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const size_t max_pairs = c->N / c->ops.tx + c->N / c->ops.ty + (dim == 3 ? c->N / c->ops.tz : 0);
        size_t blocks = (max_pairs + 255) / 256;
        if (blocks > (size_t)sms * 96) blocks = (size_t)sms * 96;   // (C4: 64 / 80 / 96 / 112 CTAs per SM: 0.133 / 0.133 / 0.129 / 0.136 ms)
        if (const char *env = std::getenv("SW_B200_MERGE_BLOCKS")) {   // test knob: another interleaving of the unions
            const long v = std::atol(env);
            if (v >= 1 && v <= 65535 * 16) blocks = (size_t)v;
        }
        c->merge_blocks = (unsigned)blocks;
    }
    p.L = (uint32_t)L; p.N = (uint32_t)c->N;
    p.k0 = (uint32_t)(seed & 0xffffffffu); p.k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { p.rk[2 * r] = p.k0 + (uint32_t)r * 0x9E3779B9u; p.rk[2 * r + 1] = p.k1 + (uint32_t)r * 0xBB67AE85u; }
    // PAPER.md:96 (garbled "p = 1 e^{2J/T}"): Ising p = 1 - exp(-2 beta); PAPER.md:152 + Eq. 2: Potts
    // p = 1 - exp(-beta).  The decision is the integer compare word < floor(p 2^32).
    const double prob = (model == SW_ISING) ? -std::expm1(-2.0 * beta) : -std::expm1(-beta);
    p.P32 = threshold32(prob);
    p.q = c->q;
    p.rx = 1.f; p.ry = 0.f; p.crefl = 0.f; p.m2beta = (float)(-2.0 * beta);
    p.clock_T = (const uint32_t *)(base + lay.table);
    p.mirror = 0; c->mirror = 0;
    p.counting = 0;
    p.nk_clear = (model == SW_POTTS) ? q : 0;
    c->force_phi = 0; c->forced_phi = 0.0; c->rx = c->ry = c->crefl = 0.f; c->sticky = 0;
    c->graph1 = nullptr; c->graphK = nullptr; c->graph_record = -1;
    c->series_dev = nullptr; c->series_cap = 0;
    c->timing = 0; c->timed_steps = 0;
    for (int k = 0; k < 3; ++k) c->kernel_ms[k] = 0.0;
    for (int k = 0; k < 4; ++k) c->ev[k] = nullptr;

    auto bail = [&](cudaError_t err, const char *what) {
        std::string m = std::string(what) + ": " + cudaGetErrorString(err);
        if (c->own_workspace) cudaFree(c->workspace);
        if (c->own_stream) cudaStreamDestroy(c->stream);
        delete c;
        return fail(SW_ECUDA, m);
    };
    e = cudaFuncSetAttribute(c->ops.bond_label, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ops.smem_bond_label);
    if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_bond_label)");
    if (model == SW_ISING || model == SW_POTTS || model == SW_XY) {
        // all of the SM's shared memory for the CTAs of the bond / label kernel (four CTAs of 54.7 KB for the 3D Ising
        // and XY tiles); the clock model keeps the default split: its threshold-table reads live on L1
        e = cudaFuncSetAttribute(c->ops.bond_label, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_bond_label, carveout)");
    }
    if (c->small) {
        e = cudaFuncSetAttribute(c->small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->small_smem);
        if (e != cudaSuccess) return bail(e, "cudaFuncSetAttribute(k_sw_small)");
    }
    c->ops.tile_origin<<<(p.ntiles + 255) / 256, 256, 0, c->stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return bail(e, "k_tile_origin launch");
    e = cudaMemsetAsync(p.acc, 0, sizeof(Acc), c->stream);
    if (e != cudaSuccess) return bail(e, "cudaMemsetAsync");
    if (model == SW_CLOCK) {
        // clock model, reading 24: component along the mirror normal |a(u)| = sin(pi u / q), u = 1..q-1;
        // bond threshold T[u_i q + u_j] = floor((1 - exp(-2 beta a_i a_j)) 2^32), in double on the host
        const double two_pi = 6.283185307179586476925286766559;
        std::vector<double> mag((size_t)q, 0.0);
        for (int u = 0; u < q; ++u) mag[u] = std::sin((two_pi / 2.0) * (double)u / (double)q);
        std::vector<uint32_t> tab((size_t)q * q, 0u);
        for (int ui = 1; ui < q; ++ui)
            for (int uj = 1; uj < q; ++uj)
                tab[(size_t)ui * q + uj] = threshold32(-std::expm1(-2.0 * beta * (mag[ui] * mag[uj])));
        e = cudaMemcpyAsync((void *)p.clock_T, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);  // tab goes out of scope
        if (e != cudaSuccess) return bail(e, "clock threshold table");
    }
    if (model == SW_ISING) launch_init<ISING>(c);
    else if (model == SW_POTTS) launch_init<POTTS>(c);
    else if (model == SW_CLOCK) launch_init<CLOCK>(c);
    else launch_init<XY>(c);
    e = cudaGetLastError();
    if (e != cudaSuccess) return bail(e, "k_init launch");
    c->stepped = false; c->bonds_valid = false; c->record_bonds = 0; c->M_fresh = false; c->E_fresh = false;
    *out = c;
    return SW_OK;
}

}  // namespace

extern "C" {

const char *sw_last_error(void) { return g_err.c_str(); }

size_t sw_workspace_bytes(int dim, int L, int model, int q)
{
    if (!valid_args(dim, L, model, q, 0.0, false)) return 0;
    return layout(dim, L, model, q).total;
}

int sw_create(sw_ctx **out, int dim, int L, int model, int q, double beta, uint64_t seed)
{
    return create_common(out, dim, L, model, q, beta, seed, nullptr, 0, nullptr, false);
}

int sw_create_in(sw_ctx **out, int dim, int L, int model, int q, double beta, uint64_t seed,
                 void *device_workspace, size_t workspace_bytes, void *cuda_stream)
{
    return create_common(out, dim, L, model, q, beta, seed, device_workspace, workspace_bytes, cuda_stream, true);
}

namespace {

constexpr int GRAPH_STEPS = 16;

// A graph of `steps` consecutive SW steps: k_bond_label -> k_merge -> k_flip, chained.  The kernels take
// the step index from device memory, so the same graph serves every step.
int build_graph(sw_ctx *c, int steps, cudaGraphExec_t *out)
{
    cudaGraph_t g = nullptr;
    SW_CUDA(c, cudaGraphCreate(&g, 0));
    Params p = c->p;
    void *args[1] = {&p};
    const dim3 grid = tile_grid(c);
    cudaGraphNode_t prev = nullptr;
    cudaError_t e = cudaSuccess;
    for (int s = 0; s < steps && e == cudaSuccess; ++s) {
        for (int k = 0; k < 3 && e == cudaSuccess; ++k) {
            cudaKernelNodeParams kp = {};
            kp.kernelParams = args;
            kp.extra = nullptr;
            if (k == 0) { kp.func = (void *)c->ops.bond_label; kp.gridDim = grid; kp.blockDim = dim3(c->ops.nt_bl); kp.sharedMemBytes = (unsigned)c->ops.smem_bond_label; }
            if (k == 1) { kp.func = (void *)c->ops.merge; kp.gridDim = dim3(c->merge_blocks); kp.blockDim = dim3(256); kp.sharedMemBytes = 0; }
            if (k == 2) { kp.func = (void *)c->ops.flip; kp.gridDim = grid; kp.blockDim = dim3(c->ops.nt); kp.sharedMemBytes = 0; }
            cudaGraphNode_t node = nullptr;
            e = cudaGraphAddKernelNode(&node, g, prev ? &prev : nullptr, prev ? 1 : 0, &kp);
            prev = node;
        }
    }
    if (e == cudaSuccess) e = cudaGraphInstantiate(out, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) return cuda_fail(c, e, "building the step graph");
    return SW_OK;
}

}  // namespace

int sw_step(sw_ctx *c, int n)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (n < 0) return fail(SW_EINVAL, "n < 0");
    const dim3 grid = tile_grid(c);
    if (c->small) {
        // one CTA holds the lattice: n steps in one launch
        if (n == 0) return SW_OK;
        c->p.bonds = c->record_bonds ? c->bonds_mem : nullptr;
        SmallArgs a;
        a.nsteps = n; a.write_labels = 1; a.series = nullptr; a.series_words = 0;
        if (c->p.counting) SW_CUDA(c, cudaMemsetAsync(c->p.acc->stats, 0, sizeof(c->p.acc->stats), c->stream));
        if (c->timing) SW_CUDA(c, cudaEventRecord(c->ev[0], c->stream));
        c->small_kernel<<<1, 1024, c->small_smem, c->stream>>>(c->p, a);
        if (c->timing) {
            SW_CUDA(c, cudaEventRecord(c->ev[1], c->stream));
            SW_CUDA(c, cudaEventSynchronize(c->ev[1]));
            float ms = 0.f;
            SW_CUDA(c, cudaEventElapsedTime(&ms, c->ev[0], c->ev[1]));
            c->kernel_ms[0] += (double)ms;
            c->timed_steps += (uint64_t)n;
        }
        SW_CUDA(c, cudaGetLastError());
        c->t += (uint64_t)n;
        c->stepped = true; c->bonds_valid = c->record_bonds != 0;
        c->M_fresh = true; c->E_fresh = true;   // the kernel leaves E and M of the new configuration in acc
        return SW_OK;
    }
    if (c->model != SW_XY && c->model != SW_CLOCK && !c->timing && !c->p.counting && n > 0 && !std::getenv("SW_B200_NO_GRAPH")) {
        // launch-bound regime (small lattices): 3 launches per step cost more host time than the
        // kernels take; replay pre-built graphs instead
        if (c->graph_record != c->record_bonds) {
            if (c->graph1) { cudaGraphExecDestroy(c->graph1); c->graph1 = nullptr; }
            if (c->graphK) { cudaGraphExecDestroy(c->graphK); c->graphK = nullptr; }
            c->p.bonds = c->record_bonds ? c->bonds_mem : nullptr;
            rc = build_graph(c, 1, &c->graph1);
            if (rc == SW_OK) rc = build_graph(c, GRAPH_STEPS, &c->graphK);
            if (rc) return rc;
            c->graph_record = c->record_bonds;
        }
        int left = n;
        while (left >= GRAPH_STEPS) { SW_CUDA(c, cudaGraphLaunch(c->graphK, c->stream)); left -= GRAPH_STEPS; }
        while (left > 0) { SW_CUDA(c, cudaGraphLaunch(c->graph1, c->stream)); --left; }
        c->t += (uint64_t)n;
        c->stepped = true; c->bonds_valid = c->record_bonds != 0;
        c->M_fresh = true; c->E_fresh = false;
        return SW_OK;
    }
    for (int s = 0; s < n; ++s) {
        Params &p = c->p;
        p.bonds = c->record_bonds ? c->bonds_mem : nullptr;
        if (c->model == SW_XY) {
            // PAPER.md:159 "randomly chosen" direction: phi uniform from one Philox word (domain 3),
            // r = (cos phi, sin phi) rounded to fp32; reflection constant c = (2 phi + pi) mod 2 pi.
            const double two_pi = 6.283185307179586476925286766559;
            const uint4 w = philox4x32_10(0u, (uint32_t)(c->t & 0xffffffffu), (uint32_t)(c->t >> 32), DOM_XYDIR, p.k0, p.k1);
            double phi = (double)w.x * (two_pi / 4294967296.0);
            if (c->force_phi) phi = c->forced_phi;
            p.rx = c->rx = (float)std::cos(phi);
            p.ry = c->ry = (float)std::sin(phi);
            p.crefl = c->crefl = (float)std::fmod(2.0 * phi + two_pi / 2.0, two_pi);
        }
        if (c->model == SW_CLOCK) {
            // "The variable ispr, which is randomly chosen, specifies the direction for
            // mirror projection": m = (word q) >> 32 from the XYDIR call of the step (reading 23)
            const uint4 w = philox4x32_10(0u, (uint32_t)(c->t & 0xffffffffu), (uint32_t)(c->t >> 32), DOM_XYDIR, p.k0, p.k1);
            p.mirror = c->mirror = (int)(((unsigned long long)w.x * (unsigned long long)c->q) >> 32);
        }
        if (p.counting) {
            SW_CUDA(c, cudaMemsetAsync(p.acc->stats, 0, sizeof(p.acc->stats), c->stream));
            const unsigned long long examined = (unsigned long long)c->N / c->ops.tx + c->N / c->ops.ty +
                                                (c->dim == 3 ? c->N / c->ops.tz : 0);
            SW_CUDA(c, cudaMemcpyAsync(&p.acc->stats[0], &examined, 8, cudaMemcpyHostToDevice, c->stream));
        }
        if (c->timing) SW_CUDA(c, cudaEventRecord(c->ev[0], c->stream));
        c->ops.bond_label<<<grid, c->ops.nt_bl, c->ops.smem_bond_label, c->stream>>>(p);
        if (c->timing) SW_CUDA(c, cudaEventRecord(c->ev[1], c->stream));
        c->ops.merge<<<c->merge_blocks, 256, 0, c->stream>>>(p);
        if (c->timing) SW_CUDA(c, cudaEventRecord(c->ev[2], c->stream));
        c->ops.flip<<<grid, c->ops.nt, 0, c->stream>>>(p);
        if (c->timing) {
            SW_CUDA(c, cudaEventRecord(c->ev[3], c->stream));
            SW_CUDA(c, cudaEventSynchronize(c->ev[3]));
            for (int k = 0; k < 3; ++k) {
                float ms = 0.f;
                SW_CUDA(c, cudaEventElapsedTime(&ms, c->ev[k], c->ev[k + 1]));
                c->kernel_ms[k] += (double)ms;
            }
            c->timed_steps += 1;
        }
        c->t += 1;
    }
    if (n > 0) {
        SW_CUDA(c, cudaGetLastError());
        c->stepped = true; c->bonds_valid = c->record_bonds != 0;
        c->M_fresh = (c->model != SW_XY && c->model != SW_CLOCK);  // XY, clock: the magnetisation is summed on request
        c->E_fresh = false;
    }
    return SW_OK;
}

int sw_observables(sw_ctx *c, double *E, double *M, double *M2, double *M4)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    rc = refresh_observables(c);
    if (rc) return rc;
    Acc h;
    SW_CUDA(c, cudaMemcpyAsync(&h, c->p.acc, offsetof(Acc, stats), cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    double e, m, m2;
    sums_to_observables(c, (const unsigned long long *)&h, h.nk, h.dk, e, m, m2);
    if (E) *E = e;
    if (M) *M = m;
    if (M2) *M2 = m2;
    if (M4) *M4 = m2 * m2;
    return SW_OK;
}

int sw_run_series(sw_ctx *c, int n, double *E, double *M, double *M2, double *M4)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (n < 0) return fail(SW_EINVAL, "n < 0");
    if (n == 0) return SW_OK;
    // per step one record of 5 + q 64-bit words = the head of Acc (E_int, E_xy, M_int, mx, my, n_k)
    const int w1 = 5 + c->q, w2 = (c->model == SW_CLOCK) ? c->q : 0, words = w1 + w2;
    const int off2 = (int)(offsetof(Acc, dk) / 8);
    cudaError_t e = cudaSuccess;
    if (c->series_cap < (size_t)n * words) {
        // (re)allocate the record buffer; it stays with the context, so that calling this in a loop
        // costs no cudaMalloc / cudaFree (both synchronise the device)
        SW_CUDA(c, cudaStreamSynchronize(c->stream));
        if (c->series_dev) cudaFree(c->series_dev);
        c->series_dev = nullptr; c->series_cap = 0;
        e = cudaMalloc(&c->series_dev, (size_t)n * words * 8);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(SW_ENOMEM, "sw_run_series: cudaMalloc of the series buffer failed"); }
        c->series_cap = (size_t)n * words;
    }
    unsigned long long *dser = c->series_dev;
    if (c->small) {
        // the one-CTA kernel records E and M (n_k) of every step itself
        c->p.bonds = c->record_bonds ? c->bonds_mem : nullptr;
        SmallArgs a;
        a.nsteps = n; a.write_labels = 1; a.series = dser; a.series_words = words;
        c->small_kernel<<<1, 1024, c->small_smem, c->stream>>>(c->p, a);
        if (cudaGetLastError() != cudaSuccess) rc = fail(SW_ECUDA, "k_sw_small launch");
        c->t += (uint64_t)n;
        c->stepped = true; c->bonds_valid = c->record_bonds != 0;
        c->M_fresh = true; c->E_fresh = true;
    }
    for (int s = 0; s < n && rc == SW_OK && !c->small; ++s) {
        rc = sw_step(c, 1);
        if (rc == SW_OK) rc = refresh_observables(c);
        if (rc == SW_OK) {
            k_snapshot<<<1, 1024, 0, c->stream>>>(c->p.acc, dser + (size_t)s * words, w1, off2, w2);
            if (cudaGetLastError() != cudaSuccess) rc = fail(SW_ECUDA, "k_snapshot launch");
        }
    }
    unsigned long long *hser = nullptr;
    if (rc == SW_OK) {
        hser = (unsigned long long *)std::malloc((size_t)n * words * 8);
        if (!hser) rc = fail(SW_ENOMEM, "sw_run_series: host buffer");
    }
    if (rc == SW_OK) {
        e = cudaMemcpyAsync(hser, dser, (size_t)n * words * 8, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = cuda_fail(c, e, "sw_run_series copy");
    } else {
        cudaStreamSynchronize(c->stream);
    }
    if (rc == SW_OK) {
        for (int s = 0; s < n; ++s) {
            const unsigned long long *rec = hser + (size_t)s * words;
            double ev, m, m2;
            sums_to_observables(c, rec, rec + 5, rec + w1, ev, m, m2);
            if (E) E[s] = ev;
            if (M) M[s] = m;
            if (M2) M2[s] = m2;
            if (M4) M4[s] = m2 * m2;
        }
    }
    std::free(hser);
    return rc;
}

int sw_destroy(sw_ctx *c)
{
    if (!c) return SW_OK;
    cudaStreamSynchronize(c->stream);
    if (c->series_dev) cudaFree(c->series_dev);
    if (c->graph1) cudaGraphExecDestroy(c->graph1);
    if (c->graphK) cudaGraphExecDestroy(c->graphK);
    for (int k = 0; k < 4; ++k) if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    if (c->own_workspace) cudaFree(c->workspace);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    cudaGetLastError();
    delete c;
    return SW_OK;
}

size_t sw_num_sites(const sw_ctx *c) { return c ? c->N : 0; }
uint64_t sw_step_index(const sw_ctx *c) { return c ? c->t : 0; }

int sw_get_spins(sw_ctx *c, void *dst, size_t bytes)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    const size_t want = c->N * spin_bytes(c->model);
    if (!dst || bytes != want) return fail(SW_EINVAL, "sw_get_spins: buffer must hold exactly N elements");
    SW_CUDA(c, cudaMemcpyAsync(dst, c->p.spins, want, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_set_spins(sw_ctx *c, const void *src, size_t bytes, uint64_t step)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    const size_t want = c->N * spin_bytes(c->model);
    if (!src || bytes != want) return fail(SW_EINVAL, "sw_set_spins: buffer must hold exactly N elements");
    SW_CUDA(c, cudaMemcpyAsync(c->p.spins, src, want, cudaMemcpyHostToDevice, c->stream));
    const unsigned long long tdev = step;
    SW_CUDA(c, cudaMemcpyAsync(&c->p.acc->t, &tdev, 8, cudaMemcpyHostToDevice, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    c->t = step;
    c->stepped = false; c->bonds_valid = false; c->M_fresh = false; c->E_fresh = false;
    return SW_OK;
}

int sw_get_bonds(sw_ctx *c, uint8_t *dst, size_t bytes)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (!c->stepped) return fail(SW_ESTATE, "no step since create / sw_set_spins");
    if (!c->bonds_valid) return fail(SW_ESTATE, "the last step did not record its bonds (sw_set_record_bonds)");
    if (!dst || bytes != c->N) return fail(SW_EINVAL, "sw_get_bonds: buffer must hold exactly N bytes");
    SW_CUDA(c, cudaMemcpyAsync(dst, c->bonds_mem, c->N, cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    return SW_OK;
}

int sw_get_labels(sw_ctx *c, uint32_t *dst, size_t bytes)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (!c->stepped) return fail(SW_ESTATE, "no step since create / sw_set_spins");
    if (!dst || bytes != c->N * 4) return fail(SW_EINVAL, "sw_get_labels: buffer must hold exactly N uint32");
    // canonical labels (minimum linear site index, linear order) are made on request, in scratch
    // device memory that lives only for this call: the step itself never needs them
    uint32_t *out = nullptr;
    cudaError_t e = cudaMalloc(&out, c->N * 4);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SW_ENOMEM, "sw_get_labels: cudaMalloc of the export buffer failed"); }
    Params q = c->p;
    q.labels_out = out;
    if (c->small) k_export_labels_linear<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(q);
    else c->ops.export_labels<<<(unsigned)((c->N + 255) / 256), 256, 0, c->stream>>>(q);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(dst, out, c->N * 4, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(out);
    if (e != cudaSuccess) return cuda_fail(c, e, "sw_get_labels");
    return SW_OK;
}

int sw_get_cluster_stats(sw_ctx *c, uint64_t *n_clusters, uint64_t *sum_nc2)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (!c->stepped) return fail(SW_ESTATE, "no step since create / sw_set_spins");
    uint32_t *sizes = nullptr;
    cudaError_t e = cudaMalloc(&sizes, c->N * 4 + 16);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SW_ENOMEM, "sw_get_cluster_stats: cudaMalloc of the size counters failed"); }
    unsigned long long *out = (unsigned long long *)(sizes + c->N);
    unsigned long long h[2] = {0ull, 0ull};
    e = cudaMemsetAsync(sizes, 0, c->N * 4 + 16, c->stream);
    if (e == cudaSuccess) {
        const unsigned g = (unsigned)(c->N / 256);
        k_cluster_sizes<<<g, 256, 0, c->stream>>>(c->p, sizes);
        k_cluster_moments<<<g, 256, 0, c->stream>>>(c->p, sizes, out);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, out, 16, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(sizes);
    if (e != cudaSuccess) return cuda_fail(c, e, "sw_get_cluster_stats");
    if (n_clusters) *n_clusters = h[0];
    if (sum_nc2) *sum_nc2 = h[1];
    return SW_OK;
}

int sw_get_counts(sw_ctx *c, int64_t *E, int64_t *M_or_nk, int n)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (c->model == SW_XY) return fail(SW_EINVAL, "sw_get_counts: integer sums are not defined for XY");
    if (c->model == SW_CLOCK) return fail(SW_EINVAL, "sw_get_counts: use sw_get_clock_hist for the clock model");
    rc = refresh_observables(c);
    if (rc) return rc;
    Acc h;
    SW_CUDA(c, cudaMemcpyAsync(&h, c->p.acc, offsetof(Acc, stats), cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    if (E) *E = (int64_t)h.E_int;
    if (M_or_nk) {
        if (c->model == SW_ISING) { if (n >= 1) M_or_nk[0] = (int64_t)h.M_int; }
        else for (int k = 0; k < n && k < c->q; ++k) M_or_nk[k] = (int64_t)h.nk[k];
    }
    return SW_OK;
}

int sw_get_clock_hist(sw_ctx *c, int64_t *D, int64_t *n, int q)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (c->model != SW_CLOCK || q != c->q) return fail(SW_EINVAL, "sw_get_clock_hist: not a clock context, or q differs");
    rc = refresh_observables(c);
    if (rc) return rc;
    Acc h;
    SW_CUDA(c, cudaMemcpyAsync(&h, c->p.acc, offsetof(Acc, stats), cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < q; ++k) {
        if (D) D[k] = (int64_t)h.dk[k];
        if (n) n[k] = (int64_t)h.nk[k];
    }
    return SW_OK;
}

int sw_get_clock_mirror(sw_ctx *c, int *m)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (c->model != SW_CLOCK) return fail(SW_EINVAL, "not a clock context");
    if (!c->stepped) return fail(SW_ESTATE, "no step since create / sw_set_spins");
    if (m) *m = c->mirror;
    return SW_OK;
}

int sw_get_xy_dir(sw_ctx *c, float *rx, float *ry, float *cr)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (c->model != SW_XY) return fail(SW_EINVAL, "not an XY context");
    if (!c->stepped) return fail(SW_ESTATE, "no step since create / sw_set_spins");
    if (rx) *rx = c->rx;
    if (ry) *ry = c->ry;
    if (cr) *cr = c->crefl;
    return SW_OK;
}

int sw_force_xy_phi(sw_ctx *c, int enable, double phi)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (c->model != SW_XY) return fail(SW_EINVAL, "not an XY context");
    c->force_phi = enable; c->forced_phi = phi;
    return SW_OK;
}

int sw_set_record_bonds(sw_ctx *c, int enable)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    c->record_bonds = enable ? 1 : 0;
    return SW_OK;
}

int sw_set_counting(sw_ctx *c, int enable)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    c->p.counting = enable ? 1 : 0;
    return SW_OK;
}

int sw_get_label_stats(sw_ctx *c, uint64_t *out, int n)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (!out || n < 0) return fail(SW_EINVAL, "sw_get_label_stats: bad buffer");
    unsigned long long h[8];
    SW_CUDA(c, cudaMemcpyAsync(h, c->p.acc->stats, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    SW_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < n && k < 8; ++k) out[k] = h[k];
    return SW_OK;
}

int sw_set_kernel_timing(sw_ctx *c, int enable)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (enable) {
        for (int k = 0; k < 4; ++k)
            if (!c->ev[k]) SW_CUDA(c, cudaEventCreate(&c->ev[k]));
    }
    c->timing = enable ? 1 : 0;
    c->timed_steps = 0;
    for (int k = 0; k < 3; ++k) c->kernel_ms[k] = 0.0;
    return SW_OK;
}

int sw_get_kernel_times(sw_ctx *c, double *ms, int n, uint64_t *steps)
{
    int rc = check_ctx(c);
    if (rc) return rc;
    if (!ms || n < 0) return fail(SW_EINVAL, "sw_get_kernel_times: bad buffer");
    for (int k = 0; k < n && k < 3; ++k) ms[k] = c->kernel_ms[k];
    if (steps) *steps = c->timed_steps;
    c->timed_steps = 0;
    for (int k = 0; k < 3; ++k) c->kernel_ms[k] = 0.0;
    return SW_OK;
}

long long sw_info(const sw_ctx *c, int item)
{
    if (!c) return -1;
    switch (item) {
    case SW_INFO_TILE_X: return c->small ? c->L : c->ops.tx;
    case SW_INFO_TILE_Y: return c->small ? c->L : c->ops.ty;
    case SW_INFO_TILE_Z: return c->small ? (c->dim == 3 ? c->L : 1) : c->ops.tz;
    case SW_INFO_ROWS_PER_THREAD: return c->small ? 1 : c->ops.rows;
    case SW_INFO_FLIP_SITES_PER_THREAD: return c->small ? 32 : (long long)c->ops.tx * c->ops.ty * c->ops.tz / c->ops.nt;
    case SW_INFO_ONE_CTA: return c->small ? 1 : 0;
    case SW_INFO_LAUNCHES_PER_STEP: return c->small ? 0 : 3;
    case SW_INFO_OBSERVABLES_COPY_BYTES: return (long long)offsetof(Acc, stats);
    default: return -1;
    }
}

int sw_micro_bench(int kind, size_t n, size_t table_words, int reps, double *host_ms)
{
    if (!host_ms || reps <= 0 || n == 0 || n > 0xffffff00ull) return fail(SW_EINVAL, "sw_micro_bench: bad arguments");
    if (kind == SW_MICRO_PHILOX_GROUP && (n % (32 * 256)) != 0) return fail(SW_EINVAL, "sw_micro_bench: n must be a multiple of 8192 sites");
    if (kind == SW_MICRO_GATHER && (table_words == 0 || (table_words & (table_words - 1)) != 0 || table_words > 0x80000000ull))
        return fail(SW_EINVAL, "sw_micro_bench: table_words must be a power of two");
    void *out = nullptr, *table = nullptr;
    const size_t out_bytes = kind == SW_MICRO_PHILOX_SITE ? n : (kind == SW_MICRO_PHILOX_GROUP ? n / 32 * 12 : n * 4);
    cudaError_t e = cudaMalloc(&out, out_bytes);
    if (e == cudaSuccess && kind == SW_MICRO_GATHER) {
        e = cudaMalloc(&table, table_words * 4);
        if (e == cudaSuccess) e = cudaMemset(table, 1, table_words * 4);
    }
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    Params p = {};
    p.P32 = 1537996873u; p.k0 = 1u; p.k1 = 0u;   // C4's threshold
    auto launch = [&]() {
        if (kind == SW_MICRO_PHILOX_SITE) k_micro_philox_site<<<(unsigned)((n + 255) / 256), 256>>>((uint8_t *)out, (uint32_t)n, p.P32, p.k0, p.k1);
        else if (kind == SW_MICRO_PHILOX_GROUP) k_micro_philox_group<<<(unsigned)(n / 32 / 256), 256>>>((uint32_t *)out, (uint32_t)(n / 32), p);
        else k_micro_gather<<<(unsigned)((n + 255) / 256), 256>>>((const uint32_t *)table, (uint32_t)(table_words - 1), (uint32_t *)out, (uint32_t)n);
    };
    float ms = 0.f;
    if (e == cudaSuccess) {
        launch();
        e = cudaDeviceSynchronize();
    }
    if (e == cudaSuccess) {
        cudaEventRecord(e0);
        for (int r = 0; r < reps; ++r) launch();
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    cudaFree(table);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SW_ECUDA, std::string("sw_micro_bench: ") + cudaGetErrorString(e)); }
    *host_ms = (double)ms / reps;
    return SW_OK;
}

int sw_philox_selftest(const uint32_t *ctr, const uint32_t *key, uint32_t *out, int count)
{
    if (!ctr || !key || !out || count <= 0) return fail(SW_EINVAL, "sw_philox_selftest: bad arguments");
    uint32_t *d = nullptr;
    const size_t n = (size_t)count;
    SW_CUDA(nullptr, cudaMalloc(&d, n * 10 * sizeof(uint32_t)));
    uint32_t *dc = d, *dk = d + 4 * n, *dout = d + 6 * n;
    cudaError_t e = cudaMemcpy(dc, ctr, n * 16, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, n * 8, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        k_philox_selftest<<<(count + 127) / 128, 128>>>(dc, dk, dout, count);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, n * 16, cudaMemcpyDeviceToHost);
    cudaFree(d);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "sw_philox_selftest");
    return SW_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// sw_cluster_stats_static (include/sw.h): cluster statistics with NO device allocation.  The size
// counters that sw_get_cluster_stats takes from cudaMalloc live in the file-scope device array below
// (SW_STATIC_MAX_SITES counters = 4 MiB, held by every GPU that loads the library until exit).
// In host code the array's name `g_static_sizes` is a host-side stand-in, not a device address: the
// address the kernels get comes from cudaGetSymbolAddress, asked once per device with that device
// current.  Every call shares the array and leaves its counters in it: a call clears the part it uses
// first, and calls that overlap on the GPU (two streams, two threads) race.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) uint32_t g_static_sizes[SW_STATIC_MAX_SITES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
uint32_t *g_static_ptr[STATIC_MAX_DEVICES];   // device address of g_static_sizes on device d, or NULL
std::mutex g_static_mutex;

// counters of this call and the two outputs start at zero
__global__ void __launch_bounds__(256) k_static_clear(uint32_t *sizes, uint32_t n, unsigned long long *out)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i < n) sizes[i] = 0u;
    if (i < 2u) out[i] = 0ull;
}

// the variant of k_cluster_sizes for canonical labels (sw_get_labels: label = a site index of the
// cluster, the same for all its sites): every site adds 1 to the counter of its label
__global__ void __launch_bounds__(256) k_static_cluster_sizes(const uint32_t *__restrict__ labels, uint32_t n, uint32_t *sizes)
{
    const uint32_t i = blockIdx.x * 256u + threadIdx.x;
    if (i >= n) return;
    const uint32_t a = labels[i];
    if (a < n) atomicAdd(&sizes[a], 1u);   // (a label outside the lattice is skipped, never written through)
}

// as k_cluster_moments, with a bound for ragged n
__global__ void __launch_bounds__(256) k_static_cluster_moments(const uint32_t *sizes, uint32_t n, unsigned long long *out)
{
    const uint32_t a = blockIdx.x * 256u + threadIdx.x;
    const unsigned long long c = a < n ? sizes[a] : 0u;
    unsigned long long cnt = c ? 1ull : 0ull, sq = c * c;
    for (int o = 16; o > 0; o >>= 1) {
        cnt += __shfl_down_sync(FULL, cnt, o);
        sq += __shfl_down_sync(FULL, sq, o);
    }
    if ((threadIdx.x & 31) == 0 && cnt) { atomicAdd(&out[0], cnt); atomicAdd(&out[1], sq); }
}

// set-up, once per device, with that device current
int static_scratch(uint32_t **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(SW_ECUDA, "sw_cluster_stats_static: no usable CUDA device (this library has no CPU fallback)"); }
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(SW_EINVAL, "sw_cluster_stats_static: device ordinal out of range");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        uint32_t *q = nullptr;
        e = cudaGetSymbolAddress((void **)&q, g_static_sizes);
        if (e != cudaSuccess || !q) {
            cudaGetLastError();
            return fail(SW_ECUDA, std::string("sw_cluster_stats_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        g_static_ptr[dev] = q;
    }
    *ptr = g_static_ptr[dev];
    return SW_OK;
}

}  // namespace

extern "C" int sw_cluster_stats_static(const uint32_t *device_labels, size_t n, uint64_t *device_out, void *cuda_stream)
{
    if (!device_labels || !device_out) return fail(SW_EINVAL, "sw_cluster_stats_static: NULL pointer");
    if (n == 0 || n > (size_t)SW_STATIC_MAX_SITES)
        return fail(SW_EINVAL, "sw_cluster_stats_static: n must be 1.." + std::to_string((size_t)SW_STATIC_MAX_SITES) +
                               " sites (SW_STATIC_MAX_SITES: the static scratch array holds one counter per site); got " + std::to_string(n));
    uint32_t *sizes = nullptr;
    const int rc = static_scratch(&sizes);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned g = (unsigned)((n + 255) / 256);
    unsigned long long *out = reinterpret_cast<unsigned long long *>(device_out);
    k_static_clear<<<g, 256, 0, st>>>(sizes, (uint32_t)n, out);
    k_static_cluster_sizes<<<g, 256, 0, st>>>(device_labels, (uint32_t)n, sizes);
    k_static_cluster_moments<<<g, 256, 0, st>>>(sizes, (uint32_t)n, out);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "sw_cluster_stats_static");
    return SW_OK;
}
