// lgf_api.cu -- the C ABI of include/lgf.h: context, workspace carving, tables, launch plans,
// CUDA-graph iteration body and the device-resident convergence loop (north_star subsystem (e)).
// Product code (sm_100a); shares nothing with oracle/.  No CPU fallback anywhere: every compute
// entry point launches kernels and reports LGF_ECUDA if that fails.
#include "../../include/lgf.h"

#include <cuda.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "lgf_fft.cuh"
#include "lgf_fft_ct.cuh"
#include "lgf_fft_inst.cuh"
#include "lgf_fft_pipe.cuh"
#include "lgf_fft_pipe_inst.cuh"
#include "lgf_site.cuh"
#include "lgf_site_mu.cuh"
#include "lgf_site_fused.cuh"
#include "lgf_wilson.cuh"
#include "lgf_cluster8.cuh"

using namespace lgf;

namespace {

thread_local char g_last_error[512] = "";

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_last_error, sizeof(g_last_error), "%s: %s", what, cudaGetErrorString(e));
    return LGF_ECUDA;
}
#define CU(call)                                              \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

// Developer A/B knobs (LGF_ZBLOCK, LGF_SITE_TILE, LGF_FUSED, ...; DESIGN.md §6 "A/B knobs") are read only when
// LGF_DEVKNOBS=1 is set: a production process cannot change which kernels run through a stray environment variable.
const char* knob(const char* name) {
    const char* on = getenv("LGF_DEVKNOBS");          // read at every lgf_create (tests switch it per case)
    return (on && atoi(on) != 0) ? getenv(name) : nullptr;
}
bool fused_requested() { const char* e = knob("LGF_FUSED"); return e && atoi(e) != 0; }

constexpr size_t kAlign = 256;
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

// thread-per-site tilings (256 sites each); wider x = longer contiguous runs per link plane
typedef SiteTile<8, 4, 4, 2> Tile0;
typedef SiteTile<16, 4, 2, 2> Tile1;
typedef SiteTile<32, 2, 2, 2> Tile2;
typedef SiteTile<16, 2, 4, 2> Tile3;
typedef SiteTile<32, 4, 2, 1> Tile4;
typedef SiteTile<32, 2, 4, 1> Tile5;
constexpr int kNumSiteTiles = 6;
const int kSiteTileDims[kNumSiteTiles][4] = {{8, 4, 4, 2}, {16, 4, 2, 2}, {32, 2, 2, 2}, {16, 2, 4, 2}, {32, 4, 2, 1}, {32, 2, 4, 1}};
// (site, direction) tilings of k5m: 64 sites x 4 directions
typedef SiteTileMu<8, 4, 2, 1> TileM0;
typedef SiteTileMu<32, 2, 1, 1> TileM1;
typedef SiteTileMu<16, 4, 1, 1> TileM2;
// shared-g K5 (k5s): sites per CTA x 4 directions
typedef SiteTileS<8, 2, 2, 2> TileS0;
typedef SiteTileS<8, 4, 2, 2> TileS1;
typedef SiteTileS<16, 2, 2, 1> TileS2;
typedef SiteTileS<32, 2, 1, 1> TileS3;
typedef SiteTileS<16, 2, 2, 2> TileS4;
constexpr int kNumSTiles = 5;
const int kSTileDims[kNumSTiles][4] = {{8, 2, 2, 2}, {8, 4, 2, 2}, {16, 2, 2, 1}, {32, 2, 1, 1}, {16, 2, 2, 2}};
constexpr int kNumMuTiles = 3;
const int kMuTileDims[kNumMuTiles][4] = {{8, 4, 2, 1}, {32, 2, 1, 1}, {16, 4, 1, 1}};
constexpr int kStageSites = 1 << 15;       // boundary staging chunk (sites)
constexpr int kMaxSmem = 200 * 1024;       // per-CTA dynamic shared memory we are willing to ask for
constexpr int kFixBatch = 8;               // iterations enqueued per polling batch in lgf_fix

bool factor23(int n, Axis* ax) {
    if (n < 2) return false;
    ax->N = n;
    ax->nstages = 0;
    ax->radices = 0;
    int m = n;
    auto push = [&](int r) { ax->radices |= (unsigned long long)r << (4 * ax->nstages); ax->nstages++; };
    while (m % 8 == 0 && ax->nstages < kMaxStages) { push(8); m /= 8; }
    while (m % 4 == 0 && ax->nstages < kMaxStages) { push(4); m /= 4; }
    while (m % 2 == 0 && ax->nstages < kMaxStages) { push(2); m /= 2; }
    while (m % 3 == 0 && ax->nstages < kMaxStages) { push(3); m /= 3; }
    return m == 1;
}

struct Layout {          // byte offsets into the workspace
    size_t state, partials, tw[4], twi[4], psq[4], links, links_bytes, delta, delta2, delta3, staging, staging_bytes, total;
    int nblocks_site;
    int nb[4];
    int nblocks_mu;          // tiling of the (site, direction) kernels
    int nbm[4];
};

bool valid_args(const int32_t L[4], int precision, int storage) {
    if (!L) return false;
    if (precision != LGF_F32 && precision != LGF_F64) return false;
    if (storage != LGF_REAL18 && storage != LGF_REAL12) return false;
    long long V = 1;
    for (int i = 0; i < 4; ++i) {
        if (L[i] < 2 || L[i] > 4096) return false;
        V *= L[i];
    }
    return V < (1ll << 31);      // the site kernels index sites with 32-bit integers
}

Layout make_layout(const int32_t L[4], int precision, int storage, bool fused, int nbatch = 1) {
    Layout lo;
    const size_t w = precision == LGF_F64 ? 8 : 4;
    const size_t V = (size_t)L[0] * L[1] * L[2] * L[3];
    size_t nb = 0;                 // most CTAs any thread-per-site tiling needs (sizes the partials)
    for (int t = 0; t < kNumSiteTiles; ++t) {
        size_t n = 1;
        for (int i = 0; i < 4; ++i) n *= (size_t)((L[i] + kSiteTileDims[t][i] - 1) / kSiteTileDims[t][i]);
        if (n > nb) nb = n;
    }
    for (int t = 0; t < kNumSTiles; ++t) {     // the (site, direction) tilings have fewer sites per CTA
        size_t n = 1;
        for (int i = 0; i < 4; ++i) n *= (size_t)((L[i] + kSTileDims[t][i] - 1) / kSTileDims[t][i]);
        if (n > nb) nb = n;
    }
    for (int i = 0; i < 4; ++i) lo.nb[i] = 0;
    lo.nblocks_site = 0;           // set by choose_site_tile()
    for (int i = 0; i < 4; ++i) lo.nbm[i] = 0;
    lo.nblocks_mu = 0;             // set at create
    size_t off = 0;
    const size_t B = (size_t)nbatch;      // every per-lattice region holds the B lattices of a batched context back to back
    lo.state = off; off += align_up(B * sizeof(DevState));
    lo.partials = off; off += align_up(B * nb * sizeof(double2));
    for (int i = 0; i < 4; ++i) { lo.tw[i] = off; off += align_up((size_t)L[i] * 2 * w); }
    for (int i = 0; i < 4; ++i) { lo.twi[i] = off; off += align_up((size_t)L[i] * 2 * w); }
    for (int i = 0; i < 4; ++i) { lo.psq[i] = off; off += align_up((size_t)L[i] * w); }
    // the fused update kernel (opt-in) writes the new field out of place into a second link buffer (DevState::cur)
    lo.links_bytes = align_up(B * 4 * (size_t)(storage / 2) * V * 2 * w);
    lo.links = off; off += (fused ? 2 : 1) * lo.links_bytes;
    lo.delta = off; off += align_up(B * 4 * V * 2 * w);
    // layout-B spectrum between K2 and K3 (pipelined FFT path): tiles padded by one z entry per t row
    lo.delta2 = off; off += align_up(B * 4 * (V / L[2]) * (size_t)(L[2] + 1) * 2 * w);
    lo.delta3 = off; off += fused ? align_up(B * 4 * V * 2 * w) : 0;   // Delta of the new links (fused path: K1/K51 out, K2 in)
    const size_t stage_sites = V < (size_t)kStageSites ? V : (size_t)kStageSites;
    lo.staging_bytes = align_up(stage_sites * 36 * 2 * w);          // two buffers: the copy of one chunk runs beside the transpose of the other
    lo.staging = off; off += 2 * lo.staging_bytes;
    lo.total = off;
    return lo;
}

}  // namespace

struct lgf_ctx {
    int32_t L[4];
    int precision, storage;
    int nbatch;                  // lattices per launch (1 unless created by lgf_create_batch)
    long long V;
    size_t wbytes;               // bytes per real
    char* ws;                    // device workspace
    bool owns_ws;
    cudaStream_t stream;
    cudaStream_t cap_stream;     // library-owned stream used only to CAPTURE graphs (the legacy default stream cannot be captured)
    Layout lo;
    Geom geom;
    Geom geom_mu;                // tiling of the (site, direction) kernels
    int site_variant;            // 0: thread per (site, direction); 1: thread per site
    int site_tile;               // index into kSiteTileDims for the thread-per-site kernels
    int mu_tile;                 // index into kMuTileDims for k5m
    int s_tile;                  // index into kSTileDims for k5s (site_variant 2)
    Geom geom_s;
    int nblocks_s;
    Axis axis[4];
    XyPass xy;                   // K2, K4
    ZtPass zt;                   // K3
    int xy_threads, zt_threads;
    size_t xy_smem, zt_smem;
    // compile-time-sized fast path (nullptr: generic kernels above)
    const XyCtEntry* xy_ct;
    const ZtCtEntry* zt_ct;
    XyArgs xy_args;
    ZtArgs zt_args;
    // pipelined fast path (lgf_fft_pipe.cuh); both set or both null
    const XyPipeEntry* xy_pipe;
    const XyPipeEntry* xy_pipe_inv;      // K4's entry (same line splits as K2's, possibly another tile shape)
    int xyp_inv_grid;
    const ZtPipeEntry* zt_pipe;
    XyPipeArgs xyp_args;
    int xyp_grid, ztp_grid;
    alignas(64) CUtensorMap zt_omap;     // fft_zt_pipe3q's output tensor (Delta~, natural layout), stored through the TMA unit
    alignas(64) CUtensorMap xy_bmap;     // fft_xy_pipe_io's output tensor (the layout-B spectrum)
    alignas(64) CUtensorMap xy_imap;     // fft_xy_inv3's input tensor (Delta~ as planes, box one pad column wider than a plane)
    // fused K5+K1 marching kernel (lgf_site_fused.cuh); -1: not used
    int fused_tile;
    MarchGeom mgeom;
    int fused_grid;
    bool cluster8;               // 8^4 (one cluster per lattice of a batched context): lgf_iterate / lgf_fix run k_cluster8_iterate (lgf_cluster8.cuh) instead of the graph
    int cur_host;                // host mirror of DevState::cur
    bool dbg_delta_tilde;        // lgf_debug_get_delta source: Delta~ (after debug_fourier_accelerate) or Delta
    bool loaded, delta_valid;
    int64_t launches;
    // iteration graph (K2 K3 K4 K5 K1), captured per alpha
    cudaGraphExec_t graph;
    double graph_alpha;
    int launches_per_iter;
    // pinned host mirror of DevState (two slots for the lgf_fix polling pipeline)
    DevState* host_state;
    cudaEvent_t ev[2];
    int64_t pending_n;           // lgf_iterate_async bookkeeping (-1: nothing pending)
    // programmatic dependent launch: set while the iteration body is captured, so that every kernel after the
    // first becomes a programmatic edge of the graph (its CTAs are scheduled while the previous kernel drains
    // and block in griddepcontrol.wait, see pdl_entry()); LGF_PDL=0 turns it off
    // deferred k1_finish: the end-of-iteration reduction runs on a second graph branch beside the next iteration's
    // K2 (which is then not gated by `done`: it only writes the spectrum buffer) and once after the last iteration
    // of a batch; LGF_DEFER_FINISH=0 puts it back behind K1
    bool defer_finish;
    cudaStream_t fin_stream;
    // lgf_load / lgf_store from / to HOST memory: the PCIe copies run on io_stream beside the layout transposes on the context's
    // stream, through two staging buffers (io_copied[b]: the copy into / out of buffer b is done; io_moved[b]: its transpose is)
    cudaStream_t io_stream;
    cudaEvent_t io_start, io_copied[2], io_moved[2];
    cudaEvent_t ev_fork, ev_join;
    bool pdl_enabled, pdl;
    int pdl_mask, pdl_idx;       // which launches of the body (bit i: i-th launch) carry the attribute
};

namespace {

// kernel launches of the iteration body (typed, and through the instantiation tables' untyped pointers)
cudaLaunchConfig_t launch_config(lgf_ctx* c, dim3 grid, dim3 block, size_t smem, cudaLaunchAttribute* at) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c->stream;
    at->id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at->val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = (c->pdl && ((c->pdl_mask >> c->pdl_idx) & 1)) ? 1 : 0;
    c->pdl_idx++;
    return cfg;
}
template <typename... KArgs, typename... Args>
cudaError_t launch_ex(lgf_ctx* c, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
    cudaLaunchAttribute at;
    const cudaLaunchConfig_t cfg = launch_config(c, grid, block, smem, &at);
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
cudaError_t launch_exc(lgf_ctx* c, const void* kernel, dim3 grid, dim3 block, void** args, size_t smem) {
    cudaLaunchAttribute at;
    const cudaLaunchConfig_t cfg = launch_config(c, grid, block, smem, &at);
    return cudaLaunchKernelExC(&cfg, kernel, args);
}

// grid of the site kernels: (x tiles, y tiles, z tiles * t tiles); see split_zt()
// (lattice b of a batched context: blockIdx.z = b * nzt + (z,t) tile)
dim3 grid3(const Geom& g, int nbatch) { return dim3((unsigned)g.nb[0], (unsigned)g.nb[1], (unsigned)(g.nb[2] * g.nb[3] * nbatch)); }
unsigned magic_of(int d) { return d > 1 ? (unsigned)((0x100000000ULL + (unsigned)d - 1) / (unsigned)d) : 0u; }
// walk order of the site kernels' (z, t) tiles (Geom::zb): z-blocks of about 16 MB of link traffic per t step once
// a whole t-slice of links no longer fits the L2 comfortably (LGF_ZBLOCK overrides: z-tiles per block, 0 = plain order)
void set_walk(Geom& g, int tz, size_t link_bytes_per_site, size_t slice_limit = (size_t)48 << 20) {
    const size_t per_ztile = (size_t)g.L[0] * g.L[1] * tz * link_bytes_per_site;
    int zb = g.nb[2];
    if (per_ztile * (size_t)g.nb[2] > slice_limit) {
        zb = (int)(((size_t)16 << 20) / per_ztile);
        if (zb < 1) zb = 1;
    }
    const char* e = knob("LGF_ZBLOCK");
    if (e) zb = atoi(e) > 0 ? atoi(e) : g.nb[2];
    if (zb > g.nb[2]) zb = g.nb[2];
    while (g.nb[2] % zb) --zb;
    g.zb = zb;
    g.zb_magic = magic_of(zb);
    g.nb3_magic = magic_of(g.nb[3]);
    g.nzt = g.nb[2] * g.nb[3];
    g.nzt_magic = magic_of(g.nzt);
    g.nblocks = g.nb[0] * g.nb[1] * g.nzt;
}

DevState* dev_state(lgf_ctx* c) { return reinterpret_cast<DevState*>(c->ws + c->lo.state); }

// (one thread per lattice of a batched context)
__global__ void reset_cur_kernel(DevState* st) { st[threadIdx.x].cur = 0; }
__global__ void init_state_kernel(DevState* st, double tol, long long max_iter) {
    st += threadIdx.x;
    st->iter = 0;
    st->done = 0;
    st->ticket = 0;
    st->pending = 0;
    st->tol = tol;
    st->max_iter = max_iter;
}
// after the initial measurement of lgf_fix: already converged (or max_iter == 0)?
__global__ void initial_test_kernel(DevState* st) {
    st += threadIdx.x;
    if (st->theta < st->tol || st->max_iter <= 0) st->done = 1;
}

// ---- FFT pass planning -------------------------------------------------------------------------
int threads_for(long long elems, const Axis& a, const Axis& b) {
    long long need = 32;
    const Axis* axes[2] = {&a, &b};
    for (int i = 0; i < 2; ++i)
        for (int s = 0; s < axes[i]->nstages; ++s) {
            const int R = int((axes[i]->radices >> (4 * s)) & 15ull);
            const int per_thread = R * (kElemsPerThread / R);
            const long long t = (elems + per_thread - 1) / per_thread;
            if (t > need) need = t;
        }
    need = (need + 31) / 32 * 32;
    return need > 4096 ? 4096 : (int)need;
}

// returns false if a transform tile cannot be held on chip
bool plan_passes(lgf_ctx* c) {
    const int* L = c->L;
    const size_t cb = 2 * c->wbytes;   // bytes per complex
    const int max_threads = c->precision == LGF_F64 ? 512 : 1024;
    for (int i = 0; i < 4; ++i) {
        if (!factor23(L[i], &c->axis[i])) return false;
        c->axis[i].tw_fwd = c->ws + c->lo.tw[i];
        c->axis[i].tw_inv = c->ws + c->lo.twi[i];
        c->axis[i].psq = c->ws + c->lo.psq[i];
    }
    const long long LxLy = (long long)L[0] * L[1], LzLt = (long long)L[2] * L[3];
    // K2 / K4
    c->xy.ax = c->axis[0];
    c->xy.ay = c->axis[1];
    c->xy.pitch = L[0] + 1;
    c->xy_threads = threads_for(LxLy, c->axis[0], c->axis[1]);
    c->xy_smem = (size_t)c->xy.pitch * L[1] * cb;
    if (c->xy_threads > max_threads || c->xy_smem > (size_t)kMaxSmem) return false;
    // K3: largest chunk of contiguous sites whose (z,t) plane fits (prefer <= 64 KB for occupancy)
    int best = 0;
    const size_t budgets[2] = {(size_t)64 * 1024, (size_t)kMaxSmem};
    for (int pass = 0; pass < 2 && !best; ++pass)
        for (int cx = 16; cx >= 1; cx /= 2) {
            if (LxLy % cx) continue;
            const size_t bytes = (size_t)cx * (L[2] + 1) * L[3] * cb;
            if (bytes <= budgets[pass] && threads_for(cx * LzLt, c->axis[2], c->axis[3]) <= max_threads) { best = cx; break; }
        }
    if (!best) return false;
    ZtPass& Z = c->zt;
    Z.az = c->axis[2];
    Z.at = c->axis[3];
    Z.cx = best;
    Z.pz = best;
    Z.pt = best * (L[2] + 1);
    Z.gz = LxLy;
    Z.gt = LxLy * L[2];
    Z.tiles_per_comp = (int)(LxLy / best);
    Z.Lx = L[0];
    Z.psq_x = c->axis[0].psq;
    Z.psq_y = c->axis[1].psq;
    double pmax = 0;
    for (int i = 0; i < 4; ++i) {
        const long double s = sinl(3.141592653589793238462643383279502884L * (long double)(L[i] / 2) / (long double)L[i]);
        pmax += (double)(4.0L * s * s);
    }
    Z.scale_num = pmax / (double)c->V;
    c->zt_threads = threads_for(best * LzLt, c->axis[2], c->axis[3]);
    c->zt_smem = (size_t)Z.pt * L[3] * cb;
    // fast path: both passes must be available, because K2's compile-time kernels leave the (x,y)
    // spectrum in digit-swapped order, which only the compile-time K3 knows how to un-swap
    c->zt_ct = find_zt_ct(c->precision, L[2], L[3], LxLy);
    c->xy_ct = c->zt_ct ? find_xy_ct(c->precision, L[0], L[1]) : nullptr;
    c->zt_pipe = find_zt_pipe(c->precision, L[2], L[3], LxLy);
    c->xy_pipe = c->zt_pipe ? find_xy_pipe(c->precision, L[0], L[1]) : nullptr;
    if (!c->xy_pipe) c->zt_pipe = nullptr;
    c->xy_pipe_inv = c->xy_pipe ? find_xy_pipe_inv(c->precision, L[0], L[1], c->xy_pipe) : nullptr;
    {   // LGF_FFT_PIPE=0: fall back to the one-tile-per-CTA kernels (A/B knob)
        const char* e = knob("LGF_FFT_PIPE");
        if (e && atoi(e) == 0) c->xy_pipe = nullptr, c->zt_pipe = nullptr;
    }
    if (knob("LGF_FORCE_GENERIC_FFT")) c->xy_ct = nullptr, c->zt_ct = nullptr, c->xy_pipe = nullptr, c->zt_pipe = nullptr;
    if (c->xy_ct) {
        c->xy_args.twx_fwd = c->axis[0].tw_fwd; c->xy_args.twx_inv = c->axis[0].tw_inv;
        c->xy_args.twy_fwd = c->axis[1].tw_fwd; c->xy_args.twy_inv = c->axis[1].tw_inv;
        c->xy_args.nplanes = (int)(4 * LzLt * c->nbatch);
    }
    if (c->xy_pipe) {
        XyPipeArgs& P = c->xyp_args;
        P.twx_fwd = c->axis[0].tw_fwd; P.twx_inv = c->axis[0].tw_inv;
        P.twy_fwd = c->axis[1].tw_fwd; P.twy_inv = c->axis[1].tw_inv;
        P.nplanes = (int)(4 * LzLt * c->nbatch);
        P.planes_per_comp = (int)LzLt;
        P.nz = L[2];
        P.pt = c->zt_pipe->cx * (L[2] + 1);
        P.tile_elems = P.pt * L[3];
        int sh = 0;
        while ((1 << sh) < c->zt_pipe->cx) ++sh;
        P.cxb_shift = sh;
        P.chunks_per_comp = (int)(LxLy >> sh);
        P.perm_c = c->zt_pipe->perm_c;
        P.perm_d = c->zt_pipe->perm_d;
        P.perm_lq = c->zt_pipe->tstore == 1 ? c->zt_pipe->perm_d / 4 : c->zt_pipe->perm_d;
        // K2 stores a plane as boxes of `store_tiles` layout-B tiles x CX sites (a tensor-map box extent is at most 256)
        int st = P.chunks_per_comp < 256 ? P.chunks_per_comp : 256;
        while (P.chunks_per_comp % st) --st;
        P.store_tiles = st;
        P.nstores = P.chunks_per_comp / st;
    }
    if (c->zt_ct || c->zt_pipe) {
        ZtArgs& A = c->zt_args;
        A.twz_fwd = c->axis[2].tw_fwd; A.twz_inv = c->axis[2].tw_inv;
        A.twt_fwd = c->axis[3].tw_fwd; A.twt_inv = c->axis[3].tw_inv;
        A.psq_x = c->axis[0].psq; A.psq_y = c->axis[1].psq; A.psq_z = c->axis[2].psq; A.psq_t = c->axis[3].psq;
        A.V = c->V;
        A.nbatch = c->nbatch;
        A.LxLy = LxLy;
        A.Lx = L[0];
        A.tiles_per_comp = (int)(LxLy / (c->zt_pipe ? c->zt_pipe->cx : c->zt_ct->cx));
        A.scale_num = Z.scale_num;
        A.x_n1 = c->xy_pipe ? c->xy_pipe->x_n1 : (c->xy_ct ? c->xy_ct->x_n1 : L[0]);
        A.x_n2 = L[0] / A.x_n1;
        A.y_n1 = c->xy_pipe ? c->xy_pipe->y_n1 : (c->xy_ct ? c->xy_ct->y_n1 : L[1]);
        A.y_n2 = L[1] / A.y_n1;
    }
    return true;
}

// The host-only part of lgf_create's planning, so that lgf_workspace_bytes and lgf_create agree on what is supported:
// does every transform tile of this lattice fit in shared memory / the thread limit?
bool tiles_fit(const int32_t L[4], int precision) {
    lgf_ctx* t = new (std::nothrow) lgf_ctx();
    if (!t) return false;
    memset(static_cast<void*>(t), 0, sizeof(*t));
    for (int i = 0; i < 4; ++i) t->L[i] = L[i];
    t->precision = precision;
    t->V = (long long)L[0] * L[1] * L[2] * L[3];
    t->wbytes = precision == LGF_F64 ? 8 : 4;
    t->nbatch = 1;
    const bool ok = plan_passes(t);
    delete t;
    return ok;
}

typedef CUresult (*TensorMapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                      const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int encode_map(lgf_ctx* c, CUtensorMap* map, int rank, void* base, const cuuint64_t* dims, const cuuint64_t* strides,
               const cuuint32_t* box) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CU(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return cuda_fail(cudaErrorNotSupported, "cuTensorMapEncodeTiled entry point");
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUresult r = reinterpret_cast<TensorMapEncodeFn>(fn)(
        map, c->precision == LGF_F64 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, (cuuint32_t)rank, base,
        dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_last_error, sizeof(g_last_error), "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return LGF_ECUDA;
    }
    return LGF_OK;
}
// The tensor maps of the kernels of the pipelined FFT path that store through the TMA unit.  Element = one real; a
// complex number is two elements, so every box starts and ends on whole sites.
//   fft_zt_pipe3q (K3, quarter tiles): the natural-layout Delta~ field D[c][t][z][y][x] as the 5-D tensor
//   (2 xy, z, t mod D, t div D, c), box (2 CX, Nz + 1, D/4, C, 1).  The (Nz+1)-th z entry of a box -- the pad of the
//   shared-memory rows -- falls outside the tensor and is clipped by the hardware.
//   fft_xy_pipe_io (K2): layout B, D'[c][tile][row][z + pad][j], as the 4-D tensor (2 j, z, row, c * tiles + tile),
//   box (2 CX, 1, 1, store_tiles).
int make_pipe_maps(lgf_ctx* c) {
    const ZtPipeEntry* e = c->zt_pipe;
    if (!e || !c->xy_pipe) return LGF_OK;
    const cuuint64_t cb = 2 * c->wbytes, LxLy = (cuuint64_t)c->L[0] * c->L[1], Nz = c->L[2], Nt = c->L[3];
    if (e->tstore == 1) {
        const cuuint64_t C = e->perm_c, D = e->perm_d;
        const cuuint64_t dims[5] = {2 * LxLy, Nz, D, C, (cuuint64_t)(4 * c->nbatch)};
        const cuuint64_t strides[4] = {LxLy * cb, LxLy * Nz * cb, D * LxLy * Nz * cb, (cuuint64_t)c->V * cb};
        const cuuint32_t box[5] = {(cuuint32_t)(2 * e->cx), (cuuint32_t)(Nz + 1), (cuuint32_t)(D / 4), (cuuint32_t)C, 1};
        const int rc = encode_map(c, &c->zt_omap, 5, c->ws + c->lo.delta, dims, strides, box);
        if (rc) return rc;
    }
    if (c->xy_pipe_inv && c->xy_pipe_inv->inv3) {
        // Delta~ (natural layout) as (2 reals x Nx, Ny, planes); the box is 1 (fp64) / 2 (fp32) columns wider than the plane:
        // the out-of-range columns are zero-filled and give the shared-memory rows a conflict-free pitch
        const XyPipeEntry* x = c->xy_pipe_inv;
        const cuuint64_t nx = c->L[0], ny = c->L[1], pad = c->precision == LGF_F64 ? 1 : 2;
        const cuuint64_t dims[3] = {2 * nx, ny, (cuuint64_t)c->xyp_args.nplanes};
        const cuuint64_t strides[2] = {nx * cb, nx * ny * cb};
        const cuuint32_t box[3] = {(cuuint32_t)(2 * (nx + pad)), (cuuint32_t)ny, (cuuint32_t)x->pb};
        const int rc = encode_map(c, &c->xy_imap, 3, c->ws + c->lo.delta, dims, strides, box);
        if (rc) return rc;
    }
    if (c->xy_pipe->io) {
        const XyPipeArgs& P = c->xyp_args;
        const cuuint64_t dims[4] = {(cuuint64_t)(2 * e->cx), Nz + 1, Nt, (cuuint64_t)(4 * c->nbatch) * P.chunks_per_comp};
        const cuuint64_t strides[3] = {(cuuint64_t)e->cx * cb, (cuuint64_t)P.pt * cb, (cuuint64_t)P.tile_elems * cb};
        const cuuint32_t box[4] = {(cuuint32_t)(2 * e->cx), 1, 1, (cuuint32_t)P.store_tiles};
        return encode_map(c, &c->xy_bmap, 4, c->ws + c->lo.delta2, dims, strides, box);
    }
    return LGF_OK;
}

template <typename T>
int upload_tables(lgf_ctx* c) {
    for (int mu = 0; mu < 4; ++mu) {
        const int n = c->L[mu];
        std::vector<Cx<T>> tw(n), twi(n);
        std::vector<T> psq(n);
        for (int j = 0; j < n; ++j) {
            // exact octant reduction is not needed at these sizes: long double keeps ~1e-19
            const long double ang = 2.0L * 3.141592653589793238462643383279502884L * (long double)j / (long double)n;
            tw[j] = Cx<T>((T)cosl(ang), (T)(-sinl(ang)));
            twi[j] = Cx<T>((T)cosl(ang), (T)(sinl(ang)));
            const long double s = sinl(3.141592653589793238462643383279502884L * (long double)j / (long double)n);
            psq[j] = (T)(4.0L * s * s);
        }
        for (int j = n / 2 + 1; j < n; ++j) psq[j] = psq[n - j];     // exactly even in k (K3 relies on it)
        if (mu == 3 && n <= 64)
            for (int j = 0; j <= n / 2; ++j) {
                if (sizeof(T) == 8) c->zt_args.psq_t_half_d[j] = (double)psq[j];
                else c->zt_args.psq_t_half_f[j] = (float)psq[j];
            }
        CU(cudaMemcpyAsync(c->ws + c->lo.tw[mu], tw.data(), n * sizeof(Cx<T>), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->ws + c->lo.twi[mu], twi.data(), n * sizeof(Cx<T>), cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(c->ws + c->lo.psq[mu], psq.data(), n * sizeof(T), cudaMemcpyHostToDevice, c->stream));
        CU(cudaStreamSynchronize(c->stream));   // the host vectors die at the end of this scope
    }
    return LGF_OK;
}

// ---- typed launchers ---------------------------------------------------------------------------
template <typename T, int NC>
struct Impl {
    static Cx<T>* links_buf(lgf_ctx* c, int which) { return reinterpret_cast<Cx<T>*>(c->ws + c->lo.links + (size_t)which * c->lo.links_bytes); }
    static Cx<T>* links(lgf_ctx* c) { return links_buf(c, c->cur_host); }     // the current field, as the host knows it
    static Cx<T>* delta(lgf_ctx* c) { return reinterpret_cast<Cx<T>*>(c->ws + c->lo.delta); }      // Delta~ (natural)
    // where K1 / K51 write Delta of the current links and K2 reads it
    static Cx<T>* delta_src(lgf_ctx* c) { return reinterpret_cast<Cx<T>*>(c->ws + (c->fused_tile >= 0 ? c->lo.delta3 : c->lo.delta)); }
    static Cx<T>* staging(lgf_ctx* c, int which = 0) { return reinterpret_cast<Cx<T>*>(c->ws + c->lo.staging + (size_t)which * c->lo.staging_bytes); }

    static int k1(lgf_ctx* c, int mode, bool with_finish = true) {
        double2* partials = reinterpret_cast<double2*>(c->ws + c->lo.partials);
#define LGF_K1_CASE(ID, TILE) case ID: launch_ex(c, k1_delta_theta_F<T, NC, TILE>, grid3(c->geom, c->nbatch), dim3(TILE::kThreads), 0, \
            links(c), delta_src(c), partials, dev_state(c), c->geom, mode); break;
        switch (c->site_tile) {
            LGF_K1_CASE(1, Tile1) LGF_K1_CASE(4, Tile4)
#ifdef LGF_DEV_VARIANTS
            LGF_K1_CASE(2, Tile2) LGF_K1_CASE(3, Tile3) LGF_K1_CASE(5, Tile5)
#endif
            default: launch_ex(c, k1_delta_theta_F<T, NC, Tile0>, grid3(c->geom, c->nbatch), dim3(Tile0::kThreads), 0,
                links(c), delta_src(c), partials, dev_state(c), c->geom, mode);
        }
#undef LGF_K1_CASE
        CU(cudaGetLastError());
        c->launches++;
        return with_finish ? k1_reduce(c, mode) : LGF_OK;
    }
    // k1_finish on the context's stream (mode 3: deferred, see lgf_ctx::defer_finish)
    static int k1_reduce(lgf_ctx* c, int mode) {
        double2* partials = reinterpret_cast<double2*>(c->ws + c->lo.partials);
        launch_ex(c, k1_finish, dim3(c->nbatch), dim3(kFinishThreads), 0, partials, c->lo.nblocks_site, dev_state(c), (double)c->V, mode);
        c->launches++;
        CU(cudaGetLastError());
        return LGF_OK;
    }
    // fused K5 + K1: update out of place, emit Delta/theta/F of the new links, swap the link buffers
    static int k51(lgf_ctx* c, double alpha) {
        double2* partials = reinterpret_cast<double2*>(c->ws + c->lo.partials);
        const Cx<T>* u0 = links_buf(c, 0);
        const Cx<T>* u1 = links_buf(c, 1);
        const Cx<T>* dt = delta(c);
        Cx<T>* dout = delta_src(c);
        const DevState* st = dev_state(c);
        T ha = (T)(0.5 * alpha);
        void* args[] = {&u0, &u1, &dt, &dout, &partials, &st, &c->mgeom, &ha};
        const FusedEntry& e = fused_entries()[c->fused_tile];
        CU(launch_exc(c, e.kernel, dim3(c->fused_grid), dim3(e.threads), args, e.smem));
        launch_ex(c, k1_finish, dim3(1), dim3(kFinishThreads), 0, partials, c->fused_grid, dev_state(c), (double)c->V, 2);
        c->launches += 2;
        CU(cudaGetLastError());
        return LGF_OK;
    }
    struct FusedEntry { int tx, ty, tz, threads; size_t smem; const void* kernel; };
    template <class Tile, int MINB> static FusedEntry fused_entry() {
        return FusedEntry{Tile::TX, Tile::TY, Tile::TZ, Tile::NS, Tile::template smem_bytes<T, NC>(),
                          (const void*)&k51_update_delta<T, NC, Tile, MINB>};
    }
    static const FusedEntry* fused_entries() {
        static const FusedEntry tab[] = {
            fused_entry<MarchTile<32, 4, 2>, 2>(),
            fused_entry<MarchTile<64, 2, 2>, 2>(),
            fused_entry<MarchTile<48, 4, 1>, 2>(),
            fused_entry<MarchTile<16, 4, 4>, 2>(),
            fused_entry<MarchTile<8, 8, 4>, 2>(),
#ifdef LGF_DEV_VARIANTS      // measured and rejected: not in the default build
            fused_entry<MarchTile<32, 4, 4>, 1>(),
            fused_entry<MarchTile<48, 4, 2>, 1>(),
            fused_entry<MarchTile<64, 4, 2>, 1>(),
            fused_entry<MarchTile<32, 4, 2, true>, 1>(),
#endif
        };
        return tab;
    }
#ifdef LGF_DEV_VARIANTS
    static constexpr int kNumFused = 9;
#else
    static constexpr int kNumFused = 5;
#endif
    // pick the marching tile for this lattice (LGF_FUSED = 0 disables the fused path, LGF_FUSED_TILE = i forces entry i)
    static int plan_fused(lgf_ctx* c) {
        c->fused_tile = -1;
        if (!c->xy_pipe || c->nbatch > 1) return LGF_OK;   // the fused path rides on the pipelined FFT buffers; single lattices only
        if (!fused_requested()) return LGF_OK;             // opt-in (LGF_DEVKNOBS=1 LGF_FUSED=1) until it beats K5 + K1 everywhere
        const char* ft = knob("LGF_FUSED_TILE");
        const FusedEntry* tab = fused_entries();
        for (int i = 0; i < kNumFused; ++i) {
            if (ft && atoi(ft) != i) continue;
            if (tab[i].tx != c->L[0] || c->L[1] % tab[i].ty || c->L[2] % tab[i].tz) continue;
            if (tab[i].smem > (size_t)227 * 1024) continue;     // e.g. the staged tile in fp64 18-real
            c->fused_tile = i;
            break;
        }
        if (c->fused_tile < 0) return LGF_OK;
        const FusedEntry& fe = tab[c->fused_tile];
        CU(cudaFuncSetAttribute(fe.kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fe.smem));
        int dev = 0, sms = 0, occ = 0;
        CU(cudaGetDevice(&dev));
        CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fe.kernel, fe.threads, fe.smem));
        if (occ < 1) { c->fused_tile = -1; return LGF_OK; }
        MarchGeom& m = c->mgeom;
        for (int i = 0; i < 4; ++i) m.L[i] = c->L[i];
        m.V = c->V;
        m.nby = c->L[1] / fe.ty;
        m.nbz = c->L[2] / fe.tz;
        m.nslices = (long long)m.nby * m.nbz * c->L[3];
        long long grid = (long long)occ * sms;
        if (grid > m.nslices) grid = m.nslices;
        c->fused_grid = (int)grid;
        return LGF_OK;
    }
    static int k5(lgf_ctx* c, double alpha) {
        if (c->site_variant == 2) {
            // resident CTAs per SM the 256-thread k5s tiles are compiled for (LGF_K5S_OCC overrides at build time)
#ifdef LGF_K5S_OCC
            constexpr int kS3 = LGF_K5S_OCC;
#else
            constexpr int kS3 = sizeof(T) == 8 ? 3 : 4;
#endif
#define LGF_K5S_CASE(ID, TILE, MINB) case ID: launch_ex(c, k5s_gbuild_update<T, NC, TILE, MINB>, grid3(c->geom_s, c->nbatch), dim3(TILE::kThreads), 0,  \
                links(c), delta(c), dev_state(c), c->geom_s, (T)(0.5 * alpha)); break;
            switch (c->s_tile) {
                LGF_K5S_CASE(1, TileS1, 1) LGF_K5S_CASE(2, TileS2, kS3) LGF_K5S_CASE(3, TileS3, kS3) LGF_K5S_CASE(4, TileS4, 1)
                default: launch_ex(c, k5s_gbuild_update<T, NC, TileS0, 2>, grid3(c->geom_s, c->nbatch), dim3(TileS0::kThreads), 0, 
                    links(c), delta(c), dev_state(c), c->geom_s, (T)(0.5 * alpha));
            }
#undef LGF_K5S_CASE
            c->launches++;
            CU(cudaGetLastError());
            return LGF_OK;
        }
        if (c->site_variant == 0) {
#define LGF_K5M_CASE(ID, TILE) case ID: launch_ex(c, k5m_gbuild_update<T, NC, TILE>, grid3(c->geom_mu, c->nbatch), dim3(TILE::kThreads), 0,  \
                links(c), delta(c), dev_state(c), c->geom_mu, (T)(0.5 * alpha)); break;
            switch (c->mu_tile) {
                LGF_K5M_CASE(1, TileM1) LGF_K5M_CASE(2, TileM2)
                default: launch_ex(c, k5m_gbuild_update<T, NC, TileM0>, grid3(c->geom_mu, c->nbatch), dim3(TileM0::kThreads), 0, 
                    links(c), delta(c), dev_state(c), c->geom_mu, (T)(0.5 * alpha));
            }
#undef LGF_K5M_CASE
            c->launches++;
            CU(cudaGetLastError());
            return LGF_OK;
        }
#define LGF_K5_CASE(ID, TILE) case ID: launch_ex(c, k5_gbuild_update<T, NC, TILE>, grid3(c->geom, c->nbatch), dim3(TILE::kThreads), 0,  \
            links(c), delta(c), dev_state(c), c->geom, (T)(0.5 * alpha)); break;
        switch (c->site_tile) {
            LGF_K5_CASE(1, Tile1) LGF_K5_CASE(4, Tile4)
#ifdef LGF_DEV_VARIANTS
            LGF_K5_CASE(2, Tile2) LGF_K5_CASE(3, Tile3) LGF_K5_CASE(5, Tile5)
#endif
            default: launch_ex(c, k5_gbuild_update<T, NC, Tile0>, grid3(c->geom, c->nbatch), dim3(Tile0::kThreads), 0, 
                links(c), delta(c), dev_state(c), c->geom, (T)(0.5 * alpha));
        }
#undef LGF_K5_CASE
        c->launches++;
        CU(cudaGetLastError());
        return LGF_OK;
    }
    static int fft(lgf_ctx* c, int k, bool gated) {
        // (batched contexts: the per-lattice `done` flags gate K5 and K1; the FFT passes run ungated)
        const int* done = (gated && c->nbatch == 1) ? &dev_state(c)->done : nullptr;
        const unsigned planes = (unsigned)(4 * (long long)c->L[2] * c->L[3] * c->nbatch);
        Cx<T>* dptr = delta(c);
        if (c->xy_pipe) {
            Cx<T>* d2 = reinterpret_cast<Cx<T>*>(c->ws + c->lo.delta2);
            if (k == 1) {
                const ZtPipeEntry* e = c->zt_pipe;
                void* args[] = {&d2, &dptr, &c->zt_args, &done, &c->zt_omap};          // layout B -> natural (fifth: fft_zt_pipe3q only)
                CU(launch_exc(c, e->kernel, dim3(c->ztp_grid), dim3(e->threads), args, e->smem));
            } else {
                const XyPipeEntry* e = k == 0 ? c->xy_pipe : c->xy_pipe_inv;
                Cx<T>* inp = k == 0 ? delta_src(c) : dptr;                 // K2 reads Delta where K1 / K51 left it
                Cx<T>* outp = k == 0 ? d2 : dptr;                          // K2: natural -> layout B; K4: in place
                void* tmap = (k == 2 && e->inv3) ? (void*)&c->xy_imap : (void*)&c->xy_bmap;      // fifth: fft_xy_inv3 / fft_xy_pipe_io only
                void* args[] = {&inp, &outp, &c->xyp_args, &done, tmap};
                CU(launch_exc(c, k == 0 ? e->k_fwd : e->k_inv, dim3(k == 0 ? c->xyp_grid : c->xyp_inv_grid), dim3(e->threads), args, e->smem));
            }
            c->launches++;
            return LGF_OK;
        }
        if (k != 1 && c->xy_ct) {
            const XyCtEntry* e = c->xy_ct;
            void* args[] = {&dptr, &c->xy_args, &done};
            CU(launch_exc(c, k == 0 ? e->k_fwd : e->k_inv, dim3((planes + e->pb - 1) / e->pb), dim3(e->threads), args, e->smem));
            c->launches++;
            return LGF_OK;
        }
        if (k == 1 && c->zt_ct) {
            const ZtCtEntry* e = c->zt_ct;
            void* args[] = {&dptr, &c->zt_args, &done};
            CU(launch_exc(c, e->kernel, dim3(4 * c->nbatch * c->zt_args.tiles_per_comp), dim3(e->threads), args, e->smem));
            c->launches++;
            return LGF_OK;
        }
        if (k == 0)
            launch_ex(c, fft_xy_kernel<T, -1>, dim3(planes), dim3(c->xy_threads), c->xy_smem, delta(c), c->xy, done);
        else if (k == 2)
            launch_ex(c, fft_xy_kernel<T, +1>, dim3(planes), dim3(c->xy_threads), c->xy_smem, delta(c), c->xy, done);
        else
            launch_ex(c, fft_zt_kernel<T>, dim3(4 * c->nbatch * c->zt.tiles_per_comp), dim3(c->zt_threads), c->zt_smem, delta(c), c->zt, c->V, done);
        c->launches++;
        CU(cudaGetLastError());
        return LGF_OK;
    }
    static int setup(lgf_ctx* c) {
        CU(cudaFuncSetAttribute(fft_xy_kernel<T, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
        CU(cudaFuncSetAttribute(fft_xy_kernel<T, +1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
        CU(cudaFuncSetAttribute(fft_zt_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMaxSmem));
        CU(prepare_ct_kernels(c->precision));
        CU(prepare_pipe_kernels(c->precision));
        if (c->xy_pipe) {   // persistent grids: one CTA per SM (or fewer when there are fewer tiles)
            int dev = 0, sms = 0, occ = 0;
            CU(cudaGetDevice(&dev));
            CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            const int xy_tiles = (c->xyp_args.nplanes + c->xy_pipe->pb - 1) / c->xy_pipe->pb;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->xy_pipe->k_fwd, c->xy_pipe->threads, c->xy_pipe->smem));
            if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources, "fft_xy_pipe does not fit on an SM");
            c->xyp_grid = xy_tiles < occ * sms ? xy_tiles : occ * sms;
            const int inv_tiles = (c->xyp_args.nplanes + c->xy_pipe_inv->pb - 1) / c->xy_pipe_inv->pb;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->xy_pipe_inv->k_inv, c->xy_pipe_inv->threads, c->xy_pipe_inv->smem));
            if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources, "fft_xy_pipe (inverse) does not fit on an SM");
            c->xyp_inv_grid = inv_tiles < occ * sms ? inv_tiles : occ * sms;
            const int zt_tiles = 4 * c->nbatch * c->zt_args.tiles_per_comp;
            CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, c->zt_pipe->kernel, c->zt_pipe->threads, c->zt_pipe->smem));
            if (occ < 1) return cuda_fail(cudaErrorLaunchOutOfResources, "fft_zt_pipe does not fit on an SM");
            c->ztp_grid = zt_tiles < occ * sms ? zt_tiles : occ * sms;
        }
        {
            const int rc = plan_fused(c);
            if (rc) return rc;
        }
        {
            const int rc = make_pipe_maps(c);
            if (rc) return rc;
        }
        {
            const int rc = cluster8_setup(c);
            if (rc) return rc;
        }
        return upload_tables<T>(c);
    }
    // The single-cluster path (lgf_cluster8.cuh) serves 8^4 lattices (one cluster each); LGF_CLUSTER=0 (developer knob) keeps the graph path.
    static int cluster8_setup(lgf_ctx* c) {
        c->cluster8 = false;
        const char* off = knob("LGF_CLUSTER");
        if (c->fused_tile >= 0 || (off && atoi(off) == 0)) return LGF_OK;
        // batched contexts: the B200 hosts 7 fp64 clusters at a time (14 in fp32, two CTAs per SM), a wave of them costs one
        // lattice's 10 us; past two waves in fp64 the batched launch graph (1.47 us per lattice-iteration) is as fast
        if (c->precision == LGF_F64 && c->nbatch > 14) return LGF_OK;
        for (int mu = 0; mu < 4; ++mu)
            if (c->L[mu] != 8) return LGF_OK;
        const void* k = (const void*)&k_cluster8_iterate<T, NC>;
        CU(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cl8<T, NC>::kSmem));
        CU(cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = Cl8<T, NC>::kCtas; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(Cl8<T, NC>::kCtas); cfg.blockDim = dim3(Cl8<T, NC>::kThreads);
        cfg.dynamicSmemBytes = Cl8<T, NC>::kSmem; cfg.attrs = attr; cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, k, &cfg) != cudaSuccess || nclusters < 1) {
            cudaGetLastError();                // a device that cannot host the 16-CTA cluster keeps the five-kernel graph
            return LGF_OK;
        }
        c->cluster8 = true;
        return LGF_OK;
    }
    // all iterations of one lgf_iterate / lgf_fix call: the kernel reads tol, max_iter and iter from DevState
    static int cluster8_run(lgf_ctx* c, double alpha) {
        Cluster8Args a;
        a.psq = c->ws + c->lo.psq[0];
        a.scale_num = c->zt_args.scale_num;
        a.half_alpha = 0.5 * alpha;
        Cx<T>* U = links(c);
        Cx<T>* D = delta_src(c);
        DevState* st = dev_state(c);
        void* args[] = {&U, &D, &st, &a};
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = Cl8<T, NC>::kCtas; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.gridDim = dim3(Cl8<T, NC>::kCtas * c->nbatch); cfg.blockDim = dim3(Cl8<T, NC>::kThreads);
        cfg.dynamicSmemBytes = Cl8<T, NC>::kSmem; cfg.stream = c->stream; cfg.attrs = attr; cfg.numAttrs = 1;
        CU(cudaLaunchKernelExC(&cfg, (const void*)&k_cluster8_iterate<T, NC>, args));
        c->launches++;
        return LGF_OK;
    }
    static int load(lgf_ctx* c, const void* src, int memspace) {
        const long long V = c->V;
        const int thr = 256;
        c->cur_host = 0;                                   // a fresh field always lands in buffer 0
        reset_cur_kernel<<<1, c->nbatch, 0, c->stream>>>(dev_state(c));
        c->launches++;
        CU(cudaGetLastError());
        int k = 0;                                         // staging chunks so far (all lattices of a batched context)
        if (memspace != LGF_DEVICE) {
            CU(cudaEventRecord(c->io_start, c->stream));   // whatever produced `src` on this stream comes first
            CU(cudaStreamWaitEvent(c->io_stream, c->io_start, 0));
        }
        for (int b = 0; b < c->nbatch; ++b) {             // the lattices of a batched context lie back to back, here and there
            Cx<T>* Ub = links(c) + (size_t)b * 4 * NC * V;
            const Cx<T>* sb = reinterpret_cast<const Cx<T>*>(src) + (size_t)b * V * 36;
            if (memspace == LGF_DEVICE) {
                const long long n = V * 36;
                aos_to_soa<T, NC><<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(sb, Ub, V, 0, V);
                c->launches++;
                CU(cudaGetLastError());
            } else {
                // chunk k is copied into staging buffer k % 2 on io_stream while chunk k - 1 is transposed on the context's stream
                for (long long s0 = 0; s0 < V; s0 += kStageSites, ++k) {
                    const long long ns = (V - s0 < kStageSites) ? V - s0 : kStageSites;
                    const int buf = k & 1;
                    if (k >= 2) CU(cudaStreamWaitEvent(c->io_stream, c->io_moved[buf], 0));      // its previous contents are consumed
                    CU(cudaMemcpyAsync(staging(c, buf), sb + (size_t)s0 * 36, (size_t)ns * 36 * sizeof(Cx<T>), cudaMemcpyHostToDevice, c->io_stream));
                    CU(cudaEventRecord(c->io_copied[buf], c->io_stream));
                    CU(cudaStreamWaitEvent(c->stream, c->io_copied[buf], 0));
                    const long long n = ns * 36;
                    aos_to_soa<T, NC><<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(staging(c, buf), Ub, V, s0, ns);
                    c->launches++;
                    CU(cudaGetLastError());
                    CU(cudaEventRecord(c->io_moved[buf], c->stream));
                }
            }
        }
        CU(cudaStreamSynchronize(c->stream));
        return LGF_OK;
    }
    static int store(lgf_ctx* c, void* dst, int memspace) {
        const long long V = c->V;
        const int thr = 256;
        int k = 0;                                         // staging chunks so far (all lattices of a batched context)
        for (int b = 0; b < c->nbatch; ++b) {
            const Cx<T>* Ub = links(c) + (size_t)b * 4 * NC * V;
            Cx<T>* db = reinterpret_cast<Cx<T>*>(dst) + (size_t)b * V * 36;
            if (memspace == LGF_DEVICE) {
                const long long n = V * 4;
                soa_to_aos<T, NC><<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(Ub, db, V, 0, V);
                c->launches++;
                CU(cudaGetLastError());
            } else {
                // chunk k is transposed into staging buffer k % 2 on the context's stream while chunk k - 1 leaves on io_stream
                for (long long s0 = 0; s0 < V; s0 += kStageSites, ++k) {
                    const long long ns = (V - s0 < kStageSites) ? V - s0 : kStageSites;
                    const long long n = ns * 4;
                    const int buf = k & 1;
                    if (k >= 2) CU(cudaStreamWaitEvent(c->stream, c->io_copied[buf], 0));        // its previous contents have left
                    soa_to_aos<T, NC><<<(unsigned)((n + thr - 1) / thr), thr, 0, c->stream>>>(Ub, staging(c, buf), V, s0, ns);
                    c->launches++;
                    CU(cudaGetLastError());
                    CU(cudaEventRecord(c->io_moved[buf], c->stream));
                    CU(cudaStreamWaitEvent(c->io_stream, c->io_moved[buf], 0));
                    CU(cudaMemcpyAsync(db + (size_t)s0 * 36, staging(c, buf), (size_t)ns * 36 * sizeof(Cx<T>), cudaMemcpyDeviceToHost, c->io_stream));
                    CU(cudaEventRecord(c->io_copied[buf], c->io_stream));
                }
            }
        }
        if (memspace != LGF_DEVICE) CU(cudaStreamSynchronize(c->io_stream));
        CU(cudaStreamSynchronize(c->stream));
        return LGF_OK;
    }
    // ---- the step after the path: temporal Wilson lines and the singlet correlator (lgf_wilson.cuh) ----
    // scratch: the two Delta-sized fields (>= 8 V complex >= 11 Vs for Lt >= 2): W (9 Vs), P (Vs), G (Vs)
    static Cx<T>* scratch(lgf_ctx* c) { return reinterpret_cast<Cx<T>*>(c->ws + c->lo.delta); }
    static int lines(lgf_ctx* c) {
        const long long Vs = c->V / c->L[3];
        const int thr = 128;
        k_wilson_lines<T, NC><<<(unsigned)((Vs + thr - 1) / thr), thr, 0, c->stream>>>(links(c), scratch(c), c->V, Vs, c->L[3]);
        c->launches++;
        CU(cudaGetLastError());
        return LGF_OK;
    }
    static int wilson_lines_out(lgf_ctx* c, void* dst, int memspace) {
        const long long Vs = c->V / c->L[3];
        int rc = lines(c);
        if (rc) return rc;
        Cx<T>* aos = memspace == LGF_DEVICE ? reinterpret_cast<Cx<T>*>(dst) : scratch(c) + (size_t)9 * Vs;
        k_lines_to_aos<T><<<(unsigned)((Vs * 9 + 255) / 256), 256, 0, c->stream>>>(scratch(c), aos, Vs);
        c->launches++;
        CU(cudaGetLastError());
        if (memspace == LGF_HOST) CU(cudaMemcpyAsync(dst, aos, (size_t)9 * Vs * sizeof(Cx<T>), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        return LGF_OK;
    }
    static int correlator(lgf_ctx* c, void* dst, int memspace) {
        const long long Vs = c->V / c->L[3], LxLy = (long long)c->L[0] * c->L[1];
        const int Lz = c->L[2], thr = 128;
        int rc = lines(c);
        if (rc) return rc;
        Cx<T>* W = scratch(c);
        Cx<T>* P = W + (size_t)9 * Vs;
        Cx<T>* G = P + (size_t)Vs;
        const int* nodone = nullptr;
        launch_ex(c, fft_xy_kernel<T, -1>, dim3((unsigned)(9 * Lz)), dim3(c->xy_threads), c->xy_smem, W, c->xy, nodone);
        const Cx<T>* twz = reinterpret_cast<const Cx<T>*>(c->axis[2].tw_fwd);
        const Cx<T>* twzi = reinterpret_cast<const Cx<T>*>(c->axis[2].tw_inv);
        k_z_power<T><<<(unsigned)((Vs + thr - 1) / thr), thr, 0, c->stream>>>(W, P, twz, LxLy, Lz);
        k_z_inverse<T><<<(unsigned)((Vs + thr - 1) / thr), thr, 0, c->stream>>>(P, G, twzi, LxLy, Lz);
        launch_ex(c, fft_xy_kernel<T, +1>, dim3((unsigned)Lz), dim3(c->xy_threads), c->xy_smem, G, c->xy, nodone);
        Cx<T>* out = memspace == LGF_DEVICE ? reinterpret_cast<Cx<T>*>(dst) : P;
        const T scale = (T)(1.0 / (3.0 * (double)Vs * (double)Vs));
        k_corr_scale<T><<<(unsigned)((Vs + 255) / 256), 256, 0, c->stream>>>(G, out, Vs, scale);
        c->launches += 5;
        CU(cudaGetLastError());
        if (memspace == LGF_HOST) CU(cudaMemcpyAsync(dst, out, (size_t)Vs * sizeof(Cx<T>), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        return LGF_OK;
    }
    static int get_delta(lgf_ctx* c, void* dst, int memspace) {
        const long long V = c->V;
        const int thr = 256;
        Cx<T>* srcp = c->dbg_delta_tilde ? delta(c) : delta_src(c);
        if (memspace == LGF_DEVICE) {
            delta_to_aos<T><<<(unsigned)((V * 4 + thr - 1) / thr), thr, 0, c->stream>>>(srcp, reinterpret_cast<Cx<T>*>(dst), V);
            c->launches++;
            CU(cudaGetLastError());
            CU(cudaStreamSynchronize(c->stream));
            return LGF_OK;
        }
        // host: copy the four component planes and interleave on the host side of the copy
        std::vector<Cx<T>> tmp((size_t)4 * V);
        CU(cudaMemcpyAsync(tmp.data(), srcp, (size_t)4 * V * sizeof(Cx<T>), cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        Cx<T>* out = reinterpret_cast<Cx<T>*>(dst);
        for (long long s = 0; s < V; ++s)
            for (int k = 0; k < 4; ++k) out[s * 4 + k] = tmp[(size_t)k * V + s];
        return LGF_OK;
    }
};

#define DISPATCH(c, CALL)                                                     \
    ((c)->precision == LGF_F64                                                \
         ? ((c)->storage == LGF_REAL18 ? Impl<double, 9>::CALL : Impl<double, 6>::CALL) \
         : ((c)->storage == LGF_REAL18 ? Impl<float, 9>::CALL : Impl<float, 6>::CALL))

int enqueue_iteration_body(lgf_ctx* c, double alpha) {
    int rc;
    c->pdl = false;                 // the first kernel of the graph has no predecessor to overlap with
    c->pdl_idx = 0;
    // only with the pipelined FFT path, whose K2 is out of place: an ungated in-place K2 (generic / one-tile-per-CTA
    // kernels) would overwrite Delta in the no-op iterations that follow the crossing inside a batch
    const bool defer = c->defer_finish && c->fused_tile < 0 && c->xy_pipe != nullptr;
    if (defer) {
        // second branch: fold the previous iteration's partials into theta / F / iter / done while K2 runs
        cudaStream_t main_stream = c->stream;
        CU(cudaEventRecord(c->ev_fork, main_stream));
        CU(cudaStreamWaitEvent(c->fin_stream, c->ev_fork, 0));
        c->stream = c->fin_stream;
        rc = DISPATCH(c, k1_reduce(c, 3));
        c->stream = main_stream;
        if (rc) return rc;
        CU(cudaEventRecord(c->ev_join, c->fin_stream));
        c->pdl_idx = 0;
    }
    if ((rc = DISPATCH(c, fft(c, 0, !defer)))) return rc;
    if (defer) CU(cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &cs) == cudaSuccess && cs == cudaStreamCaptureStatusActive) c->pdl = c->pdl_enabled;
    if ((rc = DISPATCH(c, fft(c, 1, true)))) return rc;
    if ((rc = DISPATCH(c, fft(c, 2, true)))) return rc;
    if (c->fused_tile >= 0) return DISPATCH(c, k51(c, alpha));
    if ((rc = DISPATCH(c, k5(c, alpha)))) return rc;
    if ((rc = DISPATCH(c, k1(c, 1, !defer)))) return rc;
    return LGF_OK;
}

// (Re)capture the iteration body into a CUDA graph for this alpha.
int ensure_graph(lgf_ctx* c, double alpha) {
    if (c->graph && c->graph_alpha == alpha) return LGF_OK;
    if (c->graph) { cudaGraphExecDestroy(c->graph); c->graph = nullptr; }
    const int64_t before = c->launches;
    CU(cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    cudaStream_t user = c->stream;
    c->stream = c->cap_stream;
    const int rc = enqueue_iteration_body(c, alpha);
    c->stream = user;
    c->pdl = false;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    c->launches_per_iter = (int)(c->launches - before);
    c->launches = before;   // capture launches nothing
    if (rc) { if (g) cudaGraphDestroy(g); return rc; }
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamEndCapture");
    e = cudaGraphInstantiate(&c->graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { c->graph = nullptr; return cuda_fail(e, "cudaGraphInstantiate"); }
    c->graph_alpha = alpha;
    return LGF_OK;
}

int enqueue_iterations(lgf_ctx* c, int64_t n) {
    for (int64_t i = 0; i < n; ++i) {
        CU(cudaGraphLaunch(c->graph, c->stream));
        c->launches += c->launches_per_iter;
    }
    if (n > 0 && c->defer_finish && c->fused_tile < 0 && c->xy_pipe != nullptr) return DISPATCH(c, k1_reduce(c, 3));   // the last iteration's
    return LGF_OK;
}

int init_state(lgf_ctx* c, double tol, long long max_iter) {
    init_state_kernel<<<1, c->nbatch, 0, c->stream>>>(dev_state(c), tol, max_iter);
    c->launches++;
    CU(cudaGetLastError());
    return LGF_OK;
}

int fetch_state(lgf_ctx* c, int slot) {
    CU(cudaMemcpyAsync(&c->host_state[(size_t)slot * c->nbatch], dev_state(c), (size_t)c->nbatch * sizeof(DevState), cudaMemcpyDeviceToHost, c->stream));
    return LGF_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

const char* lgf_version(void) { return "0.1"; }
const char* lgf_last_error(void) { return g_last_error; }

const char* lgf_strerror(int code) {
    switch (code) {
        case LGF_OK: return "ok";
        case LGF_EINVAL: return "invalid argument";
        case LGF_EUNSUPPORTED: return "unsupported lattice (extent not 2^a 3^b, or transform tile exceeds shared memory)";
        case LGF_ESTATE: return "no links loaded, or lgf_iterate_async pending (call lgf_wait first)";
        case LGF_ECUDA: return "CUDA error (see lgf_last_error)";
        case LGF_ENOMEM: return "host allocation failed";
        default: return "unknown error";
    }
}

size_t lgf_workspace_bytes(const int32_t L[4], int precision, int storage) {
    if (!valid_args(L, precision, storage)) return 0;
    Axis ax;
    for (int i = 0; i < 4; ++i)
        if (!factor23(L[i], &ax)) return 0;
    if (!tiles_fit(L, precision)) return 0;
    return make_layout(L, precision, storage, fused_requested()).total;
}

static int create_common(const int32_t L[4], int precision, int storage, int nbatch, void* ws, size_t ws_bytes, bool owns,
                         void* stream, lgf_ctx** out) {
    lgf_ctx* c = new (std::nothrow) lgf_ctx();
    if (!c) return LGF_ENOMEM;
    memset(static_cast<void*>(c), 0, sizeof(*c));
    for (int i = 0; i < 4; ++i) c->L[i] = L[i];
    c->precision = precision;
    c->storage = storage;
    c->nbatch = nbatch;
    c->V = (long long)L[0] * L[1] * L[2] * L[3];
    c->wbytes = precision == LGF_F64 ? 8 : 4;
    c->ws = reinterpret_cast<char*>(ws);
    c->owns_ws = owns;
    c->stream = reinterpret_cast<cudaStream_t>(stream);
    c->lo = make_layout(L, precision, storage, fused_requested() && nbatch == 1, nbatch);
    c->pending_n = -1;
    {
        const char* e = knob("LGF_PDL");
        // measured: 8^4 22.6 -> 20.5 us per iteration, 16^4 32.8 -> 32.0 us, but 32^4 fp64-12 315 -> 381 us
        // with every edge programmatic (no single edge gains more than 1.5 us there), so: launch-bound lattices only
        c->pdl_enabled = e ? atoi(e) != 0 : c->V <= 65536;
        e = knob("LGF_PDL_MASK");
        c->pdl_mask = e ? atoi(e) : 0x3e;
    }
    {   // thread-per-site tiling: widest x tile that divides Lx (LGF_SITE_TILE overrides, A/B knob)
        int t = (L[0] % 32 == 0) ? 4 : ((L[0] % 16 == 0) ? 1 : 0);
        const char* e = knob("LGF_SITE_TILE");
#ifdef LGF_DEV_VARIANTS
        if (e && atoi(e) >= 0 && atoi(e) < kNumSiteTiles) t = atoi(e);
#else
        if (e && (atoi(e) == 0 || atoi(e) == 1 || atoi(e) == 4)) t = atoi(e);      // tiles 2, 3, 5: -DLGF_DEV_VARIANTS builds only
#endif
        c->site_tile = t;
        int n = 1;
        for (int i = 0; i < 4; ++i) { c->lo.nb[i] = (L[i] + kSiteTileDims[t][i] - 1) / kSiteTileDims[t][i]; n *= c->lo.nb[i]; }
        c->lo.nblocks_site = n;
    }
    for (int i = 0; i < 4; ++i) { c->geom.L[i] = L[i]; c->geom.nb[i] = c->lo.nb[i]; }
    // (K1 reads what K5 reads and writes: half the bytes per site, so half the limit; 48^3 x 8 fp64 is then blocked
    // in both kernels: 293.1 -> 289.8 us 12-real, 360.7 -> 355.2 us 18-real)
    set_walk(c->geom, kSiteTileDims[c->site_tile][2], (size_t)4 * storage * c->wbytes, (size_t)24 << 20);
    c->geom.V = c->V;
    {   // K5 flavour: 0 = thread per (site, direction), 1 = thread per site (LGF_SITE_VARIANT / LGF_SITEMU_TILE: A/B knobs)
        const char* e = knob("LGF_SITE_VARIANT");
        // measured at 32^4: the (site, direction) split wins for fp64 18-real and fp32 12-real
        // measured at 32^4: the shared-g (site, direction) kernel k5s wins for fp64 18-real (233 vs 247 us) and
        // fp32 12-real (102 vs 107 us); thread-per-site wins for fp64 12-real (175 vs 194 us) and fp32 18-real
        c->site_variant = e ? atoi(e) : 2;
        int t = (L[0] % 16 == 0) ? 2 : 0;
        e = knob("LGF_SITEMU_TILE");
        if (e && atoi(e) >= 0 && atoi(e) < kNumMuTiles) t = atoi(e);
        c->mu_tile = t;
        int n = 1;
        for (int i = 0; i < 4; ++i) { c->lo.nbm[i] = (L[i] + kMuTileDims[t][i] - 1) / kMuTileDims[t][i]; n *= c->lo.nbm[i]; }
        c->lo.nblocks_mu = n;
    }
    c->geom_mu = c->geom;
    for (int i = 0; i < 4; ++i) c->geom_mu.nb[i] = c->lo.nbm[i];
    set_walk(c->geom_mu, kMuTileDims[c->mu_tile][2], (size_t)8 * storage * c->wbytes);
    const int mu_default_fallback = ((precision == LGF_F64 && storage == LGF_REAL18) || (precision == LGF_F32 && storage == LGF_REAL12)) ? 0 : 1;
    {   // shared-g K5 (LGF_SITE_VARIANT=2, LGF_SITES_TILE): needs every extent to be a multiple of the tile's
        const char* e = knob("LGF_SITES_TILE");
        int t = (e && atoi(e) >= 0 && atoi(e) < kNumSTiles) ? atoi(e) : (precision == LGF_F64 ? 2 : 3);
        auto divides = [&](int tile) {
            for (int k = 0; k < 4; ++k)
                if (L[k] % kSTileDims[tile][k]) return false;
            return true;
        };
        // default tile does not divide the lattice (fp32 at Lx = 48: 32 x 2 x 1 x 1): 16 x 2 x 2 x 1 next (48^3 x 8 fp32: K5 84.0 -> 81.6 us),
        // then the smallest one
        if (!e && !divides(t)) t = divides(2) ? 2 : 0;
        c->s_tile = t;
        c->geom_s = c->geom;
        int n = 1;
        bool ok = true;
        for (int i = 0; i < 4; ++i) {
            ok = ok && (L[i] % kSTileDims[t][i] == 0);
            c->geom_s.nb[i] = L[i] / kSTileDims[t][i];
            n *= c->geom_s.nb[i] > 0 ? c->geom_s.nb[i] : 1;
        }
        c->nblocks_s = n;
        set_walk(c->geom_s, kSTileDims[t][2], (size_t)8 * storage * c->wbytes);
        if (c->site_variant == 2 && !ok) c->site_variant = mu_default_fallback;

    }
    int rc = LGF_OK;
    if (ws_bytes < c->lo.total || (reinterpret_cast<uintptr_t>(ws) % kAlign) != 0) rc = LGF_EINVAL;
    if (!rc && !plan_passes(c)) rc = LGF_EUNSUPPORTED;
    if (!rc) {
        cudaError_t e = cudaMallocHost(reinterpret_cast<void**>(&c->host_state), 2 * (size_t)nbatch * sizeof(DevState));
        if (e != cudaSuccess) rc = cuda_fail(e, "cudaMallocHost");
    }
    if (!rc) {
        cudaError_t e = cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) rc = cuda_fail(e, "cudaStreamCreateWithFlags");
    }
    if (!rc) {
        const char* e = knob("LGF_DEFER_FINISH");
        c->defer_finish = !(e && atoi(e) == 0);
        cudaError_t ce = cudaStreamCreateWithFlags(&c->fin_stream, cudaStreamNonBlocking);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming);
        if (ce != cudaSuccess) rc = cuda_fail(ce, "deferred-finish stream/events");
    }
    if (!rc) {
        cudaError_t ce = cudaStreamCreateWithFlags(&c->io_stream, cudaStreamNonBlocking);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&c->io_start, cudaEventDisableTiming);
        for (int i = 0; i < 2 && ce == cudaSuccess; ++i) {
            ce = cudaEventCreateWithFlags(&c->io_copied[i], cudaEventDisableTiming);
            if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&c->io_moved[i], cudaEventDisableTiming);
        }
        if (ce != cudaSuccess) rc = cuda_fail(ce, "boundary copy stream/events");
    }
    for (int i = 0; i < 2 && !rc; ++i) {
        cudaError_t e = cudaEventCreateWithFlags(&c->ev[i], cudaEventDisableTiming);
        if (e != cudaSuccess) rc = cuda_fail(e, "cudaEventCreate");
    }
    if (!rc) rc = DISPATCH(c, setup(c));
    if (!rc) rc = init_state(c, -1.0, 0);
    if (!rc) {
        cudaError_t e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) rc = cuda_fail(e, "cudaStreamSynchronize");
    }
    if (rc) {
        c->owns_ws = false;   // the caller of create_common frees on failure
        lgf_destroy(c);
        return rc;
    }
    *out = c;
    return LGF_OK;
}

int lgf_create(const int32_t L[4], int precision, int storage, void* workspace_dev, size_t workspace_bytes,
               void* cuda_stream, lgf_ctx** out) {
    if (!out || !workspace_dev || !valid_args(L, precision, storage)) return LGF_EINVAL;
    if (lgf_workspace_bytes(L, precision, storage) == 0) return LGF_EUNSUPPORTED;
    return create_common(L, precision, storage, 1, workspace_dev, workspace_bytes, false, cuda_stream, out);
}

static bool valid_batch(const int32_t L[4], int nbatch) {
    // grid z = (z,t) tiles x lattices must stay below 2^16 for every site-kernel tiling (the smallest tile is 2 x 1 in z, t)
    return nbatch >= 1 && (long long)nbatch * ((L[2] + 1) / 2) * L[3] <= 65535;
}

size_t lgf_workspace_bytes_batch(const int32_t L[4], int precision, int storage, int32_t nbatch) {
    if (!valid_args(L, precision, storage) || !valid_batch(L, nbatch)) return 0;
    Axis ax;
    for (int i = 0; i < 4; ++i)
        if (!factor23(L[i], &ax)) return 0;
    if (!tiles_fit(L, precision)) return 0;
    return make_layout(L, precision, storage, fused_requested() && nbatch == 1, nbatch).total;
}

int lgf_create_batch(const int32_t L[4], int precision, int storage, int32_t nbatch, void* workspace_dev, size_t workspace_bytes,
                     void* cuda_stream, lgf_ctx** out) {
    if (!out || !workspace_dev || !valid_args(L, precision, storage) || nbatch < 1) return LGF_EINVAL;
    if (lgf_workspace_bytes_batch(L, precision, storage, nbatch) == 0) return LGF_EUNSUPPORTED;
    return create_common(L, precision, storage, nbatch, workspace_dev, workspace_bytes, false, cuda_stream, out);
}

int32_t lgf_batch_size(const lgf_ctx* c) { return c ? c->nbatch : 0; }

int lgf_create_simple(const int32_t L[4], int precision, int storage, lgf_ctx** out) {
    if (!out || !valid_args(L, precision, storage)) return LGF_EINVAL;
    const size_t bytes = lgf_workspace_bytes(L, precision, storage);
    if (bytes == 0) return LGF_EUNSUPPORTED;
    void* ws = nullptr;
    CU(cudaMalloc(&ws, bytes));
    const int rc = create_common(L, precision, storage, 1, ws, bytes, true, nullptr, out);
    if (rc) cudaFree(ws);
    return rc;
}

int lgf_destroy(lgf_ctx* c) {
    if (!c) return LGF_EINVAL;
    if (c->stream || c->ws) cudaStreamSynchronize(c->stream);
    if (c->graph) cudaGraphExecDestroy(c->graph);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    if (c->fin_stream) cudaStreamDestroy(c->fin_stream);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->io_stream) { cudaStreamSynchronize(c->io_stream); cudaStreamDestroy(c->io_stream); }
    if (c->io_start) cudaEventDestroy(c->io_start);
    for (int i = 0; i < 2; ++i) {
        if (c->io_copied[i]) cudaEventDestroy(c->io_copied[i]);
        if (c->io_moved[i]) cudaEventDestroy(c->io_moved[i]);
    }
    for (int i = 0; i < 2; ++i)
        if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    if (c->host_state) cudaFreeHost(c->host_state);
    if (c->owns_ws && c->ws) cudaFree(c->ws);
    delete c;
    return LGF_OK;
}

// between lgf_iterate_async and lgf_wait the device owns the context's state: every other entry point refuses
#define LGF_NOT_PENDING(c) do { if ((c)->pending_n >= 0) return LGF_ESTATE; } while (0)

int lgf_load(lgf_ctx* c, const void* links, int memspace) {
    if (!c || !links || (memspace != LGF_HOST && memspace != LGF_DEVICE)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    const int rc = DISPATCH(c, load(c, links, memspace));
    if (rc) return rc;
    c->loaded = true;
    c->delta_valid = false;
    return LGF_OK;
}

int lgf_store(lgf_ctx* c, void* links, int memspace) {
    if (!c || !links || (memspace != LGF_HOST && memspace != LGF_DEVICE)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    return DISPATCH(c, store(c, links, memspace));
}

static int finish(lgf_ctx* c, lgf_result* out, bool fix_mode) {
    int rc = fetch_state(c, 0);
    if (rc) return rc;
    CU(cudaStreamSynchronize(c->stream));
    c->cur_host = c->host_state[0].cur;
    for (int b = 0; out && b < c->nbatch; ++b) {           // one result per lattice of a batched context
        const DevState& s = c->host_state[b];
        out[b].iterations = s.iter;
        out[b].theta = s.theta;
        out[b].F = s.F;
        out[b].converged = fix_mode ? (s.theta < s.tol ? 1 : 0) : 0;
    }
    return LGF_OK;
}

int lgf_measure(lgf_ctx* c, lgf_result* out) {
    if (!c || !out) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    int rc = init_state(c, -1.0, 0);
    if (!rc) rc = DISPATCH(c, k1(c, 0));
    if (rc) return rc;
    c->delta_valid = true;
    c->dbg_delta_tilde = false;
    std::vector<lgf_result> r((size_t)c->nbatch);
    rc = finish(c, r.data(), false);
    if (rc) return rc;
    for (int b = 0; b < c->nbatch; ++b) { r[b].iterations = 0; out[b] = r[b]; }
    return LGF_OK;
}

int lgf_iterate_async(lgf_ctx* c, int64_t n, double alpha) {
    if (!c || n < 0 || !(alpha > 0)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    if (c->cluster8) {                 // one launch: measure, then n updates with the field resident in the cluster's shared memory
        int rc8 = init_state(c, -1.0, (long long)n);
        if (!rc8) rc8 = DISPATCH(c, cluster8_run(c, alpha));
        if (rc8) return rc8;
        c->delta_valid = true;
        c->dbg_delta_tilde = false;
        c->pending_n = n;
        return LGF_OK;
    }
    int rc = ensure_graph(c, alpha);
    if (!rc) rc = init_state(c, -1.0, (long long)n);
    if (!rc && (!c->delta_valid || n == 0)) rc = DISPATCH(c, k1(c, 0));
    if (!rc) { c->delta_valid = true; c->dbg_delta_tilde = false; rc = enqueue_iterations(c, n); }
    if (rc) return rc;
    c->pending_n = n;
    return LGF_OK;
}

int lgf_wait(lgf_ctx* c, lgf_result* out) {
    if (!c) return LGF_EINVAL;
    if (c->pending_n < 0) return LGF_ESTATE;
    std::vector<lgf_result> r((size_t)c->nbatch);
    const int rc = finish(c, r.data(), false);
    c->pending_n = -1;
    if (rc) return rc;
    for (int b = 0; out && b < c->nbatch; ++b) out[b] = r[b];
    return LGF_OK;
}

int lgf_iterate(lgf_ctx* c, int64_t n, double alpha, lgf_result* out) {
    if (!out) return LGF_EINVAL;
    const int rc = lgf_iterate_async(c, n, alpha);
    if (rc) return rc;
    return lgf_wait(c, out);
}

int lgf_fix(lgf_ctx* c, double alpha, double theta_tol, int64_t max_iter, lgf_result* out) {
    if (!c || !out || !(alpha > 0) || max_iter < 0 || !(theta_tol == theta_tol)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    if (c->cluster8) {                 // the whole convergence loop is one launch (stopping test on the device, every iteration)
        int rc8 = init_state(c, theta_tol, (long long)max_iter);
        if (!rc8) rc8 = DISPATCH(c, cluster8_run(c, alpha));
        if (rc8) return rc8;
        c->delta_valid = true;
        c->dbg_delta_tilde = false;
        std::vector<lgf_result> r8((size_t)c->nbatch);
        rc8 = finish(c, r8.data(), true);
        if (rc8) return rc8;
        for (int b = 0; b < c->nbatch; ++b) out[b] = r8[b];
        return LGF_OK;
    }
    int rc = ensure_graph(c, alpha);
    if (!rc) rc = init_state(c, theta_tol, (long long)max_iter);
    if (!rc) rc = DISPATCH(c, k1(c, 0));
    if (rc) return rc;
    c->delta_valid = true;
    c->dbg_delta_tilde = false;
    initial_test_kernel<<<1, c->nbatch, 0, c->stream>>>(dev_state(c));
    c->launches++;
    CU(cudaGetLastError());
    // Batches of kFixBatch gated iterations; the state block is copied to pinned memory after each
    // batch.  The host keeps one batch in flight ahead of the one it polls, so the GPU never idles
    // waiting for the host; iterations enqueued past the crossing are no-ops (DevState::done).
    int64_t enq = 0;
    int slot = 0;
    bool have_prev = false;
    int prev_slot = 0;
    bool done = false;
    while (!done) {
        const int64_t nb = (max_iter - enq < kFixBatch) ? max_iter - enq : kFixBatch;
        if (nb > 0) {
            if ((rc = enqueue_iterations(c, nb))) return rc;
            enq += nb;
        }
        if ((rc = fetch_state(c, slot))) return rc;
        CU(cudaEventRecord(c->ev[slot], c->stream));
        if (have_prev) {
            CU(cudaEventSynchronize(c->ev[prev_slot]));
            bool all = true;                               // a batched context stops when every lattice has
            for (int b = 0; b < c->nbatch; ++b) all = all && c->host_state[(size_t)prev_slot * c->nbatch + b].done;
            if (all) done = true;
        }
        if (nb <= 0 || enq >= max_iter) {
            // nothing more to enqueue: drain the last batch
            CU(cudaEventSynchronize(c->ev[slot]));
            done = true;
        }
        have_prev = true;
        prev_slot = slot;
        slot ^= 1;
    }
    std::vector<lgf_result> r((size_t)c->nbatch);
    rc = finish(c, r.data(), true);
    if (rc) return rc;
    for (int b = 0; b < c->nbatch; ++b) out[b] = r[b];
    if (c->nbatch > 1) c->delta_valid = false;     // the ungated FFT passes of a batched context went on past each lattice's crossing
    return LGF_OK;
}

int lgf_wilson_lines(lgf_ctx* c, void* lines, int memspace) {
    if (!c || !lines || (memspace != LGF_HOST && memspace != LGF_DEVICE)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    c->delta_valid = false;             // the Delta fields serve as scratch
    if (c->nbatch != 1) return LGF_EUNSUPPORTED;   // single-lattice contexts only
    return DISPATCH(c, wilson_lines_out(c, lines, memspace));
}

int lgf_singlet_correlator(lgf_ctx* c, void* corr, int memspace) {
    if (!c || !corr || (memspace != LGF_HOST && memspace != LGF_DEVICE)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    c->delta_valid = false;
    if (c->nbatch != 1) return LGF_EUNSUPPORTED;   // single-lattice contexts only
    return DISPATCH(c, correlator(c, corr, memspace));
}

int lgf_debug_get_delta(lgf_ctx* c, void* delta_packed, int memspace) {
    if (!c || !delta_packed || (memspace != LGF_HOST && memspace != LGF_DEVICE)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    if (c->nbatch != 1) return LGF_EUNSUPPORTED;   // single-lattice contexts only
    return DISPATCH(c, get_delta(c, delta_packed, memspace));
}

int lgf_debug_fourier_accelerate(lgf_ctx* c) {
    if (!c) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded || !c->delta_valid) return LGF_ESTATE;
    if (c->nbatch != 1) return LGF_EUNSUPPORTED;
    int rc;
    for (int k = 0; k < 3; ++k)
        if ((rc = DISPATCH(c, fft(c, k, false)))) return rc;
    c->delta_valid = false;
    c->dbg_delta_tilde = true;
    CU(cudaStreamSynchronize(c->stream));
    return LGF_OK;
}

int lgf_profile_iterate(lgf_ctx* c, int64_t n, double alpha, double ms[5], lgf_result* out) {
    if (!c || !ms || n <= 0 || !(alpha > 0)) return LGF_EINVAL;
    LGF_NOT_PENDING(c);
    if (!c->loaded) return LGF_ESTATE;
    int rc = init_state(c, -1.0, (long long)n);
    if (!rc && !c->delta_valid) rc = DISPATCH(c, k1(c, 0));
    if (rc) return rc;
    c->delta_valid = true;
    c->dbg_delta_tilde = false;
    cudaEvent_t ev[6];
    for (int i = 0; i < 6; ++i) CU(cudaEventCreate(&ev[i]));
    double acc[5] = {0, 0, 0, 0, 0};
    for (int64_t it = 0; it < n && !rc; ++it) {
        for (int k = 0; k < 5 && !rc; ++k) {
            CU(cudaEventRecord(ev[k], c->stream));
            if (k < 3) rc = DISPATCH(c, fft(c, k, true));
            else if (c->fused_tile >= 0) { if (k == 3) rc = DISPATCH(c, k51(c, alpha)); }   // ms[4] stays ~0
            else if (k == 3) rc = DISPATCH(c, k5(c, alpha));
            else rc = DISPATCH(c, k1(c, 1));
        }
        if (rc) break;
        CU(cudaEventRecord(ev[5], c->stream));
        CU(cudaEventSynchronize(ev[5]));
        for (int k = 0; k < 5; ++k) {
            float t = 0;
            CU(cudaEventElapsedTime(&t, ev[k], ev[k + 1]));
            acc[k] += t;
        }
    }
    for (int i = 0; i < 6; ++i) cudaEventDestroy(ev[i]);
    if (rc) return rc;
    for (int k = 0; k < 5; ++k) ms[k] = acc[k] / (double)n;
    std::vector<lgf_result> r((size_t)c->nbatch);
    rc = finish(c, r.data(), false);
    if (rc) return rc;
    for (int b = 0; out && b < c->nbatch; ++b) out[b] = r[b];
    return LGF_OK;
}

int64_t lgf_launch_count(const lgf_ctx* c) { return c ? c->launches : 0; }

int lgf_describe(const lgf_ctx* c, char* buf, size_t n) {
    if (!c || !buf || n == 0) return LGF_EINVAL;
    const char* fft = c->xy_pipe ? "pipelined (persistent, TMA-fed)" : (c->xy_ct ? "compile-time-sized, one tile per CTA" : "runtime-radix");
    char k2[96] = "-", k3[96] = "-", k4[96] = "-";
    if (c->xy_pipe)
        snprintf(k2, sizeof(k2), "%s x=%dx%d y=%dx%d planes/tile=%d", c->xy_pipe->io ? "fft_xy_pipe_io (TMA-drained)" : "fft_xy_pipe",
                 c->xy_pipe->x_n1, c->xy_pipe->nx / c->xy_pipe->x_n1, c->xy_pipe->y_n1, c->xy_pipe->ny / c->xy_pipe->y_n1, c->xy_pipe->pb);
    if (c->xy_pipe_inv)
        snprintf(k4, sizeof(k4), "%s planes/tile=%d threads=%d ring=%d", c->xy_pipe_inv->inv3 ? "fft_xy_inv3 (padded TMA tile, last stage to global)" : "fft_xy_pipe",
                 c->xy_pipe_inv->pb, c->xy_pipe_inv->threads, c->xy_pipe_inv->nbuf);
    if (c->zt_pipe)
        snprintf(k3, sizeof(k3), "%s CX=%d", c->zt_pipe->tstore == 1 ? "fft_zt_pipe3q (quarter ring, TMA tensor stores)" : "fft_zt_pipe / fft_zt_pipe3 (tile ring)",
                 c->zt_pipe->cx);
    const char* k5 = c->fused_tile >= 0 ? "k51_update_delta (fused K5+K1)" : (c->site_variant == 2 ? "k5s (shared g)" : (c->site_variant == 1 ? "k5 (thread per site)" : "k5m (thread per site, mu)"));
    snprintf(buf, n, "lattice %dx%dx%dx%d x %d, %s, %d-real; FFT path: %s; K2: %s; K3: %s; K4: %s; K5: %s; K1 tile %dx%dx%dx%d; %d launches per iteration%s",
             c->L[0], c->L[1], c->L[2], c->L[3], c->nbatch, c->precision == LGF_F64 ? "fp64" : "fp32", c->storage, fft, k2, k3, k4, k5,
             kSiteTileDims[c->site_tile][0], kSiteTileDims[c->site_tile][1], kSiteTileDims[c->site_tile][2], kSiteTileDims[c->site_tile][3],
             c->launches_per_iter,
             c->cluster8 ? "; lgf_iterate / lgf_fix: k_cluster8_iterate (one launch per call: a 16-CTA cluster holds the field in shared memory)" : "");
    return LGF_OK;
}

int lgf_path_info(const lgf_ctx* c, int32_t info[4]) {
    if (!c || !info) return LGF_EINVAL;
    info[0] = c->xy_pipe ? 2 : (c->xy_ct ? 1 : 0);
    info[1] = c->fused_tile >= 0 ? 1 : 0;
    info[2] = c->fused_tile >= 0 ? c->fused_grid : c->lo.nblocks_site;
    info[3] = c->launches_per_iter;
    return LGF_OK;
}

}  // extern "C"
