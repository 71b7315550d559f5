// inpc_raster.cu -- C ABI (include/inpc_raster.h) over the sm_100a kernels in bin.cuh / cellsort.cuh /
// blend.cuh / back.cuh / big.cuh / grad.cuh.
//
// Forward  = memset | k_write_header | k_project_count | k_scan_u32 | k_scatter | k_classify | k_cellsort |
//            k_cellsort_big x2 | [k_scan_u32 (dump)] | k_build_items | k_blend | k_big<fwd>
// Backward = k_check_backward | k_big<bwd> | k_back | memset(queue) | k_combine | k_split
// All ordered on the caller's stream (in the forward pass k_classify / k_build_items run on a library-owned side stream that
// is forked from and joined back into it with events; the backward pass is one chain), no host synchronisation.  No device memory is allocated here, no state is kept
// on the host between calls (what a later call needs to know about a workspace is read from the Header the
// forward pass wrote into it), and there is no CPU fallback.
#include "../../include/inpc_raster.h"

#include <atomic>
#include <cstring>
#include <mutex>
#include <set>
#include <string>
#include <vector>

#include "bin.cuh"
#include "big.cuh"
#include "back.cuh"
#include "blend.cuh"
#include "cellsort.cuh"
#include "common.cuh"
#include "grad.cuh"
#include "sampler.cuh"
#include "tile.cuh"

namespace inpc {

static thread_local std::string t_cuda_error;
static std::atomic<uint64_t> g_launches{0};

// Diagnostics only (inpc_raster_launch_count / inpc_raster_launched_kernels): how many kernels this process
// has launched and which template instantiations, so that a test can check that the instantiations a
// benchmark times are the ones the parity tests compared with the oracle.
static std::mutex g_names_mu;
static std::set<std::string> g_names;
static void note_launch(const std::string& name) {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    std::lock_guard<std::mutex> lk(g_names_mu);
    g_names.insert(name);
}
template <int... V> static std::string kname(const char* base) {
    std::string s = base; s += "<";
    const int v[] = {V...};
    for (size_t i = 0; i < sizeof...(V); ++i) { if (i) s += ","; s += std::to_string(v[i]); }
    return s + ">";
}

// ---- optional per-stage device timing (inpc_raster_set_kernel_timing) ---------------------------------
// Every stage the library enqueues is bracketed by two cudaEvents on the caller's stream; the
// elapsed times are summed per stage when inpc_raster_get_kernel_times is called.  Off by default.
enum Stage { kStZeroFwd = 0, kStProjectCount, kStScan, kStScatter, kStClassify, kStCellSort, kStCellSortBig, kStBuildItems,
             kStTileFwd, kStBigFwd, kStZeroBwd, kStTileBwd, kStBigBwd, kStCombine, kStSplit, kStOther, kNumStages };
static const char* const kStageNames[kNumStages] = {
    "zero_fwd", "k_project_count", "k_scan_u32", "k_scatter", "k_classify", "k_cellsort", "k_cellsort_big", "k_build_items",
    "k_blend", "k_big_fwd", "zero_bwd", "k_back", "k_big_bwd", "k_combine", "k_split", "other"};
struct Pending { int stage; cudaEvent_t a, b; };
static std::mutex g_tmu;
static bool g_timing = false;
static std::vector<Pending> g_pending;
static std::vector<cudaEvent_t> g_event_pool;
static double g_stage_ms[kNumStages];
static uint64_t g_stage_n[kNumStages];

static cudaEvent_t take_event() {
    if (!g_event_pool.empty()) { cudaEvent_t e = g_event_pool.back(); g_event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
struct StageTimer {                       // RAII: start event now, stop event at scope exit
    bool on; int stage; cudaStream_t st; cudaEvent_t a = nullptr;
    StageTimer(int stage_, cudaStream_t st_) : on(g_timing), stage(stage_), st(st_) {
        if (on) { std::lock_guard<std::mutex> lk(g_tmu); a = take_event(); if (a) cudaEventRecord(a, st); }
    }
    ~StageTimer() {
        if (on && a) {
            std::lock_guard<std::mutex> lk(g_tmu);
            cudaEvent_t b = take_event();
            if (b) { cudaEventRecord(b, st); g_pending.push_back(Pending{stage, a, b}); }
        }
    }
};

struct Layout {
    size_t header, status0, status1, cellcnt, zero_end;   // [header, zero_end) is cleared every forward
    size_t kept, cursor, A, gT, gD, dk, Ra, Rf, items, bigpix, bigcells, bigkeys;
    size_t pcur, gpt, ord, ordinfo;                       // only with INPC_SAVE_FOR_BACKWARD
    size_t pixoff;                                        // only with INPC_SAVE_SORTED
    size_t shfeat;                                        // only with INPC_FUSED_SH: per-point features out of the SH pass
    size_t sorted_idx, sorted_depth, sorted_T;            // only with INPC_SAVE_SORTED
    size_t total;
    uint32_t C, P, max_big_cells, n_status;
};

static size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

static Layout make_layout(int64_t N, int D, int W, int H, uint32_t flags) {
    Layout L{};
    const size_t n = (size_t)N;
    L.C = (uint32_t)((W + 1) * (H + 1));
    L.P = (uint32_t)(W * H);
    L.n_status = (uint32_t)((std::max(L.C, L.P) + kScanTile - 1) / kScanTile + 1);
    L.max_big_cells = (uint32_t)(n / (kCellSmall + 1) + 1);
    size_t o = 0;
    L.header = o;  o = align_up(o + sizeof(Header));
    L.status0 = o; o = align_up(o + (size_t)L.n_status * 8);
    L.status1 = o; o = align_up(o + (size_t)L.n_status * 8);
    L.cellcnt = o; o = align_up(o + ((size_t)L.C + 1) * 4);
    L.zero_end = o;
    L.kept = o;    o = align_up(o + (n / 32 + 2) * 4);
    L.cursor = o;  o = align_up(o + ((size_t)L.C + 16) * 4);
    L.A = o;       L.gT = o; L.gD = o + (n + 8) * 16;     // the emission records are dead once the cells are sorted:
    o = align_up(o + (n + 8) * 32);                       // their bytes then hold gT | gD (16 B per record each)
    L.dk = o;      o = align_up(o + (n + 16) * 4);
    L.Ra = o;      o = align_up(o + (n + 8) * 16);
    L.Rf = o;      o = align_up(o + (n + 8) * (size_t)(4 * D));
    const size_t nbase = (size_t)((W + kTileW - 1) / kTileW) * ((H + kTileH - 1) / kTileH);
    L.items = o;   o = align_up(o + ((size_t)L.P + nbase + 16 * (kMaxBands + 1)) * 4);   // (max_items below)
    L.bigpix = o;  o = align_up(o + ((size_t)L.P + 16) * 4);
    L.bigcells = o; o = align_up(o + ((size_t)L.max_big_cells + 1) * sizeof(BigCell));
    L.bigkeys = o; o = align_up(o + (n + 8) * 8);
    const size_t max_items = (size_t)L.P + nbase + 16 * (kMaxBands + 1);
    if (flags & INPC_SAVE_FOR_BACKWARD) {
        L.pcur = o; o = align_up(o + (size_t)L.P * 16);
        L.gpt = o;  o = align_up(o + n * (size_t)(D == 4 ? 32 : 64) + 64);
        L.ord = o;  o = align_up(o + (4 * n + 8 * (size_t)kTileThreads * nbase + 64) * 2);   // blocks in 8-entry units, <= one item per pixel
        L.ordinfo = o; o = align_up(o + max_items * 8);
    }
    if (flags & INPC_FUSED_SH) { L.shfeat = o; o = align_up(o + (n + 8) * 16); }
    if (flags & INPC_SAVE_SORTED) {
        L.pixoff = o;       o = align_up(o + ((size_t)L.P + 1) * 4);
        L.sorted_idx = o;   o = align_up(o + (4 * n + 8) * 4);
        L.sorted_depth = o; o = align_up(o + (4 * n + 8) * 4);
        L.sorted_T = o;     o = align_up(o + (4 * n + 8) * 4);
    }
    L.total = o;
    return L;
}

constexpr int kMaxDevices = 64;
struct DeviceInfo { int dev = 0; int sms = 0; bool ok = false; };
static std::mutex g_dev_mu;                       // guards the per-device caches below
static DeviceInfo device_info() {
    static DeviceInfo cached[kMaxDevices];
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return DeviceInfo{};
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (!cached[dev].ok) {
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return DeviceInfo{};
        cached[dev].dev = dev; cached[dev].sms = sms; cached[dev].ok = true;
    }
    return cached[dev];
}

static int cuda_fail(cudaError_t e) {
    t_cuda_error = cudaGetErrorString(e);
    return INPC_ERR_CUDA;
}
#define INPC_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) return cuda_fail(e_); } while (0)
#define INPC_LAUNCHED(...) do { note_launch(__VA_ARGS__); cudaError_t e_ = cudaGetLastError(); if (e_ != cudaSuccess) return cuda_fail(e_); } while (0)

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int check_common(int64_t N, int D, const inpc_camera* cam) {
    if (!cam || N < 0 || N >= (1ll << 30)) return INPC_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0 || !(cam->near_z < cam->far_z)) return INPC_ERR_INVALID_ARG;
    if (!(cam->near_z >= 0.f)) return INPC_ERR_INVALID_ARG;   // depth keys are the raw bits of a positive z_c
    if (D != 4 && D != 8) return INPC_ERR_UNSUPPORTED;
    if (cam->width > 4095 || cam->height > 4095) return INPC_ERR_UNSUPPORTED;
    return INPC_OK;
}

static ViewPoint view_point(const inpc_camera* c) {       // camera centre in world space: -R^T t
    ViewPoint v;
    v.cx = -(c->R[0] * c->t[0] + c->R[3] * c->t[1] + c->R[6] * c->t[2]);
    v.cy = -(c->R[1] * c->t[0] + c->R[4] * c->t[1] + c->R[7] * c->t[2]);
    v.cz = -(c->R[2] * c->t[0] + c->R[5] * c->t[1] + c->R[8] * c->t[2]);
    return v;
}

static Camera to_camera(const inpc_camera* c) {
    Camera k;
    k.fx = c->fx; k.fy = c->fy; k.cx = c->cx; k.cy = c->cy;
    for (int i = 0; i < 9; ++i) k.R[i] = c->R[i];
    for (int i = 0; i < 3; ++i) k.t[i] = c->t[i];
    k.near_z = c->near_z; k.far_z = c->far_z; k.W = c->width; k.H = c->height;
    return k;
}

// Opt-in dynamic shared memory and the persistent grid size (resident CTAs per SM x SMs) of one kernel, cached
// PER DEVICE (both are per-device properties): grid_by_dev is the kernel's own function-static table.
template <typename K>
static int persistent_grid(K kernel, int threads, size_t smem, const DeviceInfo& di, int (&grid_by_dev)[kMaxDevices],
                           int* out) {
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (grid_by_dev[di.dev] == 0) {
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return cuda_fail(e);
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem);
        if (e != cudaSuccess) return cuda_fail(e);
        if (per_sm < 1) per_sm = 1;
        grid_by_dev[di.dev] = per_sm * di.sms;
    }
    *out = grid_by_dev[di.dev];
    return INPC_OK;
}

template <int D>
static int launch_back(const BackArgs& A, const DeviceInfo& di, cudaStream_t st) {
    constexpr size_t smem = back_smem_bytes<D>();
    static int grid_by_dev[kMaxDevices] = {};
    int grid = 0;
    int rc = persistent_grid(k_back<D>, kTileThreads, smem, di, grid_by_dev, &grid);
    if (rc != INPC_OK) return rc;
    { StageTimer tm(kStTileBwd, st);
      k_back<D><<<grid, kTileThreads, smem, st>>>(A); }
    INPC_LAUNCHED(kname<D>("k_back"));
    return INPC_OK;
}

template <int D, bool SAVE, bool DUMP>
static int launch_blend(const BlendArgs& A, const DeviceInfo& di, cudaStream_t st) {
    constexpr size_t smem = blend_smem_bytes<D, SAVE>();
    static int grid_by_dev[kMaxDevices] = {};
    int grid = 0;
    int rc = persistent_grid(k_blend<D, SAVE, DUMP>, kTileThreads, smem, di, grid_by_dev, &grid);
    if (rc != INPC_OK) return rc;
    { StageTimer tm(kStTileFwd, st);
      k_blend<D, SAVE, DUMP><<<grid, kTileThreads, smem, st>>>(A); }
    INPC_LAUNCHED(kname<D, SAVE ? 1 : 0, DUMP ? 1 : 0>("k_blend"));
    return INPC_OK;
}

template <int D, int MODE>
static int launch_big(const BigArgs& A, int sms, cudaStream_t st) {
    { StageTimer tm(MODE == kBwd ? kStBigBwd : kStBigFwd, st);
      k_big<D, MODE><<<sms * 8, kLongThreads, 0, st>>>(A); }
    INPC_LAUNCHED(kname<D, MODE>("k_big"));
    return INPC_OK;
}

template <int D, int THREADS, int CHUNK>
static int launch_cellsort_big_class(const Header* hdr, uint32_t n_lo, uint32_t n_hi, uint32_t* cursor,
                                     const BigCell* bigcells, const float4* A, unsigned long long* keys, const float* feat,
                                     uint32_t* dk, float4* Ra, float4* Rf, const DeviceInfo& di, uint32_t max_big_cells,
                                     cudaStream_t st) {
    constexpr size_t smem = (size_t)CHUNK * 8;
    static int grid_by_dev[kMaxDevices] = {};
    int grid = 0;
    int rc = persistent_grid(k_cellsort_big<D, THREADS, CHUNK>, THREADS, smem, di, grid_by_dev, &grid);
    if (rc != INPC_OK) return rc;
    const int g = (int)std::min<uint32_t>((uint32_t)grid, std::max<uint32_t>(max_big_cells, 1u));
    k_cellsort_big<D, THREADS, CHUNK><<<g, THREADS, smem, st>>>(hdr, n_lo, n_hi, cursor, bigcells, A, keys, feat, dk, Ra, Rf);
    INPC_LAUNCHED(kname<D, CHUNK>("k_cellsort_big"));
    return INPC_OK;
}

// cells of kCellSmall+1 .. 1024 points, then the larger ones (two work cursors in the header)
template <int D>
static int launch_cellsort_big(Header* hdr, const BigCell* bigcells, const float4* A, unsigned long long* keys,
                               const float* feat, uint32_t* dk, float4* Ra, float4* Rf, const DeviceInfo& di,
                               uint32_t max_big_cells, cudaStream_t st) {
    StageTimer tm(kStCellSortBig, st);
    int rc = launch_cellsort_big_class<D, 128, 1024>(hdr, 0u, 1024u, &hdr->bigcell_cursor, bigcells, A, keys, feat, dk, Ra,
                                                     Rf, di, max_big_cells, st);
    if (rc != INPC_OK) return rc;
    return launch_cellsort_big_class<D, kBigThreads, kBigChunk>(hdr, 1025u, 0xFFFFFFFFu, &hdr->cellsort_cursor, bigcells, A,
                                                                keys, feat, dk, Ra, Rf, di, max_big_cells, st);
}

__global__ void k_write_header(Header* h, uint32_t flags, int W, int H, int D, uint32_t N) {
    h->magic = kMagic; h->flags = flags; h->W = W; h->H = H; h->D = D; h->n_points = N;
}

// First kernel of the backward pass: does the workspace hold the forward state these arguments describe?
// bwd_ok gates every later backward kernel (they return at once when it is 0, so a stale or foreign
// workspace is never interpreted); the reason is left in the sticky status word that
// inpc_raster_get_status returns.  Also resets the tile work cursor.
__global__ void k_check_backward(Header* h, int W, int H, int D, uint32_t N) {
    int32_t st = INPC_OK;
    if (h->magic != kMagic || !(h->flags & INPC_SAVE_FOR_BACKWARD)) st = INPC_ERR_NO_SAVED_STATE;
    else if (h->W != W || h->H != H || h->D != D || h->n_points != N) st = INPC_ERR_INVALID_ARG;
    h->bwd_ok = st == INPC_OK ? 1u : 0u;
    if (st != INPC_OK) h->status = st;
    for (int b = 0; b < kMaxBands; ++b) h->band_cursor[b] = 0;
    h->combine_cursor = 0; h->combine_q_head = 0; h->combine_q_tail = 0; h->combine_done = 0;
}

// ---- band plan + the library's own side stream --------------------------------------------------------------------
// The sort / gather kernels are bound by DRAM access rates and leave the SMs idle; the merge kernels are bound by
// shared-memory residency and latency and leave DRAM idle.  So the image is cut into bands of tile rows and the two
// kinds of work run on two streams: while band b is blended (backward: combined) on the side stream, band b + 1 is
// sorted (backward: walked) on the caller's stream.  Fork / join is by events, so from the caller's point of view
// everything is still ordered on ITS stream.  With kernel timing enabled (inpc_raster_set_kernel_timing) the side
// stream is not used: the per-stage times are then those of kernels running alone.
struct Bands {
    BandPlan plan;                         // n_bands, rows_per_band, item_base
    uint32_t sort_end[kMaxBands];          // forward: band b may be blended once the cell units < sort_end[b] are sorted
    uint32_t comb_end[kMaxBands];          // backward: once band b is walked the cell units < comb_end[b] can be combined
};

static Bands make_bands(int W, int H, uint32_t C, int want) {
    Bands B{};
    const int ntx = (W + kTileW - 1) / kTileW, nty = (H + kTileH - 1) / kTileH;
    const uint32_t n_units = (C + kCsCells - 1) / kCsCells;
    int nb = std::max(1, std::min(std::min(want, kMaxBands), nty / 8));      // at least 8 tile rows per band
    const int rpb = (nty + nb - 1) / nb;
    nb = (nty + rpb - 1) / rpb;
    B.plan.n_bands = nb; B.plan.rows_per_band = rpb;
    uint32_t base = 0;
    for (int b = 0; b < nb; ++b) {
        const int r0 = b * rpb, r1 = std::min(nty, (b + 1) * rpb);
        const int y1 = std::min(H, r1 * kTileH);                             // first pixel row behind the band
        B.plan.item_base[b] = base;
        base += (uint32_t)((size_t)(y1 - r0 * kTileH) * W + (size_t)(r1 - r0) * ntx + 16);   // worst case: one item per pixel
        // forward: the band's pixels read cell rows <= y1
        const uint64_t c_hi = (uint64_t)(y1 + 1) * (W + 1);
        B.sort_end[b] = b == nb - 1 ? n_units : (uint32_t)std::min<uint64_t>(n_units, (c_hi + kCsCells - 1) / kCsCells);
        // backward: cell row j is complete once pixel rows j - 1 and j are walked, i.e. rows j <= y1 - 1
        B.comb_end[b] = b == nb - 1 ? n_units : (uint32_t)std::min<uint64_t>(n_units, ((uint64_t)y1 * (W + 1)) / kCsCells);
    }
    return B;
}

constexpr int kDefaultBands = 1;      // measured: 4 bands cost more per kernel (tails, <1 wave per launch) than the overlap wins (1.51 -> 1.61 ms)
constexpr int kSideEvents = 2 * kMaxBands + 4;
struct Side { cudaStream_t stream = nullptr; cudaEvent_t ev[kSideEvents] = {}; bool ok = false; };
static std::mutex g_side_mu;              // serialises the enqueue of calls that use the side stream
static Side* side_for(const DeviceInfo& di) {
    static Side sides[kMaxDevices];
    Side& s = sides[di.dev];
    if (!s.ok) {
        if (cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking) != cudaSuccess) return nullptr;
        for (int i = 0; i < kSideEvents; ++i)
            if (cudaEventCreateWithFlags(&s.ev[i], cudaEventDisableTiming) != cudaSuccess) return nullptr;
        s.ok = true;
    }
    return &s;
}

template <int D>
static int forward_impl(const float* pos, const float* opacity, const float* feat, int64_t N, const inpc_camera* cam,
                        float* out_feat, float* out_alpha, unsigned char* ws, const Layout& L, uint32_t flags,
                        float out_scale, cudaStream_t st, const float* sh_coeff = nullptr) {
    const DeviceInfo di = device_info();
    if (!di.ok) return cuda_fail(cudaErrorNoDevice);
    const Camera camk = to_camera(cam);
    ImageIO io{};
    io.planar = (flags & INPC_OUT_PLANAR) ? 1 : 0; io.accumulate = (flags & INPC_ACCUMULATE) ? 1 : 0;
    io.scale = out_scale; io.P = L.P;
    const int W = cam->width, H = cam->height;
    Header* hdr = reinterpret_cast<Header*>(ws + L.header);
    uint32_t* cellcnt = reinterpret_cast<uint32_t*>(ws + L.cellcnt);
    uint32_t* kept = reinterpret_cast<uint32_t*>(ws + L.kept);
    uint32_t* cursor = reinterpret_cast<uint32_t*>(ws + L.cursor);
    float4* Arec = reinterpret_cast<float4*>(ws + L.A);
    uint32_t* dk = reinterpret_cast<uint32_t*>(ws + L.dk);
    float4* Ra = reinterpret_cast<float4*>(ws + L.Ra);
    float4* Rf = reinterpret_cast<float4*>(ws + L.Rf);
    uint32_t* items = reinterpret_cast<uint32_t*>(ws + L.items);
    uint32_t* bigpix = reinterpret_cast<uint32_t*>(ws + L.bigpix);
    BigCell* bigcells = reinterpret_cast<BigCell*>(ws + L.bigcells);
    const bool dump = (flags & INPC_SAVE_SORTED) != 0;
    const bool save = (flags & INPC_SAVE_FOR_BACKWARD) != 0;
    uint32_t* pixoff = dump ? reinterpret_cast<uint32_t*>(ws + L.pixoff) : nullptr;

    // two streams unless per-stage timing wants every kernel alone
    std::unique_lock<std::mutex> side_lock(g_side_mu, std::defer_lock);
    Side* side = nullptr;
    if (!g_timing && N > 0) { side_lock.lock(); side = side_for(di); if (!side) return cuda_fail(cudaGetLastError()); }
    cudaStream_t s2 = side ? side->stream : st;
    const Bands B = make_bands(W, H, L.C, kDefaultBands);      // a function of the image shape only: backward rebuilds it
    const int nb = B.plan.n_bands;
    int ev = 0;
    auto fork = [&](cudaStream_t from, cudaStream_t to) -> cudaError_t {      // `to` waits for what `from` has enqueued
        if (from == to) return cudaSuccess;
        cudaEvent_t e = side->ev[ev++ % kSideEvents];
        cudaError_t rc = cudaEventRecord(e, from);
        return rc != cudaSuccess ? rc : cudaStreamWaitEvent(to, e, 0);
    };

    { StageTimer tm(kStZeroFwd, st);
      INPC_CUDA(cudaMemsetAsync(ws + L.header, 0, L.zero_end - L.header, st));
      k_write_header<<<1, 1, 0, st>>>(hdr, flags, W, H, D, (uint32_t)N); }
    INPC_LAUNCHED("k_write_header");
    // grid sizes in CTAs per SM are measured optima (round-1 facts): the passes that scatter
    // (k_scatter, k_cellsort) are fastest with ONE resident wave of 4 CTAs per SM, the streaming count pass with 8
    const int bin_grid = (int)std::min<int64_t>((N + kBinChunk - 1) / kBinChunk, (int64_t)di.sms * 8);
    const int scatter_grid = (int)std::min<int64_t>((N + kBinChunk - 1) / kBinChunk, (int64_t)di.sms * 4);
    if (N > 0) {
        { StageTimer tm(kStProjectCount, st);
          k_project_count<<<bin_grid, kBinThreads, 0, st>>>(pos, (long long)N, camk, cellcnt, kept); }
        INPC_LAUNCHED("k_project_count");
    }
    { StageTimer tm(kStScan, st);
      k_scan_u32<<<(L.C + kScanTile - 1) / kScanTile, kScanThreads, 0, st>>>(
          cellcnt, L.C, reinterpret_cast<unsigned long long*>(ws + L.status0), &hdr->scan_tile_counter, &hdr->nrec, cursor); }
    INPC_LAUNCHED("k_scan_u32");

    // side stream: everything that needs only the cell offsets (per-pixel counts, large-cell list, tile work lists)
    INPC_CUDA(fork(st, s2));
    { StageTimer tm(kStClassify, s2);
      k_classify<<<(L.C + 255) / 256, 256, 0, s2>>>(cellcnt, W, H, hdr, bigcells, pixoff); }
    INPC_LAUNCHED("k_classify");
    if (dump) {
        { StageTimer tm(kStOther, s2);
          k_scan_u32<<<(L.P + kScanTile - 1) / kScanTile, kScanThreads, 0, s2>>>(
              pixoff, L.P, reinterpret_cast<unsigned long long*>(ws + L.status1), &hdr->pad0, nullptr, nullptr); }
        INPC_LAUNCHED("k_scan_u32");
    }
    const int ntx = (W + kTileW - 1) / kTileW, nty = (H + kTileH - 1) / kTileH;
    { StageTimer tm(kStBuildItems, s2);
      k_build_items<<<(ntx * nty + 127) / 128, 128, 0, s2>>>(cellcnt, W, H, TileCfg<D>::kCap, B.plan, hdr, items, bigpix); }
    INPC_LAUNCHED("k_build_items");

    // caller's stream: scatter, then the cell sort band by band
    if (N > 0) {
        { StageTimer tm(kStScatter, st);
          if (sh_coeff) {
              feat = reinterpret_cast<const float*>(ws + L.shfeat);       // from here on the features are the SH pass's
              k_scatter<true><<<scatter_grid, kBinThreads, 0, st>>>(pos, opacity, (long long)N, camk, cursor, Arec,
                                                                    reinterpret_cast<const float4*>(sh_coeff), view_point(cam),
                                                                    reinterpret_cast<float4*>(ws + L.shfeat));
          } else {
              k_scatter<false><<<scatter_grid, kBinThreads, 0, st>>>(pos, opacity, (long long)N, camk, cursor, Arec, nullptr,
                                                                     ViewPoint{}, nullptr);
          } }
        INPC_LAUNCHED(sh_coeff ? "k_scatter<1>" : "k_scatter<0>");
        INPC_CUDA(fork(s2, st));                                              // the large-cell list
        int rc = launch_cellsort_big<D>(hdr, bigcells, Arec,
                                        reinterpret_cast<unsigned long long*>(ws + L.bigkeys), feat, dk, Ra, Rf, di,
                                        L.max_big_cells, st);
        if (rc != INPC_OK) return rc;
    }

    BlendArgs A{};
    A.hdr = hdr; A.celloff = cellcnt; A.dk = dk; A.Ra = Ra; A.Rf = Rf;
    A.W = W; A.H = H; A.out_feat = out_feat; A.out_alpha = out_alpha; A.io = io;
    BigArgs Bg{};
    Bg.hdr = hdr; Bg.bigpix = bigpix; Bg.celloff = cellcnt; Bg.dk = dk; Bg.Ra = Ra; Bg.Rf = Rf;
    Bg.W = W; Bg.H = H; Bg.out_feat = out_feat; Bg.out_alpha = out_alpha; Bg.io = io;
    if (save) {
        A.gT = Bg.gT = reinterpret_cast<float*>(ws + L.gT);
        A.pcur = Bg.pcur = reinterpret_cast<uint4*>(ws + L.pcur);
        A.ord = reinterpret_cast<uint16_t*>(ws + L.ord); A.ord_cursor = &hdr->ord_cursor;
    }
    Bg.pixoff = A.pixoff = pixoff;
    if (dump) {
        Bg.sorted_idx = A.sorted_idx = reinterpret_cast<uint32_t*>(ws + L.sorted_idx);
        Bg.sorted_depth = A.sorted_depth = reinterpret_cast<uint32_t*>(ws + L.sorted_depth);
        Bg.sorted_T = A.sorted_T = reinterpret_cast<float*>(ws + L.sorted_T);
    }
    uint32_t u0 = 0;
    for (int b = 0; b < nb; ++b) {
        const uint32_t u1 = B.sort_end[b];
        if (N > 0 && u1 > u0) {
            { StageTimer tm(kStCellSort, st);
              k_cellsort<D><<<(int)std::min<uint32_t>(u1 - u0, (uint32_t)di.sms * 4), kCsThreads, 0, st>>>(
                  Arec, cellcnt, L.C, u0, u1, feat, dk, Ra, Rf); }
            INPC_LAUNCHED(kname<D>("k_cellsort"));
            u0 = u1;
        }
        // (Measured in round 3: with one band, launching the blend on the caller's stream instead of hopping to the side
        // stream and back is no faster -- train 1.370 -> 1.380 ms -- so the hop stays.)
        cudaStream_t sb = s2;
        INPC_CUDA(fork(st, sb));                                              // band b is sorted: blend it
        A.items = items + B.plan.item_base[b]; A.n_items = &hdr->band_items[b]; A.item_cursor = &hdr->band_cursor[b];
        if (save) A.ordinfo = reinterpret_cast<uint2*>(ws + L.ordinfo) + B.plan.item_base[b];
        int rc = dump ? (save ? launch_blend<D, true, true>(A, di, sb) : launch_blend<D, false, true>(A, di, sb))
                      : (save ? launch_blend<D, true, false>(A, di, sb) : launch_blend<D, false, false>(A, di, sb));
        if (rc != INPC_OK) return rc;
    }
    INPC_CUDA(fork(s2, st));                                                  // join
    int rc = INPC_OK;
    if (N > 0) rc = dump ? launch_big<D, kFwdDump>(Bg, di.sms, st) : launch_big<D, kFwd>(Bg, di.sms, st);
    return rc;
}

template <int D>
static int backward_impl(int64_t N, const inpc_camera* cam, const float* g_feat, const float* g_alpha, float* d_feat,
                         float* d_opacity, float* d_uv, float* blend_weight, unsigned char* ws, const Layout& L,
                         uint32_t flags, float grad_scale, cudaStream_t st, const float* sh_pos = nullptr) {
    const DeviceInfo di = device_info();
    if (!di.ok) return cuda_fail(cudaErrorNoDevice);
    const int W = cam->width, H = cam->height;
    ImageIO io{};
    io.planar = (flags & INPC_OUT_PLANAR) ? 1 : 0; io.accumulate = 0; io.scale = grad_scale; io.P = L.P;
    Header* hdr = reinterpret_cast<Header*>(ws + L.header);
    { StageTimer tm(kStZeroBwd, st);
      k_check_backward<<<1, 1, 0, st>>>(hdr, W, H, D, (uint32_t)N); }
    INPC_LAUNCHED("k_check_backward");
    if (N == 0) return INPC_OK;
    // (the backward pass is one chain of kernels on the caller's stream: it does not use the library's side stream)
    const uint32_t* celloff = reinterpret_cast<uint32_t*>(ws + L.cellcnt);
    const float4* Ra = reinterpret_cast<float4*>(ws + L.Ra);
    const float4* Rf = reinterpret_cast<float4*>(ws + L.Rf);
    float* gT = reinterpret_cast<float*>(ws + L.gT);
    float* gD = reinterpret_cast<float*>(ws + L.gD);
    uint4* pcur = reinterpret_cast<uint4*>(ws + L.pcur);
    float* gpt = reinterpret_cast<float*>(ws + L.gpt);
    uint32_t* items = reinterpret_cast<uint32_t*>(ws + L.items);
    // long-run pixels first: they need nothing but the forward state, and every combine below may touch their cells
    BigArgs Bg{};
    Bg.hdr = hdr; Bg.bigpix = reinterpret_cast<uint32_t*>(ws + L.bigpix); Bg.celloff = celloff;
    Bg.dk = reinterpret_cast<uint32_t*>(ws + L.dk); Bg.Ra = Ra; Bg.Rf = Rf;
    Bg.W = W; Bg.H = H; Bg.gT = gT; Bg.pcur = pcur; Bg.g_feat = g_feat; Bg.g_alpha = g_alpha; Bg.gD = gD; Bg.io = io;
    int rc = launch_big<D, kBwd>(Bg, di.sms, st);
    if (rc != INPC_OK) return rc;
    BackArgs A{};
    A.hdr = hdr; A.celloff = celloff; A.Ra = Ra; A.Rf = Rf;
    A.ord = reinterpret_cast<const uint16_t*>(ws + L.ord);
    A.W = W; A.H = H; A.gT = gT; A.pcur = pcur; A.g_feat = g_feat; A.g_alpha = g_alpha; A.gD = gD; A.io = io;
    const Bands Bf = make_bands(W, H, L.C, kDefaultBands);     // the plan the forward built the item lists with
    for (int b = 0; b < Bf.plan.n_bands; ++b) {
        A.items = items + Bf.plan.item_base[b]; A.n_items = &hdr->band_items[b]; A.item_cursor = &hdr->band_cursor[b];
        A.ordinfo = reinterpret_cast<const uint2*>(ws + L.ordinfo) + Bf.plan.item_base[b];
        rc = launch_back<D>(A, di, st);
        if (rc != INPC_OK) return rc;
    }
    { StageTimer tm(kStCombine, st);                                          // every fragment is walked: combine the records
      const uint32_t n_units = (L.C + kGradCells - 1) / kGradCells;
      // the queue of parts lives in the large-cell sort's key scratch (dead since the forward pass): <= N / kGradPart entries
      INPC_CUDA(cudaMemsetAsync(ws + L.bigkeys, 0xFF, ((size_t)N / kGradPart + 2) * 8, st));
      k_combine<D><<<(int)std::min<uint32_t>(n_units, (uint32_t)di.sms * 8), kGradThreads, 0, st>>>(
          hdr, celloff, L.C, 0u, n_units, W, H, Ra, reinterpret_cast<const float4*>(gT),
          reinterpret_cast<const float4*>(gD), pcur, g_feat, io, gpt, reinterpret_cast<unsigned long long*>(ws + L.bigkeys)); }
    INPC_LAUNCHED(kname<D>("k_combine"));
    { StageTimer tm(kStSplit, st);
      const int grid = (int)std::min<int64_t>((N + 255) / 256, (int64_t)di.sms * 16);
      const uint32_t* kept = reinterpret_cast<const uint32_t*>(ws + L.kept);
      if (sh_pos) k_split<D, true><<<grid, 256, 0, st>>>(hdr, gpt, kept, (long long)N, d_feat, d_opacity, d_uv, blend_weight,
                                                         sh_pos, view_point(cam));
      else k_split<D, false><<<grid, 256, 0, st>>>(hdr, gpt, kept, (long long)N, d_feat, d_opacity, d_uv, blend_weight,
                                                   nullptr, ViewPoint{}); }
    INPC_LAUNCHED(sh_pos ? kname<D, 1>("k_split") : kname<D, 0>("k_split"));
    return INPC_OK;
}

}  // namespace inpc

using namespace inpc;

extern "C" {

size_t inpc_raster_workspace_bytes(int64_t n_points, int32_t D, int32_t W, int32_t H, uint32_t flags) {
    if (n_points < 0 || n_points >= (1ll << 30) || (D != 4 && D != 8) || W <= 0 || H <= 0 || W > 4095 || H > 4095) return 0;
    return make_layout(n_points, D, W, H, flags).total;
}

static int forward_entry(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                         const inpc_camera* cam, float* out_feat, float* out_alpha, void* workspace,
                         size_t workspace_bytes, uint32_t flags, float out_scale, void* cuda_stream) {
    int rc = check_common(N, D, cam);
    if (rc != INPC_OK) return rc;
    if (!out_feat || !out_alpha || !workspace) return INPC_ERR_INVALID_ARG;
    if (N > 0 && (!pos || !opacity || !feat)) return INPC_ERR_INVALID_ARG;
    if (flags & ~(INPC_SAVE_FOR_BACKWARD | INPC_SAVE_SORTED | INPC_OUT_PLANAR | INPC_ACCUMULATE)) return INPC_ERR_INVALID_ARG;
    if (!aligned16(pos) || !aligned16(opacity) || !aligned16(feat) || !aligned16(out_feat) || !aligned16(out_alpha) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u))
        return INPC_ERR_INVALID_ARG;
    const Layout L = make_layout(N, D, cam->width, cam->height, flags);
    if (workspace_bytes < L.total) return INPC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    return D == 4 ? forward_impl<4>(pos, opacity, feat, N, cam, out_feat, out_alpha, ws, L, flags, out_scale, st)
                  : forward_impl<8>(pos, opacity, feat, N, cam, out_feat, out_alpha, ws, L, flags, out_scale, st);
}

int inpc_raster_forward(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                        const inpc_camera* cam, float* out_feat, float* out_alpha, void* workspace,
                        size_t workspace_bytes, uint32_t flags, void* cuda_stream) {
    if (flags & ~(INPC_SAVE_FOR_BACKWARD | INPC_SAVE_SORTED)) return INPC_ERR_INVALID_ARG;   // layout flags: _ex
    return forward_entry(pos, opacity, feat, N, D, cam, out_feat, out_alpha, workspace, workspace_bytes, flags, 1.0f,
                         cuda_stream);
}

int inpc_raster_forward_ex(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                           const inpc_camera* cam, float* out_feat, float* out_alpha, void* workspace,
                           size_t workspace_bytes, uint32_t flags, float out_scale, void* cuda_stream) {
    return forward_entry(pos, opacity, feat, N, D, cam, out_feat, out_alpha, workspace, workspace_bytes, flags, out_scale,
                         cuda_stream);
}

int inpc_raster_forward_sh(const float* pos, const float* opacity, const float* sh_coeff, int64_t N,
                           const inpc_camera* cam, float* out_feat, float* out_alpha, void* workspace,
                           size_t workspace_bytes, uint32_t flags, float out_scale, void* cuda_stream) {
    int rc = check_common(N, 4, cam);
    if (rc != INPC_OK) return rc;
    if (!out_feat || !out_alpha || !workspace) return INPC_ERR_INVALID_ARG;
    if (N > 0 && (!pos || !opacity || !sh_coeff)) return INPC_ERR_INVALID_ARG;
    if (flags & ~(INPC_SAVE_FOR_BACKWARD | INPC_SAVE_SORTED | INPC_OUT_PLANAR | INPC_ACCUMULATE | INPC_FUSED_SH)) return INPC_ERR_INVALID_ARG;
    flags |= INPC_FUSED_SH;
    if (!aligned16(pos) || !aligned16(opacity) || !aligned16(sh_coeff) || !aligned16(out_feat) || !aligned16(out_alpha) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u))
        return INPC_ERR_INVALID_ARG;
    const Layout L = make_layout(N, 4, cam->width, cam->height, flags);
    if (workspace_bytes < L.total) return INPC_ERR_WORKSPACE_TOO_SMALL;
    return forward_impl<4>(pos, opacity, nullptr, N, cam, out_feat, out_alpha, static_cast<unsigned char*>(workspace), L, flags,
                           out_scale, static_cast<cudaStream_t>(cuda_stream), N > 0 ? sh_coeff : nullptr);
}

int inpc_raster_backward_sh(const float* pos, const float* opacity, const float* sh_coeff, int64_t N,
                            const inpc_camera* cam, const float* grad_out_feat, const float* grad_out_alpha,
                            float* grad_sh_coeff, float* grad_opacity, float* grad_uv, float* blend_weight,
                            void* workspace, size_t workspace_bytes, uint32_t flags, float grad_scale, void* cuda_stream) {
    (void)opacity; (void)sh_coeff;
    int rc = check_common(N, 4, cam);
    if (rc != INPC_OK) return rc;
    if (!grad_out_feat || !workspace) return INPC_ERR_INVALID_ARG;
    if (N > 0 && !pos) return INPC_ERR_INVALID_ARG;             // (any of the gradient outputs may be NULL)
    if (flags & ~INPC_OUT_PLANAR) return INPC_ERR_INVALID_ARG;
    if (!aligned16(pos) || !aligned16(grad_out_feat) || !aligned16(grad_out_alpha) || !aligned16(grad_sh_coeff) ||
        !aligned16(grad_opacity) || !aligned16(grad_uv) || !aligned16(blend_weight) ||
        (reinterpret_cast<uintptr_t>(workspace) & 255u))
        return INPC_ERR_INVALID_ARG;
    const Layout L = make_layout(N, 4, cam->width, cam->height, INPC_SAVE_FOR_BACKWARD | INPC_FUSED_SH);
    if (workspace_bytes < L.total) return INPC_ERR_WORKSPACE_TOO_SMALL;
    return backward_impl<4>(N, cam, grad_out_feat, grad_out_alpha, grad_sh_coeff, grad_opacity, grad_uv, blend_weight,
                            static_cast<unsigned char*>(workspace), L, flags, grad_scale,
                            static_cast<cudaStream_t>(cuda_stream), N > 0 ? pos : nullptr);
}

int inpc_raster_level_camera(const inpc_camera* cam, int32_t level, inpc_camera* out) {
    if (!cam || !out || level < 0 || level > 8) return INPC_ERR_INVALID_ARG;
    *out = *cam;
    const float s = 1.0f / (float)(1 << level);              // a power of two: every product below is exact
    out->fx = cam->fx * s; out->fy = cam->fy * s; out->cx = cam->cx * s; out->cy = cam->cy * s;
    out->width = (cam->width + (1 << level) - 1) >> level;
    out->height = (cam->height + (1 << level) - 1) >> level;
    return INPC_OK;
}

int inpc_raster_forward_levels(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                               const inpc_camera* cam, int32_t n_levels, float* const* out_feat, float* const* out_alpha,
                               void* const* workspaces, const size_t* workspace_bytes, uint32_t flags, float out_scale,
                               void* cuda_stream) {
    if (n_levels < 1 || n_levels > 8 || !out_feat || !out_alpha || !workspaces || !workspace_bytes) return INPC_ERR_INVALID_ARG;
    for (int32_t l = 0; l < n_levels; ++l) {
        inpc_camera c;
        int rc = inpc_raster_level_camera(cam, l, &c);
        if (rc == INPC_OK)
            rc = forward_entry(pos, opacity, feat, N, D, &c, out_feat[l], out_alpha[l], workspaces[l], workspace_bytes[l],
                               flags, out_scale, cuda_stream);
        if (rc != INPC_OK) return rc;
    }
    return INPC_OK;
}

int inpc_raster_forward_multisample(int32_t n_clouds, const float* const* pos, const float* const* opacity,
                                    const float* const* feat, const int64_t* N, int32_t D, const inpc_camera* cam,
                                    int32_t n_levels, float* const* out_feat, float* const* out_alpha, void* workspace,
                                    size_t workspace_bytes, uint32_t flags, void* cuda_stream) {
    if (n_clouds < 1 || n_clouds > 64 || !pos || !opacity || !feat || !N) return INPC_ERR_INVALID_ARG;
    if (n_levels < 1 || n_levels > 8 || !out_feat || !out_alpha) return INPC_ERR_INVALID_ARG;
    if (flags & ~INPC_OUT_PLANAR) return INPC_ERR_INVALID_ARG;     // inference path: one workspace, nothing is saved
    const float scale = 1.0f / (float)n_clouds;
    for (int32_t s = 0; s < n_clouds; ++s)
        for (int32_t l = 0; l < n_levels; ++l) {
            inpc_camera c;
            int rc = inpc_raster_level_camera(cam, l, &c);
            if (rc == INPC_OK)
                rc = forward_entry(pos[s], opacity[s], feat[s], N[s], D, &c, out_feat[l], out_alpha[l], workspace,
                                   workspace_bytes, flags | (s > 0 ? INPC_ACCUMULATE : 0u), scale, cuda_stream);
            if (rc != INPC_OK) return rc;
        }
    return INPC_OK;
}

static int backward_entry(int64_t N, int32_t D, const inpc_camera* cam, const float* grad_out_feat,
                          const float* grad_out_alpha, float* grad_feat, float* grad_opacity, float* grad_uv,
                          float* blend_weight, void* workspace, size_t workspace_bytes, uint32_t flags, float grad_scale,
                          void* cuda_stream) {
    int rc = check_common(N, D, cam);
    if (rc != INPC_OK) return rc;
    if (!grad_out_feat || !workspace) return INPC_ERR_INVALID_ARG;
    if (flags & ~INPC_OUT_PLANAR) return INPC_ERR_INVALID_ARG;
    if (!aligned16(grad_out_feat) || !aligned16(grad_out_alpha) || !aligned16(grad_feat) || !aligned16(grad_opacity) ||
        !aligned16(grad_uv) || !aligned16(blend_weight) || (reinterpret_cast<uintptr_t>(workspace) & 255u))
        return INPC_ERR_INVALID_ARG;
    // Everything the backward pass touches lies in front of the INPC_SAVE_SORTED arrays, so its layout follows
    // from these arguments alone; whether the workspace really holds that forward is checked ON THE DEVICE
    // (k_check_backward) against the Header the forward wrote -- no host-side record of workspaces exists.
    const Layout L = make_layout(N, D, cam->width, cam->height, INPC_SAVE_FOR_BACKWARD);
    if (workspace_bytes < L.total) return INPC_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    return D == 4 ? backward_impl<4>(N, cam, grad_out_feat, grad_out_alpha, grad_feat, grad_opacity, grad_uv, blend_weight, ws, L, flags, grad_scale, st)
                  : backward_impl<8>(N, cam, grad_out_feat, grad_out_alpha, grad_feat, grad_opacity, grad_uv, blend_weight, ws, L, flags, grad_scale, st);
}

int inpc_raster_backward(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                         const inpc_camera* cam, const float* grad_out_feat, const float* grad_out_alpha,
                         float* grad_feat, float* grad_opacity, float* grad_uv, void* workspace,
                         size_t workspace_bytes, void* cuda_stream) {
    (void)pos; (void)opacity; (void)feat;   // the records saved by the forward hold what the backward needs
    return backward_entry(N, D, cam, grad_out_feat, grad_out_alpha, grad_feat, grad_opacity, grad_uv, nullptr, workspace,
                          workspace_bytes, 0u, 1.0f, cuda_stream);
}

int inpc_raster_backward_weights(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                                 const inpc_camera* cam, const float* grad_out_feat, const float* grad_out_alpha,
                                 float* grad_feat, float* grad_opacity, float* grad_uv, float* blend_weight,
                                 void* workspace, size_t workspace_bytes, void* cuda_stream) {
    (void)pos; (void)opacity; (void)feat;
    if (N > 0 && !blend_weight) return INPC_ERR_INVALID_ARG;
    return backward_entry(N, D, cam, grad_out_feat, grad_out_alpha, grad_feat, grad_opacity, grad_uv, blend_weight,
                          workspace, workspace_bytes, 0u, 1.0f, cuda_stream);
}

int inpc_raster_backward_ex(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                            const inpc_camera* cam, const float* grad_out_feat, const float* grad_out_alpha,
                            float* grad_feat, float* grad_opacity, float* grad_uv, float* blend_weight,
                            void* workspace, size_t workspace_bytes, uint32_t flags, float grad_scale, void* cuda_stream) {
    (void)pos; (void)opacity; (void)feat;
    return backward_entry(N, D, cam, grad_out_feat, grad_out_alpha, grad_feat, grad_opacity, grad_uv, blend_weight,
                          workspace, workspace_bytes, flags, grad_scale, cuda_stream);
}

// The introspection calls synchronise: they read the workspace's Header back and take shape, D and flags from it.
static int read_header(const void* workspace, int32_t W, int32_t H, cudaStream_t st, Header* h) {
    INPC_CUDA(cudaMemcpyAsync(h, workspace, sizeof(Header), cudaMemcpyDeviceToHost, st));
    INPC_CUDA(cudaStreamSynchronize(st));
    if (h->magic != kMagic) return INPC_ERR_NO_SAVED_STATE;
    if (W > 0 && (h->W != W || h->H != H)) return INPC_ERR_INVALID_ARG;
    return INPC_OK;
}

int inpc_raster_get_status(const void* workspace, void* cuda_stream) {
    if (!workspace) return INPC_ERR_INVALID_ARG;
    Header h;
    int rc = read_header(workspace, 0, 0, static_cast<cudaStream_t>(cuda_stream), &h);
    return rc != INPC_OK ? rc : h.status;
}

int inpc_raster_get_counts(const void* workspace, int32_t W, int32_t H, uint32_t* counts, void* cuda_stream) {
    if (!workspace || !counts || W <= 0 || H <= 0) return INPC_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Header h;
    int rc = read_header(workspace, W, H, st, &h);
    if (rc != INPC_OK) return rc;
    const Layout L = make_layout(h.n_points, h.D, h.W, h.H, h.flags);
    const unsigned char* ws = static_cast<const unsigned char*>(workspace);
    k_counts_out<<<(L.P + 255) / 256, 256, 0, st>>>(reinterpret_cast<const uint32_t*>(ws + L.cellcnt), W, H, counts);
    INPC_LAUNCHED("k_counts_out");
    return INPC_OK;
}

int inpc_raster_get_blended_counts(const void* workspace, int32_t W, int32_t H, uint32_t* blended, void* cuda_stream) {
    if (!workspace || !blended || W <= 0 || H <= 0) return INPC_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Header h;
    int rc = read_header(workspace, W, H, st, &h);
    if (rc != INPC_OK) return rc;
    if (!(h.flags & INPC_SAVE_FOR_BACKWARD)) return INPC_ERR_NO_SAVED_STATE;
    const Layout L = make_layout(h.n_points, h.D, h.W, h.H, h.flags);
    const unsigned char* ws = static_cast<const unsigned char*>(workspace);
    k_blended_out<<<(L.P + 255) / 256, 256, 0, st>>>(reinterpret_cast<const uint4*>(ws + L.pcur), L.P, blended);
    INPC_LAUNCHED("k_blended_out");
    return INPC_OK;
}

int inpc_raster_get_stats(const void* workspace, inpc_stats* stats, void* cuda_stream) {
    if (!workspace || !stats) return INPC_ERR_INVALID_ARG;
    Header h;
    int rc = read_header(workspace, 0, 0, static_cast<cudaStream_t>(cuda_stream), &h);
    if (rc != INPC_OK) return rc;
    stats->n_points = h.n_points;
    stats->n_kept = h.nrec;
    stats->n_fragments = h.n_fragments;
    stats->n_tile_items = 0;
    for (int b = 0; b < kMaxBands; ++b) stats->n_tile_items += h.band_items[b];
    stats->n_big_pixels = h.n_big_pixels;
    stats->n_big_fragments = h.n_big_fragments;
    stats->n_big_cells = h.n_big_cells;
    return INPC_OK;
}

int inpc_raster_get_sorted(const void* workspace, int32_t W, int32_t H, uint32_t* offsets, uint32_t* point_idx,
                           uint32_t* depth_bits, float* transmittance, uint64_t* total, void* cuda_stream) {
    if (!workspace || !total || W <= 0 || H <= 0) return INPC_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Header h;
    int rc = read_header(workspace, W, H, st, &h);
    if (rc != INPC_OK) return rc;
    if (!(h.flags & INPC_SAVE_SORTED)) return INPC_ERR_NO_SAVED_STATE;
    const Layout L = make_layout(h.n_points, h.D, h.W, h.H, h.flags);
    const unsigned char* ws = static_cast<const unsigned char*>(workspace);
    *total = h.n_fragments;
    if (!offsets) return INPC_OK;
    if (!point_idx || !depth_bits) return INPC_ERR_INVALID_ARG;
    INPC_CUDA(cudaMemcpyAsync(offsets, ws + L.pixoff, ((size_t)L.P + 1) * 4, cudaMemcpyDeviceToDevice, st));
    if (h.n_fragments) {
        INPC_CUDA(cudaMemcpyAsync(point_idx, ws + L.sorted_idx, (size_t)h.n_fragments * 4, cudaMemcpyDeviceToDevice, st));
        INPC_CUDA(cudaMemcpyAsync(depth_bits, ws + L.sorted_depth, (size_t)h.n_fragments * 4, cudaMemcpyDeviceToDevice, st));
        if (transmittance)
            INPC_CUDA(cudaMemcpyAsync(transmittance, ws + L.sorted_T, (size_t)h.n_fragments * 4, cudaMemcpyDeviceToDevice, st));
    }
    INPC_CUDA(cudaStreamSynchronize(st));
    return INPC_OK;
}

// ---- NEXT row f4: view-specific sampling (sampler.cuh) ---------------------------------------------------------------
struct SampleLayout { size_t head, phat, cdf, tiles, guide, total; uint32_t n_tiles; };
static SampleLayout sample_layout(int64_t L) {
    SampleLayout S{};
    S.n_tiles = (uint32_t)((L + kScan64Tile - 1) / kScan64Tile);
    size_t o = 0;
    S.head = o;  o = align_up(o + 64);                       // max_bits, total, n_valid
    S.phat = o;  o = align_up(o + (size_t)L * 8);
    S.cdf = o;   o = align_up(o + (size_t)L * 8);
    S.tiles = o; o = align_up(o + ((size_t)S.n_tiles + 1) * 8);
    S.guide = o; o = align_up(o + ((size_t)kGuide + 1) * 4);   // guide table of the inverse CDF (sampler.cuh)
    S.total = o;
    return S;
}

size_t inpc_sample_workspace_bytes(int64_t n_leaves) {
    if (n_leaves < 1 || n_leaves > (1ll << 24)) return 0;
    return sample_layout(n_leaves).total;
}

static int sample_view_impl(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                            float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                            void* workspace, size_t workspace_bytes, uint32_t flags, void* cuda_stream) {
    if (flags & ~INPC_SAMPLE_NO_RESAMPLE) return INPC_ERR_INVALID_ARG;
    if (!cam || !leaf_centre || !leaf_level || !leaf_prob || !workspace || N < 0 || N >= (1ll << 31)) return INPC_ERR_INVALID_ARG;
    if (n_leaves < 1 || n_leaves > (1ll << 24) || !(root_side > 0.f)) return INPC_ERR_INVALID_ARG;
    if (cam->width <= 0 || cam->height <= 0 || !(cam->near_z < cam->far_z)) return INPC_ERR_INVALID_ARG;
    if (!(cam->near_z >= 0.f)) return INPC_ERR_INVALID_ARG;      // the camera rule of check_common: the rasterizer refuses it too
    if (N > 0 && (!pos || !leaf)) return INPC_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(workspace) & 255u) return INPC_ERR_INVALID_ARG;
    const SampleLayout S = sample_layout(n_leaves);
    if (workspace_bytes < S.total) return INPC_ERR_WORKSPACE_TOO_SMALL;
    const DeviceInfo di = device_info();
    if (!di.ok) return cuda_fail(cudaErrorNoDevice);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    unsigned long long* head = reinterpret_cast<unsigned long long*>(ws + S.head);
    double* phat = reinterpret_cast<double*>(ws + S.phat);
    unsigned long long* cdf = reinterpret_cast<unsigned long long*>(ws + S.cdf);
    unsigned long long* tiles = reinterpret_cast<unsigned long long*>(ws + S.tiles);
    uint32_t* guide = reinterpret_cast<uint32_t*>(ws + S.guide);
    const Camera camk = to_camera(cam);
    const uint32_t L = (uint32_t)n_leaves;
    INPC_CUDA(cudaMemsetAsync(head, 0, 64, st));
    k_leaf_weight<<<std::min<uint32_t>((L + 255) / 256, (uint32_t)di.sms * 8), 256, 0, st>>>(leaf_centre, leaf_level, leaf_prob, L,
                                                                                            root_side, camk, phat, head);
    INPC_LAUNCHED("k_leaf_weight");
    k_cdf_local<<<S.n_tiles, kScan64Threads, 0, st>>>(phat, L, head, cdf, tiles);
    INPC_LAUNCHED("k_cdf_local");
    k_cdf_tiles<<<1, 1024, 0, st>>>(tiles, S.n_tiles, head + 1);
    INPC_LAUNCHED("k_cdf_tiles");
    k_cdf_add<<<S.n_tiles, kScan64Threads, 0, st>>>(cdf, L, tiles);
    INPC_LAUNCHED("k_cdf_add");
    if (N > 0) {
        k_cdf_guide<<<kGuide / 256 + 1, 256, 0, st>>>(cdf, L, head + 1, guide);
        INPC_LAUNCHED("k_cdf_guide");
        k_sample<<<(int)std::min<int64_t>((N + 255) / 256, (int64_t)di.sms * 8), 256, 0, st>>>(
            cdf, L, head + 1, leaf_centre, leaf_level, root_side, camk, (unsigned long long)seed, (long long)N, pos, leaf, head + 2,
            (flags & INPC_SAMPLE_NO_RESAMPLE) ? 1 : kSampleAttempts, guide);
        INPC_LAUNCHED("k_sample");
    }
    return INPC_OK;
}

int inpc_sample_view(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                     float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                     void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return sample_view_impl(leaf_centre, leaf_level, leaf_prob, n_leaves, root_side, cam, seed, N, pos, leaf, workspace,
                            workspace_bytes, 0u, cuda_stream);
}

int inpc_sample_view_ex(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                        float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                        void* workspace, size_t workspace_bytes, uint32_t flags, void* cuda_stream) {
    return sample_view_impl(leaf_centre, leaf_level, leaf_prob, n_leaves, root_side, cam, seed, N, pos, leaf, workspace,
                            workspace_bytes, flags, cuda_stream);
}

// ---- inpc_sample_view for callers that cannot allocate device memory ------------------------------------------------
// Some users of the sampler have no way to obtain a workspace: a renderer plugin running inside a host application
// that has handed the whole GPU to its own memory pool, a real-time loop in which cudaMalloc's implicit device-wide
// synchronisation is forbidden, code that runs after the process has hit its memory budget.  For them the sampler's
// scratch (p^, the integer CDF, the tile sums, the guide table and the three statistics words: 16 bytes per leaf plus
// 258 KB) is carved out of the library image itself: the array below is part of the module, so every device that loads
// the library pays its 4.25 MiB from the moment the module is loaded until the process exits, whether or not this entry point is ever used.
//
// g_sample_scratch is a DEVICE symbol.  The name, used in host code, is only the host-side shadow the runtime keeps
// for it -- not an address a kernel may dereference -- so the device address is looked up per device with
// cudaGetSymbolAddress (each device has its own copy of the array) and it is that address the kernels are given.
constexpr int64_t kStaticSampleMaxLeaves = 1ll << 18;
constexpr size_t kStaticSampleBytes =       // sample_layout(kStaticSampleMaxLeaves).total, spelled out so that it is a constant
    256 + 2 * (size_t)kStaticSampleMaxLeaves * 8 + ((kStaticSampleMaxLeaves / kScan64Tile + 1) * 8 + 255) / 256 * 256 +
    (((size_t)kGuide + 1) * 4 + 255) / 256 * 256;
static __device__ __align__(256) unsigned char g_sample_scratch[kStaticSampleBytes];

static void* static_sample_scratch(const DeviceInfo& di, cudaError_t* err) {
    static void* ptr_by_dev[kMaxDevices] = {};
    std::lock_guard<std::mutex> lk(g_dev_mu);
    if (!ptr_by_dev[di.dev]) {                    // first call on this device (it is the current one: device_info() read it)
        void* p = nullptr;
        *err = cudaGetSymbolAddress(&p, g_sample_scratch);
        if (*err != cudaSuccess) return nullptr;
        ptr_by_dev[di.dev] = p;
    }
    return ptr_by_dev[di.dev];
}

int64_t inpc_sample_static_max_leaves(void) { return kStaticSampleMaxLeaves; }

int inpc_sample_view_static(const float* leaf_centre, const int32_t* leaf_level, const float* leaf_prob, int64_t n_leaves,
                            float root_side, const inpc_camera* cam, uint64_t seed, int64_t N, float* pos, int32_t* leaf,
                            void* cuda_stream) {
    if (n_leaves > kStaticSampleMaxLeaves) return INPC_ERR_STATIC_LIMIT;
    if (n_leaves >= 1 && sample_layout(n_leaves).total > sizeof(g_sample_scratch)) return INPC_ERR_STATIC_LIMIT;
    const DeviceInfo di = device_info();
    if (!di.ok) return cuda_fail(cudaErrorNoDevice);
    cudaError_t e = cudaSuccess;
    void* scratch = static_sample_scratch(di, &e);
    if (!scratch) return cuda_fail(e);
    // From here on this IS inpc_sample_view, with the library's array as its workspace: same kernels, same argument
    // checks, same results.  It clears the statistics words itself and overwrites every other byte it later reads, so
    // what an earlier call left in the array does not matter.
    return inpc_sample_view(leaf_centre, leaf_level, leaf_prob, n_leaves, root_side, cam, seed, N, pos, leaf, scratch,
                            sizeof(g_sample_scratch), cuda_stream);
}

int inpc_sample_get_stats(const void* workspace, uint64_t* n_valid, uint64_t* cdf_total, double* max_weight, void* cuda_stream) {
    if (!workspace) return INPC_ERR_INVALID_ARG;
    unsigned long long h[3];
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    INPC_CUDA(cudaMemcpyAsync(h, workspace, sizeof(h), cudaMemcpyDeviceToHost, st));
    INPC_CUDA(cudaStreamSynchronize(st));
    if (max_weight) { double m; std::memcpy(&m, &h[0], 8); *max_weight = m; }
    if (cdf_total) *cdf_total = h[1];
    if (n_valid) *n_valid = h[2];
    return INPC_OK;
}

const char* inpc_raster_strerror(int status) {
    switch (status) {
        case INPC_OK: return "ok";
        case INPC_ERR_INVALID_ARG: return "invalid argument";
        case INPC_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
        case INPC_ERR_CUDA: return "CUDA error (see inpc_raster_last_cuda_error)";
        case INPC_ERR_NO_SAVED_STATE: return "workspace holds no matching forward state";
        case INPC_ERR_UNSUPPORTED: return "unsupported D or image size";
        case INPC_ERR_STATIC_LIMIT: return "more leaves than inpc_sample_view_static's built-in scratch holds (see inpc_sample_static_max_leaves)";
        default: return "unknown status";
    }
}

int inpc_raster_set_kernel_timing(int enable) {
    std::lock_guard<std::mutex> lk(g_tmu);
    g_timing = enable != 0;
    return INPC_OK;
}

int inpc_raster_kernel_count(void) { return kNumStages; }

const char* inpc_raster_kernel_name(int i) { return (i >= 0 && i < kNumStages) ? kStageNames[i] : ""; }

int inpc_raster_get_kernel_times(double* ms, uint64_t* launches, int reset) {
    if (!ms || !launches) return INPC_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lk(g_tmu);
    for (const Pending& p : g_pending) {
        cudaError_t e = cudaEventSynchronize(p.b);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, p.a, p.b);
        if (e != cudaSuccess) { g_pending.clear(); return cuda_fail(e); }
        g_stage_ms[p.stage] += (double)t;
        g_stage_n[p.stage] += 1;
        g_event_pool.push_back(p.a);
        g_event_pool.push_back(p.b);
    }
    g_pending.clear();
    for (int i = 0; i < kNumStages; ++i) {
        ms[i] = g_stage_ms[i]; launches[i] = g_stage_n[i];
        if (reset) { g_stage_ms[i] = 0.0; g_stage_n[i] = 0; }
    }
    return INPC_OK;
}

const char* inpc_raster_last_cuda_error(void) { return t_cuda_error.c_str(); }

uint64_t inpc_raster_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

size_t inpc_raster_launched_kernels(char* buf, size_t buf_bytes, int reset) {
    std::lock_guard<std::mutex> lk(g_names_mu);
    std::string all;
    for (const std::string& n : g_names) { if (!all.empty()) all += ";"; all += n; }
    if (reset) g_names.clear();
    if (buf && buf_bytes) {
        const size_t k = std::min(buf_bytes - 1, all.size());
        std::memcpy(buf, all.data(), k);
        buf[k] = 0;
    }
    return all.size() + 1;
}

}  // extern "C"
