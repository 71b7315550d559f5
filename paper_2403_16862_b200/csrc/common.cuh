// common.cuh -- shared device/host definitions of the rasterizer kernels (sm_100a only).
//
// Data layout in HBM (all inside the caller's workspace):
//   cell grid   : (W+1) x (H+1) cells; cell (i, j) holds the kept points whose top-left pixel is
//                 (x0, y0) = (i-1, j-1), x0 = floor(u-0.5).  Pixel (x, y) receives exactly the points of
//                 cells (x, y), (x+1, y), (x, y+1), (x+1, y+1)  => its fragments are FOUR cell lists, two
//                 contiguous slot ranges of the cell-ordered arrays (cell rows y and y+1).
//   celloff[C+1]: exclusive sum of the per-cell point counts (device-wide scan), C = (W+1)(H+1).
//   A[nrec]     : 32-byte emission records in arrival order inside each cell (written by k_scatter):
//                 { depth_bits, point_idx, tx, ty | opacity, cell, 0, 0 }   (tx = fu - x0, ty = fv - y0, exact)
//   dk[nrec]    : depth bits, every cell sorted ascending by (depth_bits, point_idx)   (k_cellsort)
//   Ra[nrec]    : { tx, ty, opacity, point_idx } in the same order (16 B; staged by the tile kernels and turned
//                 into the four per-corner alphas in shared memory), Rf[nrec] : feat[D] in the same order
//   kept[N/32]  : 1 bit per point = survived the cull; cursor[C] : copy of celloff the scatter hands slots out of
//   Because every cell list is sorted, a pixel's depth-ordered fragment run is the 4-way MERGE of its
//   four cell lists; no per-pixel sort exists anywhere.
//   gT[4*nrec]  : transmittance in front of fragment (slot, corner), written by the forward pass
//   gD[4*nrec]  : dL/da of fragment (slot, corner), written by the backward pass   (gT|gD reuse A's bytes)
//   pcur[P]     : per pixel, how many records of each of its four lists were blended before the cut-off
//   ord[], ordinfo[items] : the blend order the forward pass took, 16 bits per fragment (record * 16 + 4 * corner,
//                 tile-local), one block per tile item; ordinfo[item] = { first entry, entries }   (blend.cuh, back.cuh)
//   gpt[N]      : per-point gradient records (8 or 16 floats), one or two full 32-byte sectors each
// Corner c = 2*dy + dx is the pixel's offset from the record's top-left pixel; list j of a pixel
// (0: cell (x,y), 1: (x+1,y), 2: (x,y+1), 3: (x+1,y+1)) holds its fragments of corner 3 - j.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace inpc {

// ---- tunables -------------------------------------------------------------------------------------
#ifndef INPC_TILE_LW
#define INPC_TILE_LW 4
#endif
#ifndef INPC_CAP4
#define INPC_CAP4 1216
#endif
#ifndef INPC_CAP8
#define INPC_CAP8 1024
#endif
constexpr int kTileLW      = INPC_TILE_LW;     // log2(kTileW)
constexpr int kTileW       = 1 << kTileLW;    // base screen tile (pixels); halved (larger side first) down to kMinTilePix
constexpr int kTileH       = 8;
constexpr int kTileLH      = 3;     // log2(kTileH)
constexpr int kTileThreads = kTileW * kTileH;   // one thread per pixel
constexpr int kMinTilePix  = 8;     // a sub-tile this small that misses the capacity by more than 2x goes to the long-run path
constexpr int kCellSmall   = 256;   // cells up to this many points are ranked by counting; larger: bitonic
constexpr int kBigThreads  = 512;
constexpr int kBigChunk    = 8192;  // keys sorted in shared memory at a time by the large-cell sort
constexpr int kMaxBands    = 8;     // bands of tile rows the forward / backward pipelines overlap (see inpc_raster.cu)
constexpr float kTMin      = 1e-4f; // transmittance cut-off (BASELINE.json north_star)
constexpr uint32_t kSentHi = 0xFFFFFFFFu;   // "list exhausted" for the ascending merge (depth bits < 0x7F800000)

template <int D> struct TileCfg;
template <> struct TileCfg<4> { static constexpr int kCap = INPC_CAP4; };   // records per tile item
template <> struct TileCfg<8> { static constexpr int kCap = INPC_CAP8; };
// The merge kernels keep a list cursor as a 16-bit byte offset "record * 16 + 4 * corner" (pack_list, the entries of
// ord[], the (nx >> 2) & 0x3ffc mask), and stage records four at a time: INPC_CAP4 / INPC_CAP8 are build-time overridable,
// so the limits are checked here.
constexpr size_t kMaxSmemPerCta = 227 * 1024;    // sm_100a opt-in dynamic shared memory per CTA
static_assert(TileCfg<4>::kCap % 4 == 0 && TileCfg<4>::kCap * 16 <= 65536, "INPC_CAP4: a multiple of 4, at most 4096 records");
static_assert(TileCfg<8>::kCap % 4 == 0 && TileCfg<8>::kCap * 16 <= 65536, "INPC_CAP8: a multiple of 4, at most 4096 records");

struct Camera {
    float fx, fy, cx, cy;
    float R[9], t[3];
    float near_z, far_z;
    int32_t W, H;
};

// Device-resident header at the start of the workspace.
struct Header {
    uint32_t magic;
    uint32_t flags;
    int32_t  W, H, D;
    uint32_t n_points;
    uint32_t nrec;                 // kept points (= celloff[C]), written by the scan
    uint32_t n_items;              // (unused; the tile work items are counted per band, below)
    uint32_t item_cursor;
    uint32_t big_cursor;
    uint32_t scan_tile_counter;
    uint32_t pad0;
    unsigned long long n_fragments;
    uint32_t n_big_pixels;         // pixels routed to the long-run path
    uint32_t n_big_cells;          // cells larger than kCellSmall (bitonic-sorted)
    unsigned long long n_big_fragments;
    uint32_t bigcell_cursor;
    uint32_t bigcell_keys;         // running offset into the large-cell key scratch
    uint32_t cellsort_cursor;
    uint32_t bwd_ok;               // written by the backward pass's header check: 1 = the workspace matches its arguments
    int32_t  status;               // sticky inpc_status of device-side checks (read by inpc_raster_get_status)
    uint32_t ord_cursor;           // bump allocator of the per-tile blocks of the saved blend order (entries)
    uint32_t combine_cursor;       // work cursor of k_combine (reset by the backward pass's header check)
    uint32_t combine_q_head, combine_q_tail, combine_done;   // queue of the parts of large units (k_combine)
    uint32_t pad[4];
    // Tile work items, one list per BAND of tile rows (kMaxBands bands): a band's tiles can be blended as soon as
    // its cell rows are sorted, while the next band's cells are still being sorted on another stream.
    uint32_t band_items[8];        // items of band b
    uint32_t band_cursor[8];       // persistent-kernel work cursor of band b (forward, then backward)
};
static_assert(sizeof(Header) % 16 == 0, "header alignment");

struct BigCell { uint32_t cell, start, n, pad; };   // a cell with more than kCellSmall points

constexpr uint32_t kMagic = 0x494E5043u;  // "INPC"

// ---- small PTX helpers -----------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// Shared-memory loads through 32-bit shared-window addresses: the merge loops address their records with plain
// integer arithmetic (a generic pointer costs a window-base rematerialisation per access inside the loop).
__device__ __forceinline__ float lds_f32(uint32_t a) {
    float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t a) {
    uint16_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a)); return v;
}
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v) : "memory");
}
__device__ __forceinline__ float4 lds_v4(uint32_t a) {
    float4 v; asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a)); return v;
}
// One 256-bit store: a whole 32-byte sector in ONE instruction.  A lane-divergent store costs L1 wavefronts
// per instruction, so two 128-bit stores to the same sector cost twice (k_scatter 222 -> 173 us).
__device__ __forceinline__ void st_sector(void* p, float4 lo, float4 hi) {
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(lo.x), "f"(lo.y), "f"(lo.z),
                 "f"(lo.w), "f"(hi.x), "f"(hi.y), "f"(hi.z), "f"(hi.w)
                 : "memory");
}
// TMA bulk copy global -> shared (1-D, no tensor map): 16-byte aligned src/dst, size multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// TMA bulk copy shared -> global (1-D): same alignment rules; completion is tracked per thread by bulk groups.
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read() {        // the issuing thread's bulk stores have finished READING shared memory
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ---- step a1: canonical fp32 projection (Eq. 6; reading R1) ------------
// Every operation is one IEEE fp32 operation (_rn intrinsics are never contracted to FMA), in the
// order the specification fixes.  Used by BOTH the count pass and the scatter pass so they agree.
struct Proj {
    float    tx, ty;       // fractional position inside the cell, in [0,1)
    uint32_t depth_bits;   // raw bits of z_c (> 0 => unsigned order = numeric order)
    int32_t  cell;         // j * (W+1) + i, or -1 when culled
};
__device__ __forceinline__ Proj project_point(const Camera& c, float x, float y, float z) {
    Proj p;
    p.cell = -1; p.tx = 0.f; p.ty = 0.f; p.depth_bits = 0;
    const float xc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[0], x), __fmul_rn(c.R[1], y)), __fmul_rn(c.R[2], z)), c.t[0]);
    const float yc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[3], x), __fmul_rn(c.R[4], y)), __fmul_rn(c.R[5], z)), c.t[1]);
    const float zc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[6], x), __fmul_rn(c.R[7], y)), __fmul_rn(c.R[8], z)), c.t[2]);
    if (!(zc > c.near_z && zc < c.far_z)) return p;                     // strict; false for NaN
    const float u = __fadd_rn(__fdiv_rn(__fmul_rn(c.fx, xc), zc), c.cx);
    const float v = __fadd_rn(__fdiv_rn(__fmul_rn(c.fy, yc), zc), c.cy);
    const float inf = __int_as_float(0x7f800000);
    if (!(fabsf(u) < inf) || !(fabsf(v) < inf)) return p;               // non-finite => culled
    const float fu = __fsub_rn(u, 0.5f), fv = __fsub_rn(v, 0.5f);
    const float x0 = floorf(fu), y0 = floorf(fv);
    if (!(x0 >= -1.0f && x0 <= (float)(c.W - 1) && y0 >= -1.0f && y0 <= (float)(c.H - 1))) return p;
    p.tx = __fsub_rn(fu, x0);                                            // exact
    p.ty = __fsub_rn(fv, y0);
    p.depth_bits = __float_as_uint(zc);
    p.cell = ((int)y0 + 1) * (c.W + 1) + ((int)x0 + 1);
    return p;
}

// ---- how a feature image (forward) or its gradient (backward) is laid out and combined (NEXT row f3) ------------
// planar 0: [H][W][D] pixel-interleaved (one 16-byte store per pixel and four channels); 1: [D][H][W], what a CNN
// wants.  Forward: out = (accumulate ? out : 0) + scale * result -- the per-pixel average of several
// point clouds ("multisampling") is S calls with scale 1/S.  Backward: grad_out is read through the same
// layout and multiplied by scale.  scale = 1 and accumulate = 0 reproduce the plain result bit for bit.
struct ImageIO {
    int planar, accumulate;
    float scale;
    uint32_t P;                // W * H
};
template <int D>
__device__ __forceinline__ void store_pixel(const ImageIO& io, float* __restrict__ out_feat, float* __restrict__ out_alpha,
                                            size_t pix, const float (&acc)[D], float accA) {
    if (!io.planar) {
        float4* o = reinterpret_cast<float4*>(out_feat + pix * D);
#pragma unroll
        for (int v = 0; v < D / 4; ++v) {
            float4 r = make_float4(io.scale * acc[4 * v], io.scale * acc[4 * v + 1], io.scale * acc[4 * v + 2], io.scale * acc[4 * v + 3]);
            if (io.accumulate) { const float4 b = o[v]; r.x += b.x; r.y += b.y; r.z += b.z; r.w += b.w; }
            o[v] = r;
        }
    } else {
#pragma unroll
        for (int d = 0; d < D; ++d) {
            float* o = out_feat + (size_t)d * io.P + pix;
            float r = io.scale * acc[d];
            if (io.accumulate) r += *o;
            *o = r;
        }
    }
    float a = io.scale * accA;
    if (io.accumulate) a += out_alpha[pix];
    out_alpha[pix] = a;
}
template <int D>
__device__ __forceinline__ void load_pixel_grad(const ImageIO& io, const float* __restrict__ g_feat,
                                                const float* __restrict__ g_alpha, size_t pix, float (&g)[D], float& gA) {
    if (!io.planar) {
#pragma unroll
        for (int v = 0; v < D / 4; ++v) {
            const float4 t = __ldg(reinterpret_cast<const float4*>(g_feat + pix * D) + v);
            g[4 * v] = io.scale * t.x; g[4 * v + 1] = io.scale * t.y; g[4 * v + 2] = io.scale * t.z; g[4 * v + 3] = io.scale * t.w;
        }
    } else {
#pragma unroll
        for (int d = 0; d < D; ++d) g[d] = io.scale * __ldg(g_feat + (size_t)d * io.P + pix);
    }
    gA = g_alpha ? io.scale * __ldg(g_alpha + pix) : 0.f;
}

// Work-item encoding for the tile kernel: X (12 bits) | Y (12) | log2 tw (3) | log2 th (2)
__host__ __device__ __forceinline__ uint32_t encode_item(int X, int Y, int lw, int lh) {
    return (uint32_t)X | ((uint32_t)Y << 12) | ((uint32_t)lw << 24) | ((uint32_t)lh << 27);
}

}  // namespace inpc
