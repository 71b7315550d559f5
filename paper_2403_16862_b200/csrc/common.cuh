// common.cuh -- shared device/host definitions of the rasterizer kernels (sm_100a only).
//
// Data layout in HBM (all inside the caller's workspace):
//   cell grid   : (W+1) x (H+1) cells; cell (i, j) holds the kept points whose top-left pixel is
//                 (x0, y0) = (i-1, j-1), x0 = floor(u-0.5).  Pixel (x, y) receives exactly the points of
//                 cells (x, y), (x+1, y), (x, y+1), (x+1, y+1)  => its fragment run is two contiguous
//                 record ranges of the cell-sorted record array (cell rows y and y+1).
//   celloff[C+1]: exclusive sum of the per-cell point counts (device-wide scan), C = (W+1)(H+1).
//   rec[nrec]   : cell-sorted point records, RB = 16 + 4*D bytes each:
//                 { depth_bits, point_idx, tx, ty, feat[0..D) }  (tx = fu - x0, ty = fv - y0, exact)
//   rop[nrec]   : opacity of each record (separate 4-byte array so that rec stays 16-byte granular).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace inpc {

// ---- tunables -------------------------------------------------------------------------------------
constexpr int kTileW      = 16;    // base screen tile (pixels); halved alternately down to 1x1
constexpr int kTileH      = 8;
constexpr int kTileLW     = 4;     // log2(kTileW)
constexpr int kTileLH     = 3;     // log2(kTileH)
constexpr int kTileThreads = 256;
constexpr int kTileWarps  = kTileThreads / 32;
constexpr int kPixMax     = 256;   // deepest pixel the tile kernel sorts itself (per-warp smem scratch)
constexpr int kBigThreads = 512;
constexpr int kBigChunk   = 8192;  // keys sorted in shared memory at a time by the long-run path
constexpr float kTMin     = 1e-4f; // transmittance cut-off (BASELINE.json north_star)

template <int D> struct TileCfg;
template <> struct TileCfg<4> { static constexpr int kCap = 1600; };   // records per tile item
template <> struct TileCfg<8> { static constexpr int kCap = 1280; };

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
    uint32_t n_items;              // tile work items
    uint32_t item_cursor;          // persistent-kernel work cursors
    uint32_t big_cursor;
    uint32_t scan_tile_counter;
    uint32_t pad0;
    unsigned long long n_fragments;
    unsigned long long big_packed; // (n_big << 40) | n_big_fragments, bumped with one atomic
    uint32_t pad[16];
};
static_assert(sizeof(Header) % 16 == 0, "header alignment");

struct BigEntry {                  // one pixel deeper than kPixMax
    uint32_t pix;                  // y * W + x
    uint32_t n;                    // fragments
    uint32_t start;                // offset of its run in bigkeys
    uint32_t nb;                   // blended count (written by the forward)
    uint32_t tin_base;             // offset of its per-chunk incoming transmittances in bigtin
    uint32_t pad[3];
};

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
// TMA bulk copy global -> shared (1-D, no tensor map): 16-byte aligned src/dst, size multiple of 16.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d)
                 : "memory");
}
__device__ __forceinline__ void red_add_v2(float* addr, float a, float b) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" ::"l"(addr), "f"(a), "f"(b) : "memory");
}
__device__ __forceinline__ void red_add(float* addr, float a) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(a) : "memory");
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

// Work-item encoding for the tile kernel: X (12 bits) | Y (12) | log2 tw (3) | log2 th (2)
__host__ __device__ __forceinline__ uint32_t encode_item(int X, int Y, int lw, int lh) {
    return (uint32_t)X | ((uint32_t)Y << 12) | ((uint32_t)lw << 24) | ((uint32_t)lh << 27);
}

}  // namespace inpc
