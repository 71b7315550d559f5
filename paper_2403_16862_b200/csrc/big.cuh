// big.cuh -- the long-run path: pixels whose neighbourhood does not fit a shared-memory tile even at
// kMinTilePix pixels (depth-complexity stress, BASELINE.json config 5: tens of thousands of fragments in
// one pixel).  Their cell lists are already sorted (cellsort.cuh), so the pixel is the same 4-way merge
// as in the tile kernel, read straight from global memory: one thread per pixel, double-precision
// transmittance and backward carry (an fp32 product of > 10^4 factors drifts past the 1e-5 gradient
// floor).  The cut-off T < 1e-4 ends the walk long before a deep list is exhausted,
// so only the front of each list is ever touched.
#pragma once
#include "common.cuh"
#include "tile.cuh"

namespace inpc {

constexpr int kLongThreads = 64;

struct BigArgs {
    const Header* hdr;
    const uint32_t* bigpix;
    const uint32_t* celloff;
    const uint32_t* dk;
    const float4* Ra;
    const float4* Rf;
    int W, H;
    float* out_feat;
    float* out_alpha;
    float* gT;
    uint4* pcur;
    const uint32_t* pixoff;
    uint32_t* sorted_idx;
    uint32_t* sorted_depth;
    float* sorted_T;
    const float* g_feat;
    const float* g_alpha;
    float* gD;
    ImageIO io;
};

template <int D, int MODE>
__global__ void __launch_bounds__(kLongThreads) k_big(BigArgs A) {
    if (MODE == kBwd && !A.hdr->bwd_ok) return;          // backward on a workspace that holds no matching forward
    const uint32_t n_big = A.hdr->n_big_pixels;
    const int W = A.W;
    for (uint32_t b = blockIdx.x * kLongThreads + threadIdx.x; b < n_big; b += gridDim.x * kLongThreads) {
        const uint32_t pix = A.bigpix[b];
        const int y = pix / W, x = pix - y * W;
        const uint32_t r0 = (uint32_t)y * (W + 1) + x, r1 = r0 + (W + 1);
        PixLists L;
        L.c0 = __ldg(&A.celloff[r0]); L.e0 = __ldg(&A.celloff[r0 + 1]); L.c1 = L.e0; L.e1 = __ldg(&A.celloff[r0 + 2]);
        L.c2 = __ldg(&A.celloff[r1]); L.e2 = __ldg(&A.celloff[r1 + 1]); L.c3 = L.e2; L.e3 = __ldg(&A.celloff[r1 + 2]);
        if (MODE != kBwd) {
            float acc[D]; float accA;
            uint4 consumed = make_uint4(0, 0, 0, 0);
            const uint32_t obase = (MODE == kFwdDump) ? A.pixoff[pix] : 0u;
            blend_pixel<D, MODE == kFwdDump, double>(A.dk, A.Ra, A.Rf, L, 0u, 0u, A.gT, acc, accA, consumed, A.sorted_idx,
                                                     A.sorted_depth, A.sorted_T, obase);
            store_pixel<D>(A.io, A.out_feat, A.out_alpha, (size_t)pix, acc, accA);
            if (A.gT) A.pcur[pix] = consumed;
        } else {
            const uint4 consumed = A.pcur[pix];
            L.e0 = L.c0 + consumed.x; L.e1 = L.c1 + consumed.y; L.e2 = L.c2 + consumed.z; L.e3 = L.c3 + consumed.w;
            float g[D], gA;
            load_pixel_grad<D>(A.io, A.g_feat, A.g_alpha, (size_t)pix, g, gA);
            backward_pixel<D, double>(A.dk, A.Ra, A.Rf, A.gT, L, 0u, 0u, g, gA, A.gD);
        }
    }
}

}  // namespace inpc
