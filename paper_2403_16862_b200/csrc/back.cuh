// back.cuh -- step a5 of the hot path, first half: the reverse traversal of every pixel's blended fragments
// ("process them in the same order as in the forward pass" -- here backwards through it).
//
// Same persistent tile kernel shape as blend.cuh: one work item = a screen tile whose records fit shared memory,
// staged exactly as the forward pass staged it (same cell rows, same 4-record alignment => the same shared-memory
// record indices), with cp.async.bulk onto one mbarrier: per record the { tx, ty, opacity, idx } word (turned into
// the four per-corner alphas in place), the features and the four transmittances gT the forward pass saved.
// The depth order is NOT merged again: the forward pass left, for every pixel, the list of (record, corner) it
// blended, in order (ord, 16 bits per fragment, blend.cuh); a tile's lists are th contiguous runs of that array
// and are staged with the same bulk copies.  ONE THREAD PER PIXEL (lanes in descending order of the blended
// count) walks its list from the last blended fragment to the first with the division-free recurrence
//     dL/da_k = T_k (G_k - B_k),    B_{k-1} = a_k G_k + (1 - a_k) B_k,    G_k = <feat_k, g_img[p]> + g_alpha[p]
// and writes dL/da_k to gD[(slot, corner)]; grad.cuh combines the four corners of every record.  No address in
// the loop depends on the recurrence, so the loads of four fragments are issued together and the only dependent
// chain is B.
#pragma once
#include "common.cuh"

namespace inpc {

struct BackArgs {
    const Header* hdr;
    uint32_t* item_cursor;   // this band's work cursor ...
    const uint32_t* n_items; // ... and item count (device)
    const uint32_t* items;
    const uint32_t* celloff;
    const float4* Ra;
    const float4* Rf;
    int W, H;
    const float* gT;
    const uint4* pcur;
    const uint32_t* pixoff;  // start of every pixel's order list
    const uint16_t* ord;     // (record * 16 + 4 * corner) of the k-th blended fragment, tile-local (forward pass)
    const float* g_feat;
    const float* g_alpha;
    ImageIO io;
    float* gD;
};

constexpr int kOrdPad = 8 * 2 * kTileH;      // entries: every tile row's run is widened to 16-byte boundaries at both ends

template <int D> __host__ __device__ constexpr size_t back_smem_bytes() {
    return (size_t)TileCfg<D>::kCap * (16 + 4 * D + 16 + 8) + 2 * kOrdPad;     // alphas, features, gT, order lists
}

template <int D>
__global__ void __launch_bounds__(kTileThreads, 3) k_back(BackArgs A) {
    constexpr int FV  = D / 4;
    constexpr int CAP = TileCfg<D>::kCap;
    extern __shared__ __align__(128) unsigned char smem[];
    float4*   s_a4  = reinterpret_cast<float4*>(smem);
    float4*   s_f   = reinterpret_cast<float4*>(smem + (size_t)CAP * 16);
    float4*   s_t4  = reinterpret_cast<float4*>(smem + (size_t)CAP * (16 + 16 * FV));
    uint16_t* s_ord = reinterpret_cast<uint16_t*>(smem + (size_t)CAP * (32 + 16 * FV));

    __shared__ uint32_t s_off[kTileH + 1][kTileW + 2];
    __shared__ uint32_t s_sbase[kTileH + 1], s_a4row[kTileH + 1];
    __shared__ uint32_t s_rowblk[kTileH], s_rowg[kTileH];     // order-list run of pixel row r: smem entry s_rowblk[r] <-> global entry s_rowg[r]
    __shared__ uint32_t s_hist[64];
    __shared__ uint32_t s_pixbase[kTileThreads];
    __shared__ uint8_t  s_perm[kTileThreads];
    __shared__ uint32_t s_next, s_next_code, s_tot;
    __shared__ __align__(8) uint64_t s_bar;

    const int tid = threadIdx.x;
    const int W = A.W, H = A.H;
    if (!A.hdr->bwd_ok) return;                          // the header check failed: touch nothing
    const uint32_t n_items = *A.n_items;

    if (tid == 0) {
        mbar_init(&s_bar, 1); fence_mbar_init();
        const uint32_t nx = atomicAdd(A.item_cursor, 1u);
        s_next = nx; s_next_code = nx < n_items ? A.items[nx] : 0u;
    }
    uint32_t parity = 0;

    while (true) {
        __syncthreads();                                  // everyone is done with the previous item's smem
        const uint32_t item_i = s_next;
        if (item_i >= n_items) break;
        const uint32_t it = s_next_code;
        const int X = it & 0xfff, Y = (it >> 12) & 0xfff, lw = (it >> 24) & 7, lh = (it >> 27) & 3;
        const int tw = 1 << lw, th = 1 << lh;

        // this thread's pixel in natural order: its blended count and the start of its order list (loads in flight early)
        const int ly0 = tid >> lw, lx0 = tid & (tw - 1);
        const bool live0 = tid < tw * th && X + lx0 < W && Y + ly0 < H;
        uint32_t n_mine = 0, po_mine = 0;
        if (live0) {
            const size_t p0 = (size_t)(Y + ly0) * W + X + lx0;
            const uint4 cn = __ldg(&A.pcur[p0]);
            n_mine = cn.x + cn.y + cn.z + cn.w;
            po_mine = __ldg(&A.pixoff[p0]);
        }
        // cell offsets of the tile's (th+1) x (tw+2) window
        for (int e = tid; e < (th + 1) * (tw + 2); e += kTileThreads) {
            const int r = e / (tw + 2), c = e - r * (tw + 2);
            const int j = Y + r;
            uint32_t v = 0;
            if (j <= H) v = __ldg(&A.celloff[(uint32_t)j * (W + 1) + min(X + c, W + 1)]);
            s_off[r][c] = v;
        }
        if (tid < 64) s_hist[tid] = 0;
        __syncthreads();
        if (tid == 32) {                                  // fetch the next work item while this one is processed
            const uint32_t nx = atomicAdd(A.item_cursor, 1u);
            s_next = nx; s_next_code = nx < n_items ? A.items[nx] : 0u;
        }
        if (tid < 32) {                                   // warp 0: one lane per cell row / pixel row issues that row's copies
            // order-list run of pixel row `tid`: global entries [g0, g1), widened to 8-entry (16-byte) boundaries
            uint32_t gs = 0, olen = 0;
            if (tid < th && Y + tid < H) {
                const size_t pr = (size_t)(Y + tid) * W;
                const uint32_t g0 = __ldg(&A.pixoff[pr + X]), g1 = __ldg(&A.pixoff[pr + min(X + tw, W)]);
                gs = g0 & ~7u;
                olen = g1 > g0 ? ((g1 + 7u) & ~7u) - gs : 0u;
            }
            const bool row = tid <= th;
            uint32_t a4 = 0, len = 0;
            if (row) {
                const uint32_t a = s_off[tid][0], b = s_off[tid][tw + 1];
                a4 = a & ~3u;
                len = b > a ? ((b + 3u) & ~3u) - a4 : 0u;
            }
            uint32_t inc = len, oinc = olen;
#pragma unroll
            for (int d = 1; d < 16; d <<= 1) {
                const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d), u = __shfl_up_sync(0xffffffffu, oinc, d);
                if (tid >= d) { inc += t; oinc += u; }
            }
            const uint32_t sb = inc - len, ob = oinc - olen;
            const uint32_t tot = __shfl_sync(0xffffffffu, inc, 15), otot = __shfl_sync(0xffffffffu, oinc, 15);
            if (row) { s_a4row[tid] = a4; s_sbase[tid] = sb; }
            if (tid < th) { s_rowblk[tid] = ob; s_rowg[tid] = gs; }
            fence_proxy_async();
            if (tid == 0) {
                s_tot = tot;
                if (tot > 0) mbar_arrive_expect_tx(&s_bar, tot * (uint32_t)(16 + 16 * FV + 16) + otot * 2u);
            }
            __syncwarp();
            if (tot > 0) {
                if (len) {
                    bulk_g2s(s_a4 + sb, A.Ra + a4, len * 16, &s_bar);
                    bulk_g2s(s_f + (size_t)sb * FV, A.Rf + (size_t)a4 * FV, len * FV * 16, &s_bar);
                    bulk_g2s(s_t4 + sb, reinterpret_cast<const float4*>(A.gT) + a4, len * 16, &s_bar);
                }
                if (olen) bulk_g2s(s_ord + ob, A.ord + gs, olen * 2, &s_bar);
            }
        }
        // while the copies fly: the lane permutation by descending blended count
        const uint32_t bucket = 63u - min(n_mine >> 2, 63u);
        const uint32_t rank_in_bucket = atomicAdd(&s_hist[bucket], 1u);
        __syncthreads();
        if (tid < 32) {                                                // exclusive scan of the 64 buckets
            const uint32_t b0 = s_hist[2 * tid], b1 = s_hist[2 * tid + 1];
            uint32_t inc = b0 + b1;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            s_hist[2 * tid] = inc - b0 - b1;
            s_hist[2 * tid + 1] = inc - b1;
        }
        if (live0) s_pixbase[tid] = s_rowblk[ly0] + (po_mine - s_rowg[ly0]);
        __syncthreads();
        s_perm[s_hist[bucket] + rank_in_bucket] = (uint8_t)tid;
        const uint32_t tot = s_tot;
        if (tot > 0) { mbar_wait(&s_bar, parity); parity ^= 1u; }
        // per-corner alphas in place: { tx, ty, opacity, idx } -> { a_0, a_1, a_2, a_3 }, corner c = 2 dy + dx
        for (uint32_t r = tid; r < tot; r += kTileThreads) {
            const float4 q = s_a4[r];
            const float wx0 = 1.f - q.x, wy0 = 1.f - q.y;
            s_a4[r] = make_float4(q.z * (wx0 * wy0), q.z * (q.x * wy0), q.z * (wx0 * q.y), q.z * (q.x * q.y));
        }
        __syncthreads();

        // ---------------------------------------------------------------- one thread per pixel
        const int q = s_perm[tid];
        const int ly = q >> lw, lx = q & (tw - 1);
        const int x = X + lx, y = Y + ly;
        if (q >= tw * th || x >= W || y >= H) continue;
        const size_t pix = (size_t)y * W + x;
        const uint4 cn = __ldg(&A.pcur[pix]);             // blended records of each of the four lists
        const uint32_t nb = cn.x + cn.y + cn.z + cn.w;
        if (nb == 0u) continue;
        // smem record of global slot g in cell row r: g + (s_sbase[r] - s_a4row[r]); corners 2, 3 lie in the top cell row
        const uint32_t bt = s_sbase[ly] - s_a4row[ly], bb = s_sbase[ly + 1] - s_a4row[ly + 1];
        float* gDtop = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bt));
        float* gDbot = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bb));
        float g[D], gA;
        load_pixel_grad<D>(A.io, A.g_feat, A.g_alpha, pix, g, gA);
        const uint32_t sa = smem_u32(s_a4), sf = smem_u32(s_f), st = smem_u32(s_t4);
        const uint32_t so = smem_u32(s_ord) + 2u * s_pixbase[q];

        float B = 0.f;
// one fragment: its loads ...
#define INPC_BACK_LOAD(i, kk)                                                                                             \
        const uint32_t e##i = lds_u16(so + 2u * (kk));                                                                    \
        const float a##i = lds_f32(sa + e##i), T##i = lds_f32(st + e##i);                                                 \
        float4 f##i[FV];                                                                                                  \
        _Pragma("unroll") for (int v = 0; v < FV; ++v) f##i[v] = lds_v4(sf + (e##i & 0xfff0u) * FV + 16 * v);
// ... and its step of the recurrence
#define INPC_BACK_STEP(i)                                                                                                 \
        {                                                                                                                 \
            float G = gA;                                                                                                 \
            _Pragma("unroll") for (int v = 0; v < FV; ++v)                                                                \
                G += f##i[v].x * g[4 * v] + f##i[v].y * g[4 * v + 1] + f##i[v].z * g[4 * v + 2] + f##i[v].w * g[4 * v + 3]; \
            ((e##i & 8u) ? gDtop : gDbot)[e##i >> 2] = T##i * (G - B);                                                    \
            B = a##i * G + (1.f - a##i) * B;                                                                              \
        }
        uint32_t k = nb;
        for (; k >= 4u; k -= 4u) {
            INPC_BACK_LOAD(0, k - 1u) INPC_BACK_LOAD(1, k - 2u) INPC_BACK_LOAD(2, k - 3u) INPC_BACK_LOAD(3, k - 4u)
            INPC_BACK_STEP(0) INPC_BACK_STEP(1) INPC_BACK_STEP(2) INPC_BACK_STEP(3)
        }
        for (; k >= 1u; --k) {
            INPC_BACK_LOAD(0, k - 1u)
            INPC_BACK_STEP(0)
        }
#undef INPC_BACK_LOAD
#undef INPC_BACK_STEP
    }
}

}  // namespace inpc
