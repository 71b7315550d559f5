// back.cuh -- step a5 of the hot path, first half: the reverse traversal of every pixel's blended fragments
// ("process them in the same order as in the forward pass" -- here backwards through it).
//
// Same persistent tile kernel shape as blend.cuh: one work item = a screen tile whose records fit shared memory,
// staged exactly as the forward pass staged it (same cell rows, same 4-record alignment => the same shared-memory
// record indices), with cp.async.bulk onto one mbarrier: per record the { tx, ty, opacity, idx } word (turned into
// the four per-corner alphas in place), the features and the four transmittances gT the forward pass saved.
// The depth order is NOT merged again: the forward pass left, for every tile item, one block of ord[] holding the
// item's per-pixel lists of blended (record, corner) in blend order (16 bits per fragment, blend.cuh); the block
// is staged by one more bulk copy.  ONE THREAD PER PIXEL (lanes in descending order of the blended count) walks
// its list from the last blended fragment to the first with the division-free recurrence
//     dL/da_k = T_k (G_k - B_k),    B_{k-1} = a_k G_k + (1 - a_k) B_k,    G_k = <feat_k, g_img[p]> + g_alpha[p]
// and writes dL/da_k to gD[(slot, corner)]; grad.cuh combines the four corners of every record.  No address in
// the loop depends on the recurrence, so the loads of four fragments are issued together and the only dependent
// chain is B.
// What bounds a tile is latency, not work, so everything a tile needs BEFORE its bulk copies can be issued (cell
// offsets, block position) and everything its pixels need (blended counts, image gradients) is loaded into
// registers one tile ahead, while the previous tile is walked.
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
    const uint2* ordinfo;    // per item of this band: { first entry of its block of ord[], entries }
    const uint16_t* ord;     // (record * 16 + 4 * corner) of the k-th blended fragment, tile-local (forward pass)
    const float* g_feat;
    const float* g_alpha;
    ImageIO io;
    float* gD;
};

template <int D> __host__ __device__ constexpr size_t back_smem_bytes() {
    return (size_t)TileCfg<D>::kCap * (16 + 4 * D + 16 + 8) + 16;     // alphas, features, gT, order lists
}
static_assert(back_smem_bytes<4>() + 12288 <= kMaxSmemPerCta && back_smem_bytes<8>() + 12288 <= kMaxSmemPerCta,
              "k_back: tile capacity exceeds the shared memory of one CTA (dynamic + < 12 KB static)");

// What a thread loads one tile ahead: up to two entries of the (th+1) x (tw+2) window of cell offsets, its pixel's
// (natural order) blended counts and image gradient, and (thread 0) the tile's block of the saved order.
template <int D> struct BackPrefetch {
    uint32_t off0, off1;
    uint4 cn;
    float g[D], gA;
    uint2 info;
};

template <int D>
__device__ __forceinline__ void back_prefetch(const BackArgs& A, uint32_t item_i, uint32_t it, bool valid, BackPrefetch<D>& P) {
    const int tid = threadIdx.x;
    const int W = A.W, H = A.H;
    const int X = it & 0xfff, Y = (it >> 12) & 0xfff, lw = (it >> 24) & 7, lh = (it >> 27) & 3;
    const int tw = 1 << lw, th = 1 << lh;
    P.off0 = P.off1 = 0u;
    P.cn = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int d = 0; d < D; ++d) P.g[d] = 0.f;
    P.gA = 0.f;
    P.info = make_uint2(0, 0);
    if (!valid) return;
    const int n_off = (th + 1) * (tw + 2);
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int e = tid + h * kTileThreads;
        if (e < n_off) {
            const int r = e / (tw + 2), c = e - r * (tw + 2);
            const int j = Y + r;
            const uint32_t v = j <= H ? __ldg(&A.celloff[(uint32_t)j * (W + 1) + min(X + c, W + 1)]) : 0u;
            if (h == 0) P.off0 = v; else P.off1 = v;
        }
    }
    const int ly0 = tid >> lw, lx0 = tid & (tw - 1);
    if (tid < tw * th && X + lx0 < W && Y + ly0 < H) {
        const size_t p0 = (size_t)(Y + ly0) * W + X + lx0;
        P.cn = __ldg(&A.pcur[p0]);
        // raw loads only: nothing here may wait for a load (the values are scaled when they go to shared memory)
        if (!A.io.planar) {
#pragma unroll
            for (int v = 0; v < D / 4; ++v) {
                const float4 t = __ldg(reinterpret_cast<const float4*>(A.g_feat + p0 * D) + v);
                P.g[4 * v] = t.x; P.g[4 * v + 1] = t.y; P.g[4 * v + 2] = t.z; P.g[4 * v + 3] = t.w;
            }
        } else {
#pragma unroll
            for (int d = 0; d < D; ++d) P.g[d] = __ldg(A.g_feat + (size_t)d * A.io.P + p0);
        }
        P.gA = A.g_alpha ? __ldg(A.g_alpha + p0) : 0.f;
    }
    if (tid == 0) P.info = __ldg(&A.ordinfo[item_i]);
}

template <int D>
__global__ void __launch_bounds__(kTileThreads, 384 / kTileThreads) k_back(BackArgs A) {
    constexpr int FV  = D / 4;
    constexpr int CAP = TileCfg<D>::kCap;
    static_assert((kTileH + 1) * (kTileW + 2) <= 2 * kTileThreads, "two window entries per thread");
    extern __shared__ __align__(128) unsigned char smem[];
    float4*   s_a4  = reinterpret_cast<float4*>(smem);
    float4*   s_f   = reinterpret_cast<float4*>(smem + (size_t)CAP * 16);
    float4*   s_t4  = reinterpret_cast<float4*>(smem + (size_t)CAP * (16 + 16 * FV));
    uint16_t* s_ord = reinterpret_cast<uint16_t*>(smem + (size_t)CAP * (32 + 16 * FV));

    __shared__ uint32_t s_off[(kTileH + 1) * (kTileW + 2)];   // window of cell offsets, row stride tw + 2
    __shared__ uint32_t s_sbase[kTileH + 1], s_a4row[kTileH + 1];
    __shared__ uint32_t s_hist[64];
    __shared__ uint32_t s_pixbase[kTileThreads], s_wsum[kTileThreads / 32];
    __shared__ uint4    s_cn[kTileThreads];                   // per pixel (natural order): blended records of its four lists
    __shared__ float    s_g[kTileThreads][D + 1];             // ... and its image gradient (g_img[D], g_alpha)
    __shared__ uint8_t  s_perm[kTileThreads];
    __shared__ uint32_t s_next, s_next_code, s_tot, s_ordn;
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
    __syncthreads();
    BackPrefetch<D> P;
    back_prefetch<D>(A, s_next, s_next_code, s_next < n_items, P);
    uint32_t parity = 0;

    while (true) {
        fence_proxy_async();                              // each thread's generic accesses to the tile's arrays, before the next bulk loads overwrite them
        __syncthreads();                                  // (A) everyone is done with the previous item's smem
        const uint32_t item_i = s_next;
        if (item_i >= n_items) break;
        const uint32_t it = s_next_code;
        const int X = it & 0xfff, Y = (it >> 12) & 0xfff, lw = (it >> 24) & 7, lh = (it >> 27) & 3;
        const int tw = 1 << lw, th = 1 << lh, ws = tw + 2;
        // what was loaded one tile ahead goes to shared memory
        if (tid < (th + 1) * ws) s_off[tid] = P.off0;
        if (tid + kTileThreads < (th + 1) * ws) s_off[tid + kTileThreads] = P.off1;
        s_cn[tid] = P.cn;
#pragma unroll
        for (int d = 0; d < D; ++d) s_g[tid][d] = A.io.scale * P.g[d];     // as load_pixel_grad: the gradient image's scale
        s_g[tid][D] = A.io.scale * P.gA;
        if (tid == 0) s_ordn = P.info.y;
        const uint32_t ord_base = P.info.x;               // (thread 0)
        const uint32_t n_bl = P.cn.x + P.cn.y + P.cn.z + P.cn.w;
        if (tid < 64) s_hist[tid] = 0;
        __syncthreads();                                  // (B)
        if (tid == 32) {                                  // fetch the next work item while this one is processed
            const uint32_t nx = atomicAdd(A.item_cursor, 1u);
            s_next = nx; s_next_code = nx < n_items ? A.items[nx] : 0u;
        }
        if (tid < 32) {                                   // warp 0: one lane per cell row issues that row's copies
            const bool row = tid <= th;
            uint32_t a4 = 0, len = 0;
            if (row) {
                const uint32_t a = s_off[tid * ws], b = s_off[tid * ws + tw + 1];
                a4 = a & ~3u;
                len = b > a ? ((b + 3u) & ~3u) - a4 : 0u;
            }
            uint32_t inc = len;
#pragma unroll
            for (int d = 1; d < 16; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            const uint32_t sb = inc - len;
            const uint32_t tot = __shfl_sync(0xffffffffu, inc, 15);
            if (row) { s_a4row[tid] = a4; s_sbase[tid] = sb; }
            const uint32_t n8 = (s_ordn + 7u) & ~7u;      // the forward pass wrote the block in 8-entry (16-byte) units
            fence_proxy_async();
            if (tid == 0) {
                s_tot = tot;
                if (tot > 0) {
                    mbar_arrive_expect_tx(&s_bar, tot * (uint32_t)(16 + 16 * FV + 16) + n8 * 2u);
                    if (n8) bulk_g2s(s_ord, A.ord + ord_base, n8 * 2u, &s_bar);
                }
            }
            __syncwarp();
            if (tot > 0 && len) {
                bulk_g2s(s_a4 + sb, A.Ra + a4, len * 16, &s_bar);
                bulk_g2s(s_f + (size_t)sb * FV, A.Rf + (size_t)a4 * FV, len * FV * 16, &s_bar);
                bulk_g2s(s_t4 + sb, reinterpret_cast<const float4*>(A.gT) + a4, len * 16, &s_bar);
            }
        }
        // while the copies fly: the lane permutation by descending blended count; the starts of the order lists are the
        // exclusive scan of the pixels' fragment counts in natural order (exactly what the forward pass laid out)
        const int ly0 = tid >> lw, lx0 = tid & (tw - 1);
        uint32_t n_all = 0;
        if (tid < tw * th && X + lx0 < W && Y + ly0 < H)
            n_all = (s_off[ly0 * ws + lx0 + 2] - s_off[ly0 * ws + lx0]) + (s_off[(ly0 + 1) * ws + lx0 + 2] - s_off[(ly0 + 1) * ws + lx0]);
        const uint32_t bucket = 63u - min(n_bl >> 2, 63u);
        const uint32_t rank_in_bucket = atomicAdd(&s_hist[bucket], 1u);
        uint32_t inc_all = n_all;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc_all, d); if ((tid & 31) >= d) inc_all += t; }
        if ((tid & 31) == 31) s_wsum[tid >> 5] = inc_all;
        __syncthreads();                                  // (C)
        if (tid < 32) {                                   // exclusive scan of the 64 buckets
            const uint32_t b0 = s_hist[2 * tid], b1 = s_hist[2 * tid + 1];
            uint32_t inc = b0 + b1;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            s_hist[2 * tid] = inc - b0 - b1;
            s_hist[2 * tid + 1] = inc - b1;
        }
        {
            uint32_t before = 0;
#pragma unroll
            for (int w = 0; w < kTileThreads / 32; ++w) before += w < (tid >> 5) ? s_wsum[w] : 0u;
            s_pixbase[tid] = before + inc_all - n_all;
        }
        __syncthreads();                                  // (D)
        s_perm[s_hist[bucket] + rank_in_bucket] = (uint8_t)tid;
        const uint32_t tot = s_tot;
        if (tot > 0) { mbar_wait(&s_bar, parity); parity ^= 1u; }
        // per-corner alphas in place: { tx, ty, opacity, idx } -> { a_0, a_1, a_2, a_3 }, corner c = 2 dy + dx
        for (uint32_t r = tid; r < tot; r += kTileThreads) {
            const float4 q = s_a4[r];
            const float wx0 = 1.f - q.x, wy0 = 1.f - q.y;
            s_a4[r] = make_float4(q.z * (wx0 * wy0), q.z * (q.x * wy0), q.z * (wx0 * q.y), q.z * (q.x * q.y));
        }
        __syncthreads();                                  // (E)
        // the next tile's metadata: in flight while this one is walked
        { const uint32_t nx = s_next; back_prefetch<D>(A, nx, s_next_code, nx < n_items, P); }

        // ---------------------------------------------------------------- one thread per pixel
        const int q = s_perm[tid];
        const int ly = q >> lw, lx = q & (tw - 1);
        if (q >= tw * th || X + lx >= W || Y + ly >= H) continue;
        const uint4 cn = s_cn[q];                         // blended records of each of the four lists
        const uint32_t nb = cn.x + cn.y + cn.z + cn.w;
        if (nb == 0u) continue;
        // smem record of global slot g in cell row r: g + (s_sbase[r] - s_a4row[r]); corners 2, 3 lie in the top cell row
        const uint32_t bt = s_sbase[ly] - s_a4row[ly], bb = s_sbase[ly + 1] - s_a4row[ly + 1];
        float* gDtop = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bt));
        float* gDbot = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bb));
        float g[D];
#pragma unroll
        for (int d = 0; d < D; ++d) g[d] = s_g[q][d];
        const float gA = s_g[q][D];
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
