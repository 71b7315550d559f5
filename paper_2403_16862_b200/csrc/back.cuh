// back.cuh -- step a5 of the hot path, first half: the reverse traversal of every pixel's blended fragments
// ("process them in the same order as in the forward pass" -- here backwards through it).
//
// Same persistent tile kernel shape as blend.cuh (one work item = a screen tile whose records fit shared
// memory; the tile's th+1 cell rows staged with cp.async.bulk onto one mbarrier; { tx, ty, opacity, idx }
// turned into per-corner alphas in place; pixels handed to lanes in descending order of their BLENDED
// fragment count, which the forward pass left in pcur).  Staged per record: depth key, alphas, features and
// the four transmittances gT the forward pass saved.  ONE THREAD PER PIXEL starts from the four stop
// positions pcur and merges the four lists BACKWARDS (maximum head first) with the division-free recurrence
//     dL/da_k = T_k (G_k - B_k),    B_{k-1} = a_k G_k + (1 - a_k) B_k,    G_k = <feat_k, g_img[p]> + g_alpha[p]
// and writes dL/da_k to gD[(slot, corner)]; grad.cuh combines the four corners of every record.
// The iteration is branch-free (cursor | list start packed in one register, predicates select the list) and
// software-pipelined like the forward loop: iteration k selects fragment k and issues its shared-memory
// loads, then finishes fragment k+1 (the one selected before) while they are in flight.
#pragma once
#include "common.cuh"
#include "blend.cuh"

namespace inpc {

struct BackArgs {
    const Header* hdr;
    uint32_t* item_cursor;   // this band's work cursor ...
    const uint32_t* n_items; // ... and item count (device)
    const uint32_t* items;
    const uint32_t* celloff;
    const uint32_t* dk;
    const float4* Ra;
    const float4* Rf;
    int W, H;
    const float* gT;
    const uint4* pcur;
    const float* g_feat;
    const float* g_alpha;
    ImageIO io;
    float* gD;
};

template <int D> __host__ __device__ constexpr size_t back_smem_bytes() {
    return (size_t)TileCfg<D>::kCap * (4 + 16 + 4 * D + 16);       // dk, alphas, features, gT
}

template <int D>
__global__ void __launch_bounds__(kTileThreads) k_back(BackArgs A) {
    constexpr int FV  = D / 4;
    constexpr int CAP = TileCfg<D>::kCap;
    extern __shared__ __align__(128) unsigned char smem[];
    uint32_t* s_dk = reinterpret_cast<uint32_t*>(smem);
    float4*   s_a4 = reinterpret_cast<float4*>(smem + (size_t)CAP * 4);
    float4*   s_f  = reinterpret_cast<float4*>(smem + (size_t)CAP * 20);
    float4*   s_t4 = reinterpret_cast<float4*>(smem + (size_t)CAP * (20 + 16 * FV));
    const unsigned char* s_ab = smem + (size_t)CAP * 4;                       // alphas, byte-addressed
    const unsigned char* s_tb = smem + (size_t)CAP * (20 + 16 * FV);          // transmittances, same offsets

    __shared__ uint32_t s_off[kTileH + 1][kTileW + 2];
    __shared__ uint32_t s_sbase[kTileH + 1], s_a4row[kTileH + 1];
    __shared__ uint32_t s_hist[64];
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
        if (tid < 32) {                                   // warp 0: one lane per cell row issues that row's copies
            const bool row = tid <= th;
            uint32_t a4 = 0, len = 0;
            if (row) {
                const uint32_t a = s_off[tid][0], b = s_off[tid][tw + 1];
                a4 = a & ~3u;
                len = b > a ? ((b + 3u) & ~3u) - a4 : 0u;
            }
            uint32_t inc = len;
#pragma unroll
            for (int d = 1; d < 16; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            const uint32_t sb = inc - len;
            const uint32_t tot = __shfl_sync(0xffffffffu, inc, 15);
            if (row) { s_a4row[tid] = a4; s_sbase[tid] = sb; }
            fence_proxy_async();
            if (tid == 0) {
                s_tot = tot;
                if (tot > 0) mbar_arrive_expect_tx(&s_bar, tot * (uint32_t)(4 + 16 + 16 * FV + 16));
            }
            __syncwarp();
            if (len) {
                bulk_g2s(s_dk + sb, A.dk + a4, len * 4, &s_bar);
                bulk_g2s(s_a4 + sb, A.Ra + a4, len * 16, &s_bar);
                bulk_g2s(s_f + (size_t)sb * FV, A.Rf + (size_t)a4 * FV, len * FV * 16, &s_bar);
                bulk_g2s(s_t4 + sb, reinterpret_cast<const float4*>(A.gT) + a4, len * 16, &s_bar);
            }
        }
        // while the copies fly: this thread's pixel, its blended fragment count, and the count histogram
        const int ly0 = tid >> lw, lx0 = tid & (tw - 1);
        uint32_t n_mine = 0;
        if (tid < tw * th && X + lx0 < W && Y + ly0 < H) {
            const uint4 cn = __ldg(&A.pcur[(size_t)(Y + ly0) * W + X + lx0]);
            n_mine = cn.x + cn.y + cn.z + cn.w;
        }
        const uint32_t bucket = 63u - min(n_mine >> 2, 63u);          // descending count
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
        if ((cn.x | cn.y | cn.z | cn.w) == 0u) continue;
        // smem record of global slot g in cell row r: g + (s_sbase[r] - s_a4row[r])
        const uint32_t bt = s_sbase[ly] - s_a4row[ly], bb = s_sbase[ly + 1] - s_a4row[ly + 1];
        const uint32_t st0 = s_off[ly][lx] + bt, st1 = s_off[ly][lx + 1] + bt;
        const uint32_t st2 = s_off[ly + 1][lx] + bb, st3 = s_off[ly + 1][lx + 1] + bb;
        // list j holds the pixel's fragments of corner 3 - j.  Packed state: low 16 bits = byte offset
        // (record * 16 + 4 * corner) of the list's LAST not yet visited blended fragment, high 16 = its first.
        auto pack_rev = [](uint32_t st, uint32_t n, uint32_t corner) -> uint32_t {
            const uint32_t first = st * 16u + 4u * corner;
            return (n ? first + (n - 1u) * 16u : first) | (first << 16);
        };
        uint32_t ce0 = pack_rev(st0, cn.x, 3), ce1 = pack_rev(st1, cn.y, 2);
        uint32_t ce2 = pack_rev(st2, cn.z, 1), ce3 = pack_rev(st3, cn.w, 0);
        uint32_t h0 = cn.x ? s_dk[st0 + cn.x - 1u] : 0u, h1 = cn.y ? s_dk[st1 + cn.y - 1u] : 0u;
        uint32_t h2 = cn.z ? s_dk[st2 + cn.z - 1u] : 0u, h3 = cn.w ? s_dk[st3 + cn.w - 1u] : 0u;
        // global float index of (slot, corner) = (cursor >> 2) + 4 * (slot - smem record)
        float* gDtop = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bt));
        float* gDbot = A.gD + 4 * ((ptrdiff_t)(int32_t)(0u - bb));
        float g[D], gA;
        load_pixel_grad<D>(A.io, A.g_feat, A.g_alpha, pix, g, gA);

        float B = 0.f;
        float pa = 0.f, pT = 0.f;                         // pending fragment: alpha, transmittance, features, gD address
        float4 pf[FV];
#pragma unroll
        for (int v = 0; v < FV; ++v) pf[v] = make_float4(0.f, 0.f, 0.f, 0.f);
        float* pg = nullptr;
        bool have = false;
        uint32_t m = max(max(h0, h1), max(h2, h3));
        while (m != 0u) {                                 // depth bits are > 0 (z_c > near_z >= 0): 0 = list exhausted
            bool p0 = h0 == m, p1 = h1 == m, p2 = h2 == m, p3 = h3 == m;
            if ((p0 & (p1 | p2 | p3)) | (p1 & (p2 | p3)) | (p2 & p3)) {
                uint32_t best = 0u;                       // reverse order: descending point index
                int jb = 0;
                if (p0) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce0 & 0xffffu) >> 4) - bt]).w); if (i >= best) { best = i; jb = 0; } }
                if (p1) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce1 & 0xffffu) >> 4) - bt]).w); if (i >= best) { best = i; jb = 1; } }
                if (p2) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce2 & 0xffffu) >> 4) - bb]).w); if (i >= best) { best = i; jb = 2; } }
                if (p3) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce3 & 0xffffu) >> 4) - bb]).w); if (i >= best) { best = i; jb = 3; } }
                p0 = jb == 0; p1 = jb == 1; p2 = jb == 2; p3 = jb == 3;
            }
            const uint32_t ce = p0 ? ce0 : (p1 ? ce1 : (p2 ? ce2 : ce3));
            const uint32_t cur = ce & 0xffffu;
            // issue the loads of fragment k
            const float na = *reinterpret_cast<const float*>(s_ab + cur);
            const float nT = *reinterpret_cast<const float*>(s_tb + cur);
            float4 nf[FV];
#pragma unroll
            for (int v = 0; v < FV; ++v) nf[v] = s_f[(cur >> 4) * FV + v];
            const uint32_t nh = cur > (ce >> 16) ? s_dk[(cur >> 4) - 1u] : 0u;
            const uint32_t nx = ce - 16u;
            float* ng = ((p0 | p1) ? gDtop : gDbot) + (cur >> 2);
            // finish the fragment selected one iteration ago
            float G = gA;
#pragma unroll
            for (int v = 0; v < FV; ++v)
                G += pf[v].x * g[4 * v] + pf[v].y * g[4 * v + 1] + pf[v].z * g[4 * v + 2] + pf[v].w * g[4 * v + 3];
            if (have) *pg = pT * (G - B);
            B = pa * G + (1.f - pa) * B;
            h0 = p0 ? nh : h0; ce0 = p0 ? nx : ce0;
            h1 = p1 ? nh : h1; ce1 = p1 ? nx : ce1;
            h2 = p2 ? nh : h2; ce2 = p2 ? nx : ce2;
            h3 = p3 ? nh : h3; ce3 = p3 ? nx : ce3;
            pa = na; pT = nT; pg = ng; have = true;
#pragma unroll
            for (int v = 0; v < FV; ++v) pf[v] = nf[v];
            m = max(max(h0, h1), max(h2, h3));
        }
        if (have) {
            float G = gA;
#pragma unroll
            for (int v = 0; v < FV; ++v)
                G += pf[v].x * g[4 * v] + pf[v].y * g[4 * v + 1] + pf[v].z * g[4 * v + 2] + pf[v].w * g[4 * v + 3];
            *pg = pT * (G - B);
        }
    }
}

}  // namespace inpc
