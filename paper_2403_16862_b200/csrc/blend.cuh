// blend.cuh -- step a4 of the hot path: per-pixel 4-way merge of the sorted cell lists and front-to-back
// compositing (Eq. 1; cut-off T < 1e-4 from BASELINE.json north_star).
//
// One persistent CTA per work item (a screen tile of tw x th <= 128 pixels whose records fit in shared
// memory).  The tile's th+1 cell rows are contiguous slot ranges of the cell-sorted arrays dk / Ra / Rf
// and are staged with cp.async.bulk (TMA, 1-D) onto one mbarrier.  Then
//   1. one thread per staged record turns { tx, ty, opacity, idx } into the four per-corner alphas
//      a_c = opacity * w_c (Eq. 7) in place, so the merge loop reads ONE float per fragment;
//   2. the tile's pixels are handed to lanes in descending order of their fragment count (counting sort on
//      count / 4), so that the 32 pixels of a warp run about equally long
//      (round-1 facts: neighbouring pixels gave 10 of 32 lanes active);
//   3. ONE THREAD PER PIXEL merges its four lists.  The iteration is branch-free: every list's cursor and
//      end are packed into one register (byte offset of the fragment's alpha | end << 16), the minimum
//      head key selects the list with predicates, and only "two heads with equal depth bits" (ascending
//      point index decides, read from global memory) and the two loop exits are branches.
// With INPC_SAVE_FOR_BACKWARD the transmittance in front of every blended fragment goes to
// gT[(slot, corner)], the four list positions at the stop to pcur[pixel], and the ORDER itself is kept: which
// staged (record, corner) was blended k-th (16 bits: the fragment's byte offset record * 16 + 4 * corner inside the
// tile's staged records), one list per pixel, the tile's lists back to back in shared memory and written out as
// ONE block of ord[] by a bulk (TMA) store while the next tile is already being staged; ordinfo[item] = { start of
// the block, entries }.  The backward pass stages the same tile the same way and walks those lists backwards
// without merging anything again (back.cuh).
#pragma once
#include "common.cuh"

namespace inpc {

struct BlendArgs {
    const Header* hdr;
    uint32_t* item_cursor;   // this band's work cursor ...
    const uint32_t* n_items; // ... and item count (device)
    const uint32_t* items;
    const uint32_t* celloff;
    const uint32_t* dk;
    const float4* Ra;
    const float4* Rf;
    int W, H;
    float* out_feat;
    float* out_alpha;
    ImageIO io;
    float* gT;               // NULL unless INPC_SAVE_FOR_BACKWARD
    uint4* pcur;
    uint16_t* ord;           // blend order, one block per tile item (INPC_SAVE_FOR_BACKWARD)
    uint2* ordinfo;          // per item of this band: { first entry of its block, entries }
    uint32_t* ord_cursor;    // bump allocator of the blocks
    // dump (INPC_SAVE_SORTED)
    const uint32_t* pixoff;  // exclusive scan of the per-pixel fragment counts
    uint32_t* sorted_idx;
    uint32_t* sorted_depth;
    float* sorted_T;         // transmittance in front of every blended fragment, -1 behind the cut-off
};

// per staged record: depth key, alphas, features; with SAVE also the tile's order lists (2 bytes per fragment)
template <int D, bool SAVE> __host__ __device__ constexpr size_t blend_smem_bytes() {
    return (size_t)TileCfg<D>::kCap * (4 + 16 + 4 * D + (SAVE ? 8 : 0));
}
static_assert(blend_smem_bytes<4, true>() + 4096 <= kMaxSmemPerCta && blend_smem_bytes<8, true>() + 4096 <= kMaxSmemPerCta,
              "k_blend: tile capacity exceeds the shared memory of one CTA (dynamic + < 4 KB static)");

// Packed list state: low 16 bits = byte offset of the head fragment's alpha inside s_a (record * 16 +
// 4 * corner), high 16 bits = the same for the list's end.  One record further = + 16.
__device__ __forceinline__ uint32_t pack_list(uint32_t start_rec, uint32_t end_rec, int corner) {
    return (start_rec * 16u + 4u * corner) | ((end_rec * 16u + 4u * corner) << 16);
}

// Two heads with equal depth bits (rare): ascending point index decides, read from global memory.  A macro, not a
// lambda: with by-reference captures of the list predicates the compiler kept a branch inside the merge loop
// (k_blend 301 -> 352 us).
#define INPC_BLEND_RESOLVE_TIE()                                                                                          \
    do {                                                                                                                  \
        uint32_t best = 0xFFFFFFFFu;                                                                                      \
        int jb = 0;                                                                                                       \
        if (p0) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce0 & 0xffffu) >> 4) - bt]).w); if (i < best) { best = i; jb = 0; } } \
        if (p1) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce1 & 0xffffu) >> 4) - bt]).w); if (i < best) { best = i; jb = 1; } } \
        if (p2) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce2 & 0xffffu) >> 4) - bb]).w); if (i < best) { best = i; jb = 2; } } \
        if (p3) { const uint32_t i = __float_as_uint(__ldg(&A.Ra[((ce3 & 0xffffu) >> 4) - bb]).w); if (i < best) { best = i; jb = 3; } } \
        p0 = jb == 0; p1 = jb == 1; p2 = jb == 2; p3 = jb == 3;                                                           \
    } while (0)

template <int D, bool SAVE, bool DUMP>
__global__ void __launch_bounds__(kTileThreads, 512 / kTileThreads) k_blend(BlendArgs A) {
    constexpr int FV  = D / 4;                     // float4 of features per record
    constexpr int CAP = TileCfg<D>::kCap;
    extern __shared__ __align__(128) unsigned char smem[];
    uint32_t* s_dk = reinterpret_cast<uint32_t*>(smem);
    float4*   s_a4 = reinterpret_cast<float4*>(smem + (size_t)CAP * 4);
    float4*   s_f  = reinterpret_cast<float4*>(smem + (size_t)CAP * 20);
    const unsigned char* s_ab = smem + (size_t)CAP * 4;
    uint16_t* s_ord = reinterpret_cast<uint16_t*>(smem + (size_t)CAP * (20 + 16 * FV));   // SAVE only
    __shared__ uint32_t s_pixbase[kTileThreads], s_wsum[kTileThreads / 32], s_ordtot, s_ordbase;   // SAVE: starts of the tile's order lists, its block of ord[]

    __shared__ uint32_t s_off[kTileH + 1][kTileW + 2];
    __shared__ uint32_t s_sbase[kTileH + 1], s_a4row[kTileH + 1];
    __shared__ uint32_t s_hist[64];
    __shared__ uint8_t  s_perm[kTileThreads];
    __shared__ uint32_t s_next, s_next_code, s_tot;
    __shared__ __align__(8) uint64_t s_bar;

    const int tid = threadIdx.x;
    const int W = A.W, H = A.H;
    const uint32_t n_items = *A.n_items;

    if (tid == 0) {
        mbar_init(&s_bar, 1); fence_mbar_init();
        const uint32_t nx = atomicAdd(A.item_cursor, 1u);
        s_next = nx; s_next_code = nx < n_items ? A.items[nx] : 0u;
    }
    uint32_t parity = 0;
    bool have_prev = false;                               // SAVE: the previous item's order lists still sit in shared memory

    while (true) {
        // Every thread's generic-proxy accesses to the tile's shared memory (the order lists it wrote, the alphas it wrote
        // in place, the records it read) are ordered before the async-proxy copies thread 0 / warp 0 issue behind the
        // barrier (bulk store of the order lists, bulk loads over the record arrays): each writer fences, then the barrier.
        fence_proxy_async();
        __syncthreads();                                  // everyone is done with the previous item's smem
        if constexpr (SAVE) {
            // The previous tile's order lists (back to back in shared memory, pixels in natural order) go out to ord[] as
            // one block: a bulk store issued by one thread; it has finished reading before this tile's walk overwrites them.
            if (tid == 0 && have_prev) {
                const uint32_t n8 = (s_ordtot + 7u) & ~7u;
                if (n8) { fence_proxy_async(); bulk_s2g(A.ord + s_ordbase, s_ord, n8 * 2u); }
            }
        }
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
                if (tot > 0) mbar_arrive_expect_tx(&s_bar, tot * (uint32_t)(4 + 16 + 16 * FV));
            }
            __syncwarp();
            if (len) {
                bulk_g2s(s_dk + sb, A.dk + a4, len * 4, &s_bar);
                bulk_g2s(s_a4 + sb, A.Ra + a4, len * 16, &s_bar);
                bulk_g2s(s_f + (size_t)sb * FV, A.Rf + (size_t)a4 * FV, len * FV * 16, &s_bar);
            }
        }
        // while the copies fly: this thread's pixel, its fragment count, and the count histogram
        const int ly0 = tid >> lw, lx0 = tid & (tw - 1);
        uint32_t n_mine = 0;
        const bool live0 = tid < tw * th && X + lx0 < W && Y + ly0 < H;
        if (live0)
            n_mine = (s_off[ly0][lx0 + 2] - s_off[ly0][lx0]) + (s_off[ly0 + 1][lx0 + 2] - s_off[ly0 + 1][lx0]);
        const uint32_t bucket = 63u - min(n_mine >> 2, 63u);          // descending count
        const uint32_t rank_in_bucket = atomicAdd(&s_hist[bucket], 1u);
        uint32_t inc_mine = n_mine;                                    // SAVE: scan of the counts in natural pixel order
        if constexpr (SAVE) {
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc_mine, d); if ((tid & 31) >= d) inc_mine += t; }
            if ((tid & 31) == 31) s_wsum[tid >> 5] = inc_mine;
        }
        __syncthreads();
        if constexpr (SAVE) {
            uint32_t before = 0;
#pragma unroll
            for (int w = 0; w < kTileThreads / 32; ++w) before += w < (tid >> 5) ? s_wsum[w] : 0u;
            s_pixbase[tid] = before + inc_mine - n_mine;
            if (tid == kTileThreads - 1) {                 // this tile's block of ord[]: reserved here, off warp 0's path
                const uint32_t total = before + inc_mine, n8 = (total + 7u) & ~7u;
                const uint32_t base = n8 ? atomicAdd(A.ord_cursor, n8) : 0u;
                s_ordtot = total; s_ordbase = base;
                A.ordinfo[item_i] = make_uint2(base, total);
            }
            have_prev = true;
        }
        if (tid < 32) {                                                // exclusive scan of the 64 buckets
            const uint32_t h0 = s_hist[2 * tid], h1 = s_hist[2 * tid + 1];
            uint32_t inc = h0 + h1;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (tid >= d) inc += t; }
            s_hist[2 * tid] = inc - h0 - h1;
            s_hist[2 * tid + 1] = inc - h1;
        }
        __syncthreads();
        s_perm[s_hist[bucket] + rank_in_bucket] = (uint8_t)tid;
        const uint32_t tot = s_tot;
        if (tot > 0) { mbar_wait(&s_bar, parity); parity ^= 1u; }
        // 1. per-corner alphas in place: { tx, ty, opacity, idx } -> { a_0, a_1, a_2, a_3 }, corner c = 2 dy + dx
        for (uint32_t r = tid; r < tot; r += kTileThreads) {
            const float4 q = s_a4[r];
            const float wx0 = 1.f - q.x, wy0 = 1.f - q.y;
            s_a4[r] = make_float4(q.z * (wx0 * wy0), q.z * (q.x * wy0), q.z * (wx0 * q.y), q.z * (q.x * q.y));
        }
        if constexpr (SAVE) { if (tid == 0) bulk_wait_read(); }       // the previous tile's order lists have left shared memory
        __syncthreads();

        // The next work item is drawn HERE, behind the tile's last set-up barrier: its two dependent round trips (ticket,
        // item code) used to sit between two of those barriers, where the whole CTA waited for them.
        if (tid == kTileThreads - 1) {
            const uint32_t nx = atomicAdd(A.item_cursor, 1u);
            s_next = nx; s_next_code = nx < n_items ? A.items[nx] : 0u;
        }
        // ---------------------------------------------------------------- 3. one thread per pixel
        const int q = s_perm[tid];
        const int ly = q >> lw, lx = q & (tw - 1);
        const int x = X + lx, y = Y + ly;
        if (q >= tw * th || x >= W || y >= H) continue;
        const size_t pix = (size_t)y * W + x;
        // smem record of global slot g in cell row r: g + (s_sbase[r] - s_a4row[r])
        const uint32_t bt = s_sbase[ly] - s_a4row[ly], bb = s_sbase[ly + 1] - s_a4row[ly + 1];
        const uint32_t st0 = s_off[ly][lx] + bt, st1 = s_off[ly][lx + 1] + bt, en1 = s_off[ly][lx + 2] + bt;
        const uint32_t st2 = s_off[ly + 1][lx] + bb, st3 = s_off[ly + 1][lx + 1] + bb, en3 = s_off[ly + 1][lx + 2] + bb;
        // list j holds the pixel's fragments of corner 3 - j
        uint32_t ce0 = pack_list(st0, st1, 3), ce1 = pack_list(st1, en1, 2);
        uint32_t ce2 = pack_list(st2, st3, 1), ce3 = pack_list(st3, en3, 0);
        uint32_t h0 = st0 < st1 ? s_dk[st0] : kSentHi, h1 = st1 < en1 ? s_dk[st1] : kSentHi;
        uint32_t h2 = st2 < st3 ? s_dk[st2] : kSentHi, h3 = st3 < en3 ? s_dk[st3] : kSentHi;
        // global float index of (slot, corner) = (cursor >> 2) + 4 * (slot - smem record)
        float* gTtop = SAVE ? A.gT + 4 * ((ptrdiff_t)(int32_t)(0u - bt)) : nullptr;
        float* gTbot = SAVE ? A.gT + 4 * ((ptrdiff_t)(int32_t)(0u - bb)) : nullptr;
        (void)gTtop; (void)gTbot;

        float acc[D];
#pragma unroll
        for (int d = 0; d < D; ++d) acc[d] = 0.f;
        float accA = 0.f, T = 1.f;
        // ONE loop body for every instantiation (SAVE adds the gT store, DUMP the order stores and the tail below).
        //
        // The loop is bound by the LATENCY of one pixel's chain, not by throughput: a tile's shared memory is held
        // until its deepest pixel is done, and that pixel's warp runs mostly alone (ncu: 41 % of the warp samples
        // sit at the end-of-tile barrier, the running warps issue once per ~3 cycles).  So the body is arranged for
        // few instructions and a short dependent chain:
        //   * two register sets (A, B), the loop unrolled by two: the loads of fragment k (alpha, features) land
        //     in one set while fragment k-1 is blended out of the other -- no register is read in the half-step
        //     that loaded it;
        //   * the cut-off is tested LAZILY: fragment k+1 is selected (list advanced, loads issued) before
        //     T_{k+1} = T_k (1 - a_k) is known; the test then uses an alpha that arrived a half-step ago, and
        //     when it fails the selection is rolled back (its list steps back by one), so the cursors still
        //     count exactly the blended fragments.  The arithmetic of the test is unchanged:
        //     fragment k+1 is blended iff the fp32 product T_k (1 - a_k) >= 1e-4;
        //   * shared memory is addressed through 32-bit shared-window addresses (lds_*).
        // Invariant at the top of a half-step: the pending fragment (set X) is one that WILL be blended.
        const uint32_t sa = smem_u32(s_ab), sf = smem_u32(s_f), sk = smem_u32(s_dk);
        uint32_t kd = 0;                              // DUMP: position of the next fragment in the pixel's sorted list
        const uint32_t obase = DUMP ? A.pixoff[pix] : 0u;
        uint32_t so = SAVE ? smem_u32(s_ord) + 2u * s_pixbase[q] : 0u;   // next entry of this pixel's order list
        (void)so;
        uint32_t m01 = min(h0, h1), m23 = min(h2, h3);
        uint32_t m = min(m01, m23);
        bool p0, p1, p2, p3;
        float aA = 0.f, aB = 0.f;
        float4 fA[FV], fB[FV];
        uint32_t curA = 0, curB = 0, kdA = 0, kdB = 0;
        (void)kdA; (void)kdB;

// which list holds the minimum head; two heads with equal depth bits (rare) are resolved by point index
#define INPC_PICK()                                                                                                       \
        {                                                                                                                 \
            p0 = h0 == m; p1 = h1 == m; p2 = h2 == m; p3 = h3 == m;                                                       \
            /* two heads share the minimum iff the two pair minima are equal or a pair's heads are equal to it */       \
            if ((m01 == m23) | ((h0 == h1) & p0) | ((h2 == h3) & p2)) INPC_BLEND_RESOLVE_TIE();                           \
        }
// issue the loads of the picked fragment into set X, advance its list, recompute the minimum head
#define INPC_SELECT(X)                                                                                                    \
        {                                                                                                                 \
            const uint32_t ce = p0 ? ce0 : (p1 ? ce1 : (p2 ? ce2 : ce3));                                                 \
            cur##X = ce & 0xffffu;                                                                                        \
            const uint32_t nx = ce + 16u;                                                                                 \
            a##X = lds_f32(sa + cur##X);                                                                                  \
            _Pragma("unroll") for (int v = 0; v < FV; ++v) f##X[v] = lds_v4(sf + (cur##X & 0xfff0u) * FV + 16 * v);       \
            uint32_t nh = kSentHi;                                                                                        \
            if ((nx & 0xffffu) < (nx >> 16)) nh = lds_u32(sk + ((nx >> 2) & 0x3ffcu));                                    \
            if constexpr (DUMP) {                                                                                         \
                const uint32_t slot = (cur##X >> 4) - ((p0 | p1) ? bt : bb);                                              \
                A.sorted_idx[obase + kd] = __float_as_uint(__ldg(&A.Ra[slot]).w);                                         \
                A.sorted_depth[obase + kd] = m;                                                                           \
                kd##X = kd++;                                                                                             \
            }                                                                                                             \
            h0 = p0 ? nh : h0; ce0 = p0 ? nx : ce0;                                                                       \
            h1 = p1 ? nh : h1; ce1 = p1 ? nx : ce1;                                                                       \
            h2 = p2 ? nh : h2; ce2 = p2 ? nx : ce2;                                                                       \
            h3 = p3 ? nh : h3; ce3 = p3 ? nx : ce3;                                                                       \
            m01 = min(h0, h1); m23 = min(h2, h3); m = min(m01, m23);                                                      \
        }
// composite the pending fragment of set X (Eq. 1); lists 0, 1 (corners 3, 2: bit 3 of the cursor) lie in the top cell row
#define INPC_BLEND(X)                                                                                                     \
        {                                                                                                                 \
            const float c = T * a##X;                                                                                     \
            accA += c;                                                                                                    \
            _Pragma("unroll") for (int v = 0; v < FV; ++v) {                                                              \
                acc[4 * v] += c * f##X[v].x; acc[4 * v + 1] += c * f##X[v].y;                                             \
                acc[4 * v + 2] += c * f##X[v].z; acc[4 * v + 3] += c * f##X[v].w;                                         \
            }                                                                                                             \
            if constexpr (SAVE) { ((cur##X & 8u) ? gTtop : gTbot)[cur##X >> 2] = T; sts_u16(so, cur##X); so += 2u; }        \
            if constexpr (DUMP) A.sorted_T[obase + kd##X] = T;                                                            \
            T *= (1.f - a##X);                                                                                            \
        }
// the fragment selected into set X turned out to lie behind the cut-off: step its list (3 - corner) back by one
#define INPC_ROLLBACK(X)                                                                                                  \
        {                                                                                                                 \
            const uint32_t cj = (cur##X >> 2) & 3u;                                                                       \
            ce0 -= cj == 3u ? 16u : 0u; ce1 -= cj == 2u ? 16u : 0u; ce2 -= cj == 1u ? 16u : 0u; ce3 -= cj == 0u ? 16u : 0u; \
            if constexpr (DUMP) {                                                                                         \
                const uint32_t hk = s_dk[cur##X >> 4];                                                                    \
                h0 = cj == 3u ? hk : h0; h1 = cj == 2u ? hk : h1; h2 = cj == 1u ? hk : h2; h3 = cj == 0u ? hk : h3;       \
                m01 = min(h0, h1); m23 = min(h2, h3); m = min(m01, m23);                                                  \
                --kd;                                                                                                     \
            }                                                                                                             \
        }

        if (m != kSentHi) {
            INPC_PICK();
            INPC_SELECT(A);                           // fragment 0: T_0 = 1, always blended
            while (true) {
                if (m == kSentHi) { INPC_BLEND(A); break; }          // pending: A
                INPC_PICK();
                INPC_SELECT(B);
                INPC_BLEND(A);
                if (T < kTMin) { INPC_ROLLBACK(B); break; }
                if (m == kSentHi) { INPC_BLEND(B); break; }          // pending: B
                INPC_PICK();
                INPC_SELECT(A);
                INPC_BLEND(B);
                if (T < kTMin) { INPC_ROLLBACK(A); break; }
            }
        }
#undef INPC_SELECT
#undef INPC_BLEND
#undef INPC_ROLLBACK
        const uint4 consumed = make_uint4(((ce0 & 0xffffu) >> 4) - st0, ((ce1 & 0xffffu) >> 4) - st1,
                                          ((ce2 & 0xffffu) >> 4) - st2, ((ce3 & 0xffffu) >> 4) - st3);
        if constexpr (DUMP) {
            // order-only tail: the fragments behind the cut-off are merged on, recorded and not blended
            while (m != kSentHi) {
                INPC_PICK();
                const uint32_t ce = p0 ? ce0 : (p1 ? ce1 : (p2 ? ce2 : ce3));
                const uint32_t cur = ce & 0xffffu;
                const uint32_t nx = ce + 16u;
                const uint32_t nc = nx & 0xffffu;
                const uint32_t nh = nc < (nx >> 16) ? s_dk[nc >> 4] : kSentHi;
                const uint32_t slot = (cur >> 4) - ((p0 | p1) ? bt : bb);
                A.sorted_idx[obase + kd] = __float_as_uint(__ldg(&A.Ra[slot]).w);
                A.sorted_depth[obase + kd] = m;
                A.sorted_T[obase + kd] = -1.f;                     // not blended
                ++kd;
                h0 = p0 ? nh : h0; ce0 = p0 ? nx : ce0;
                h1 = p1 ? nh : h1; ce1 = p1 ? nx : ce1;
                h2 = p2 ? nh : h2; ce2 = p2 ? nx : ce2;
                h3 = p3 ? nh : h3; ce3 = p3 ? nx : ce3;
                m01 = min(h0, h1); m23 = min(h2, h3); m = min(m01, m23);
            }
        }
#undef INPC_PICK
        store_pixel<D>(A.io, A.out_feat, A.out_alpha, pix, acc, accA);
        if constexpr (SAVE) A.pcur[pix] = consumed;
    }
    if constexpr (SAVE) { if (tid == 0) bulk_wait_read(); }           // the last block has left shared memory
}

#undef INPC_BLEND_RESOLVE_TIE

}  // namespace inpc
