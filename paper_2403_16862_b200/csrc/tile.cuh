// tile.cuh -- steps a3/a4/a5 of the hot path for pixels up to kPixMax fragments deep.
//
// One persistent CTA per work item (a screen tile of tw x th pixels whose records fit in shared
// memory).  The tile's th+1 cell rows are contiguous ranges of the cell-sorted record array and are
// staged with cp.async.bulk (TMA, 1-D) + one mbarrier.  Then one WARP per pixel:
//   a3  segmented key sort of the pixel's fragment run by (depth bits, point index): a bitonic
//       network over the 32 lanes (shuffles) for runs <= 32, over per-warp shared scratch above.
//   a4  front-to-back compositing, Eq. 1: 32 fragments per step, warp-level inclusive
//       prefix product of (1 - a), T >= 1e-4 prefix mask, per-lane partial sums, one reduction.
//   a5  backward: the run is re-sorted (nothing but the records is saved), T is
//       rebuilt front to back, then chunks are walked back to front with a warp-level suffix scan of
//       the affine maps B -> a G + (1-a) B (division-free).  Per-fragment (T a, dL/da) go to a
//       shared-memory slot per (record, corner); after the tile is done each record combines its four
//       corners with the bilinear weights and is written once -- plain stores when all
//       its pixels belong to this tile, red.global.add only for the tile-straddling ones.
#pragma once
#include "common.cuh"

namespace inpc {

enum TileMode { kFwd = 0, kFwdDump = 1, kBwd = 2 };

struct TileArgs {
    const Header* hdr;
    uint32_t* item_cursor;
    const uint32_t* items;
    const uint32_t* celloff;
    const float4* rec;
    const float* rop;
    int W, H;
    // forward
    float* out_feat;
    float* out_alpha;
    // dump (INPC_SAVE_SORTED)
    const uint32_t* pixoff;
    uint32_t* sorted_idx;
    uint32_t* sorted_depth;
    // backward
    const float* g_feat;
    const float* g_alpha;
    float* d_feat;
    float* d_opacity;
    float* d_uv;
};

template <int D> __host__ __device__ constexpr int tile_rec_bytes() { return 16 + 4 * D; }
template <int D, int MODE> __host__ __device__ constexpr size_t tile_smem_bytes() {
    size_t b = (size_t)TileCfg<D>::kCap * tile_rec_bytes<D>()      // records
               + (size_t)TileCfg<D>::kCap * 4                       // opacities
               + (size_t)kTileWarps * kPixMax * 8;                  // per-warp sort scratch
    if (MODE == kBwd) b += (size_t)TileCfg<D>::kCap * 4 * 8;        // (T a, dL/da) per (record, corner)
    return b;
}

// (depth, idx) order on packed keys  depth_bits << 32 | (ref << 2 | corner);  a != b assumed.
__device__ __forceinline__ bool key_less(unsigned long long a, unsigned long long b, const float4* s_rec, int RV) {
    const uint32_t da = (uint32_t)(a >> 32), db = (uint32_t)(b >> 32);
    if (da != db) return da < db;
    // equal depth bits (rare): tie-break by point index, fetched from the staged records
    const uint32_t ia = __float_as_uint(s_rec[(((uint32_t)a) >> 2) * RV].y);
    const uint32_t ib = __float_as_uint(s_rec[(((uint32_t)b) >> 2) * RV].y);
    return ia < ib;
}

__device__ __forceinline__ float warp_incl_prod(float v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const float t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v *= t;
    }
    return v;
}

template <int D, int MODE>
__global__ void __launch_bounds__(kTileThreads) k_tile(TileArgs A) {
    constexpr int RV  = 1 + D / 4;                 // float4 per record
    constexpr int CAP = TileCfg<D>::kCap;
    extern __shared__ __align__(128) unsigned char smem[];
    float4* s_rec = reinterpret_cast<float4*>(smem);
    float*  s_op  = reinterpret_cast<float*>(smem + (size_t)CAP * RV * 16);
    unsigned long long* s_sort_all = reinterpret_cast<unsigned long long*>(smem + (size_t)CAP * RV * 16 + (size_t)CAP * 4);
    float2* s_frag = reinterpret_cast<float2*>(smem + (size_t)CAP * RV * 16 + (size_t)CAP * 4 + (size_t)kTileWarps * kPixMax * 8);

    __shared__ uint32_t s_off[kTileH + 1][kTileW + 2];
    __shared__ uint32_t s_sbase[kTileH + 1], s_a4[kTileH + 1], s_ra[kTileH + 1], s_rb[kTileH + 1];
    __shared__ uint32_t s_item, s_tot;
    __shared__ __align__(8) uint64_t s_bar;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned long long* s_sort = s_sort_all + warp * kPixMax;
    const int W = A.W, H = A.H;
    const uint32_t n_items = A.hdr->n_items;

    if (tid == 0) { mbar_init(&s_bar, 1); fence_mbar_init(); }
    uint32_t parity = 0;

    while (true) {
        if (tid == 0) s_item = atomicAdd(A.item_cursor, 1u);
        __syncthreads();
        const uint32_t item_i = s_item;
        if (item_i >= n_items) break;
        const uint32_t it = A.items[item_i];
        const int X = it & 0xfff, Y = (it >> 12) & 0xfff, lw = (it >> 24) & 7, lh = (it >> 27) & 3;
        const int tw = 1 << lw, th = 1 << lh;

        // cell offsets of the tile's (th+1) x (tw+2) window
        if (tid < (th + 1) * (tw + 2)) {
            const int r = tid / (tw + 2), c = tid - r * (tw + 2);
            const int j = Y + r;
            uint32_t v = 0;
            if (j <= H) v = __ldg(&A.celloff[(uint32_t)j * (W + 1) + min(X + c, W + 1)]);
            s_off[r][c] = v;
        }
        __syncthreads();
        if (tid == 0) {
            uint32_t tot = 0;
            for (int r = 0; r <= th; ++r) {
                const uint32_t a = s_off[r][0], b = s_off[r][tw + 1];
                const uint32_t a4 = a & ~3u, b4 = (b + 3u) & ~3u;
                s_ra[r] = a; s_rb[r] = b; s_a4[r] = a4; s_sbase[r] = tot;
                tot += (b > a) ? (b4 - a4) : 0u;
            }
            s_tot = tot;
            if (tot > 0) {
                fence_proxy_async();
                mbar_arrive_expect_tx(&s_bar, tot * (uint32_t)(RV * 16 + 4));
                for (int r = 0; r <= th; ++r) {
                    const uint32_t a = s_ra[r], b = s_rb[r];
                    if (b <= a) continue;
                    const uint32_t a4 = s_a4[r], len = ((b + 3u) & ~3u) - a4;
                    bulk_g2s(s_rec + (size_t)s_sbase[r] * RV, A.rec + (size_t)a4 * RV, len * RV * 16, &s_bar);
                    bulk_g2s(s_op + s_sbase[r], A.rop + a4, len * 4, &s_bar);
                }
            }
        }
        __syncthreads();
        const uint32_t tot = s_tot;
        if (MODE == kBwd) {
            float4* z = reinterpret_cast<float4*>(s_frag);
            for (uint32_t q = tid; q < tot * 2; q += kTileThreads) z[q] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (tot > 0) { mbar_wait(&s_bar, parity); parity ^= 1u; }
        if (MODE == kBwd) __syncthreads();

        // ---------------------------------------------------------------- one warp per pixel
        for (int q = warp; q < tw * th; q += kTileWarps) {
            const int ly = q >> lw, lx = q & (tw - 1);
            const int x = X + lx, y = Y + ly;
            if (x >= W || y >= H) continue;
            const uint32_t o00 = s_off[ly][lx], o01 = s_off[ly][lx + 1], o02 = s_off[ly][lx + 2];
            const uint32_t o10 = s_off[ly + 1][lx], o11 = s_off[ly + 1][lx + 1], o12 = s_off[ly + 1][lx + 2];
            const uint32_t n0 = o02 - o00, n = n0 + (o12 - o10);
            const size_t pix = (size_t)y * W + x;
            if (n > (uint32_t)kPixMax) continue;                 // long-run path owns this pixel
            if (n == 0) {
                if (MODE != kBwd && lane == 0) {
#pragma unroll
                    for (int v = 0; v < D / 4; ++v) reinterpret_cast<float4*>(A.out_feat + pix * D)[v] = make_float4(0.f, 0.f, 0.f, 0.f);
                    A.out_alpha[pix] = 0.f;
                }
                continue;
            }
            // fragment l of the run -> (record in smem, corner): cell row y first (dy = 1), then row y+1
            auto make_key = [&](uint32_t l) -> unsigned long long {
                uint32_t g, row, dy, dx;
                if (l < n0) { g = o00 + l; row = ly; dy = 1u; dx = g < o01 ? 1u : 0u; }
                else        { g = o10 + (l - n0); row = ly + 1; dy = 0u; dx = g < o11 ? 1u : 0u; }
                const uint32_t ref = s_sbase[row] + (g - s_a4[row]);
                const uint32_t depth = __float_as_uint(s_rec[ref * RV].x);
                return ((unsigned long long)depth << 32) | (unsigned long long)((ref << 2) | (dy << 1) | dx);
            };

            // ------------------------------------------------------------ a3: sort
            unsigned long long rkey = ~0ull;
            if (n <= 32) {
                if ((uint32_t)lane < n) rkey = make_key(lane);
                for (uint32_t k = 2; (k >> 1) < n; k <<= 1) {
                    {   // flip stage: partner = lane ^ (k-1)
                        const unsigned long long o = __shfl_xor_sync(0xffffffffu, rkey, k - 1);
                        const bool lower = (lane & (k >> 1)) == 0;
                        bool take = false;
                        if (o != rkey) take = lower ? key_less(o, rkey, s_rec, RV) : key_less(rkey, o, s_rec, RV);
                        if (take) rkey = o;
                    }
                    for (uint32_t j = k >> 2; j > 0; j >>= 1) {
                        const unsigned long long o = __shfl_xor_sync(0xffffffffu, rkey, j);
                        const bool lower = (lane & j) == 0;
                        bool take = false;
                        if (o != rkey) take = lower ? key_less(o, rkey, s_rec, RV) : key_less(rkey, o, s_rec, RV);
                        if (take) rkey = o;
                    }
                }
            } else {
                for (uint32_t l = lane; l < n; l += 32) s_sort[l] = make_key(l);
                __syncwarp();
                uint32_t np2 = 64; while (np2 < n) np2 <<= 1;
                for (uint32_t k = 2; k <= np2; k <<= 1) {
                    const uint32_t hk = k >> 1;
                    for (uint32_t c = lane; c < (np2 >> 1); c += 32) {       // flip stage
                        const uint32_t i = ((c / hk) * k) + (c & (hk - 1));
                        const uint32_t l = i ^ (k - 1);
                        if (l < n) {
                            const unsigned long long a = s_sort[i], b = s_sort[l];
                            if (key_less(b, a, s_rec, RV)) { s_sort[i] = b; s_sort[l] = a; }
                        }
                    }
                    __syncwarp();
                    for (uint32_t j = k >> 2; j > 0; j >>= 1) {
                        for (uint32_t c = lane; c < (np2 >> 1); c += 32) {
                            const uint32_t i = ((c / j) * (j << 1)) + (c & (j - 1));
                            const uint32_t l = i + j;
                            if (l < n) {
                                const unsigned long long a = s_sort[i], b = s_sort[l];
                                if (key_less(b, a, s_rec, RV)) { s_sort[i] = b; s_sort[l] = a; }
                            }
                        }
                        __syncwarp();
                    }
                }
            }

            // per-lane fragment fetch for chunk base `cb`: returns a (= opacity * w) and fills refs
            auto fetch = [&](uint32_t cb, uint32_t& ref, uint32_t& corner, float& a, float& op, float4& k4) -> bool {
                const uint32_t kk = cb + lane;
                const bool valid = kk < n;
                unsigned long long key = ~0ull;
                if (valid) key = (n <= 32) ? rkey : s_sort[kk];
                ref = ((uint32_t)key) >> 2; corner = ((uint32_t)key) & 3u;
                a = 0.f; op = 0.f; k4 = make_float4(0.f, 0.f, 0.f, 0.f);
                if (valid) {
                    k4 = s_rec[ref * RV];
                    op = s_op[ref];
                    const float wx = (corner & 1u) ? k4.z : 1.f - k4.z;
                    const float wy = (corner & 2u) ? k4.w : 1.f - k4.w;
                    a = op * (wx * wy);
                }
                return valid;
            };

            if (MODE != kBwd) {
                // -------------------------------------------------------- a4: front-to-back blend
                float acc[D]; float accA = 0.f;
#pragma unroll
                for (int d = 0; d < D; ++d) acc[d] = 0.f;
                float T_in = 1.f;
                const uint32_t obase = (MODE == kFwdDump) ? A.pixoff[pix] : 0u;
                for (uint32_t cb = 0; cb < n; cb += 32) {
                    uint32_t ref, corner; float a, op; float4 k4;
                    const bool valid = fetch(cb, ref, corner, a, op, k4);
                    const float incl = warp_incl_prod(1.f - a, lane);
                    float excl = __shfl_up_sync(0xffffffffu, incl, 1);
                    if (lane == 0) excl = 1.f;
                    const float T = T_in * excl;
                    if (valid && T >= kTMin) {
                        const float c = T * a;
                        accA += c;
#pragma unroll
                        for (int v = 0; v < D / 4; ++v) {
                            const float4 f = s_rec[ref * RV + 1 + v];
                            acc[4 * v] += c * f.x; acc[4 * v + 1] += c * f.y; acc[4 * v + 2] += c * f.z; acc[4 * v + 3] += c * f.w;
                        }
                    }
                    if (MODE == kFwdDump && valid) {
                        A.sorted_idx[obase + cb + lane] = __float_as_uint(k4.y);
                        A.sorted_depth[obase + cb + lane] = __float_as_uint(k4.x);
                    }
                    T_in *= __shfl_sync(0xffffffffu, incl, 31);
                    if (MODE != kFwdDump && T_in < kTMin) break;     // T is monotone: nothing behind is blended
                }
#pragma unroll
                for (int s = 16; s > 0; s >>= 1) {
                    accA += __shfl_xor_sync(0xffffffffu, accA, s);
#pragma unroll
                    for (int d = 0; d < D; ++d) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], s);
                }
                if (lane == 0) {
#pragma unroll
                    for (int v = 0; v < D / 4; ++v)
                        reinterpret_cast<float4*>(A.out_feat + pix * D)[v] = make_float4(acc[4 * v], acc[4 * v + 1], acc[4 * v + 2], acc[4 * v + 3]);
                    A.out_alpha[pix] = accA;
                }
            } else {
                // -------------------------------------------------------- a5: backward
                float g[D];
#pragma unroll
                for (int v = 0; v < D / 4; ++v) {
                    const float4 t = __ldg(reinterpret_cast<const float4*>(A.g_feat + pix * D) + v);
                    g[4 * v] = t.x; g[4 * v + 1] = t.y; g[4 * v + 2] = t.z; g[4 * v + 3] = t.w;
                }
                const float gA = A.g_alpha ? __ldg(A.g_alpha + pix) : 0.f;
                // front-to-back: transmittance entering every 32-fragment chunk (lane c keeps chunk c's)
                float tin_reg = 0.f, T_in = 1.f;
                int last = -1;
                const int nchunks = (int)((n + 31) >> 5);
                for (int c = 0; c < nchunks; ++c) {
                    if (lane == c) tin_reg = T_in;
                    if (T_in < kTMin) break;
                    last = c;
                    if (c + 1 < nchunks) {
                        uint32_t ref, corner; float a, op; float4 k4;
                        fetch((uint32_t)c << 5, ref, corner, a, op, k4);
                        const float incl = warp_incl_prod(1.f - a, lane);
                        T_in *= __shfl_sync(0xffffffffu, incl, 31);
                    }
                }
                // back-to-front
                float B_in = 0.f;
                for (int c = last; c >= 0; --c) {
                    const float Tc = __shfl_sync(0xffffffffu, tin_reg, c);
                    uint32_t ref, corner; float a, op; float4 k4;
                    const bool valid = fetch((uint32_t)c << 5, ref, corner, a, op, k4);
                    const float incl = warp_incl_prod(1.f - a, lane);
                    float excl = __shfl_up_sync(0xffffffffu, incl, 1);
                    if (lane == 0) excl = 1.f;
                    const float T = Tc * excl;
                    const bool bl = valid && T >= kTMin;
                    float G = gA;
                    if (bl) {
#pragma unroll
                        for (int v = 0; v < D / 4; ++v) {
                            const float4 f = s_rec[ref * RV + 1 + v];
                            G += f.x * g[4 * v] + f.y * g[4 * v + 1] + f.z * g[4 * v + 2] + f.w * g[4 * v + 3];
                        }
                    }
                    // suffix scan of the affine maps  phi_l(B) = a_l G_l + (1 - a_l) B
                    float M = bl ? 1.f - a : 1.f, C = bl ? a * G : 0.f;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const float M2 = __shfl_down_sync(0xffffffffu, M, d);
                        const float C2 = __shfl_down_sync(0xffffffffu, C, d);
                        if (lane + d < 32) { C = C + M * C2; M = M * M2; }
                    }
                    const float Mn = __shfl_down_sync(0xffffffffu, M, 1), Cn = __shfl_down_sync(0xffffffffu, C, 1);
                    const float B = lane < 31 ? Cn + Mn * B_in : B_in;
                    if (bl) s_frag[ref * 4 + corner] = make_float2(T * a, T * (G - B));
                    B_in = __shfl_sync(0xffffffffu, C, 0) + __shfl_sync(0xffffffffu, M, 0) * B_in;
                }
            }
        }

        if (MODE == kBwd) {
            // ------------------------------------------------------------ per-record combine
            __syncthreads();
            for (uint32_t r = tid; r < tot; r += kTileThreads) {
                int row = 0;
                while (row < th && r >= s_sbase[row + 1]) ++row;
                const uint32_t gidx = s_a4[row] + (r - s_sbase[row]);
                if (gidx < s_ra[row] || gidx >= s_rb[row]) continue;          // alignment padding
                int col = 0;                                                   // last col with s_off[row][col] <= gidx
                while (col < tw && s_off[row][col + 1] <= gidx) ++col;
                const int x0 = X + col - 1, y0 = Y + row - 1;
                const float4 k4 = s_rec[r * RV];
                const float op = s_op[r];
                const uint32_t idx = __float_as_uint(k4.y);
                const float tx = k4.z, ty = k4.w;
                float df[D];
#pragma unroll
                for (int d = 0; d < D; ++d) df[d] = 0.f;
                float dop = 0.f, du = 0.f, dv = 0.f;
                bool complete = true;
#pragma unroll
                for (int c = 0; c < 4; ++c) {
                    const int dx = c & 1, dy = c >> 1;
                    const int px = x0 + dx, py = y0 + dy;
                    if (px < 0 || px >= W || py < 0 || py >= H) continue;      // fragment does not exist
                    if (px < X || px >= X + tw || py < Y || py >= Y + th) { complete = false; continue; }
                    const float2 fr = s_frag[r * 4 + c];
                    const float wx = dx ? tx : 1.f - tx, wy = dy ? ty : 1.f - ty;
                    dop += wx * wy * fr.y;
                    du += (dx ? wy : -wy) * fr.y;
                    dv += (dy ? wx : -wx) * fr.y;
                    if (fr.x != 0.f) {
                        const size_t pp = (size_t)py * W + px;
#pragma unroll
                        for (int v = 0; v < D / 4; ++v) {
                            const float4 t = __ldg(reinterpret_cast<const float4*>(A.g_feat + pp * D) + v);
                            df[4 * v] += fr.x * t.x; df[4 * v + 1] += fr.x * t.y; df[4 * v + 2] += fr.x * t.z; df[4 * v + 3] += fr.x * t.w;
                        }
                    }
                    // a pixel deeper than kPixMax is owned by the long-run path, which adds atomically later
                    if (complete) {
                        const int qx = px - X, qy = py - Y;
                        const uint32_t np = (s_off[qy][qx + 2] - s_off[qy][qx]) + (s_off[qy + 1][qx + 2] - s_off[qy + 1][qx]);
                        if (np > (uint32_t)kPixMax) complete = false;
                    }
                }
                du *= op; dv *= op;
                float* pf = A.d_feat + (size_t)idx * D;
                if (complete) {
#pragma unroll
                    for (int v = 0; v < D / 4; ++v)
                        reinterpret_cast<float4*>(pf)[v] = make_float4(df[4 * v], df[4 * v + 1], df[4 * v + 2], df[4 * v + 3]);
                    A.d_opacity[idx] = dop;
                    reinterpret_cast<float2*>(A.d_uv)[idx] = make_float2(du, dv);
                } else {
#pragma unroll
                    for (int v = 0; v < D / 4; ++v) red_add_v4(pf + 4 * v, df[4 * v], df[4 * v + 1], df[4 * v + 2], df[4 * v + 3]);
                    red_add(A.d_opacity + idx, dop);
                    red_add_v2(A.d_uv + 2 * (size_t)idx, du, dv);
                }
            }
        }
    }
}

}  // namespace inpc
