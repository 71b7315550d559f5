// bin.cuh -- steps a1/a2 of the hot path: projection, per-cell counting, device-wide scan, record
// emission, per-pixel counts and tile work-list construction.
//
// Path rows (SURVEY.md section 8a / DESIGN.md section 1):
//   a1  k_project_count + k_scatter : Eq. 6 projection, cull, bilinear cell + fractions (Eq. 7 inputs)
//   a2  k_project_count (count), k_scan_u32 (device-wide exclusive scan, decoupled look-back),
//       k_classify (per-pixel fragment counts = 2x2 box sum of the cell counts)
#pragma once
#include "common.cuh"
#include "sh.cuh"

namespace inpc {

constexpr int kBinThreads = 256;
constexpr int kBinPPT     = 4;                          // points per thread
constexpr int kBinChunk   = kBinThreads * kBinPPT;      // points per CTA iteration

// Coalesced, vectorised staging of a chunk of positions: 3*chunk floats = 768 float4 -> smem.
__device__ __forceinline__ void stage_positions(const float* __restrict__ pos, long long base, long long N,
                                                float* s_pos) {
    const long long f0 = base * 3;                      // first float of the chunk (multiple of 4)
    const long long fend = N * 3;
    for (int v = threadIdx.x; v < kBinChunk * 3 / 4; v += kBinThreads) {
        const long long f = f0 + 4ll * v;
        float4 q;
        if (f + 3 < fend) {
            q = __ldcs(reinterpret_cast<const float4*>(pos + f));
        } else {
            q.x = f + 0 < fend ? pos[f + 0] : 0.f;
            q.y = f + 1 < fend ? pos[f + 1] : 0.f;
            q.z = f + 2 < fend ? pos[f + 2] : 0.f;
            q.w = 0.f;
        }
        reinterpret_cast<float4*>(s_pos)[v] = q;
    }
}

// a1 + a2: project every point and bump its cell counter with a fire-and-forget reduction (RED: no return
// value, so the pass is bound by reading the positions, not by atomic latency).  One global atomic per
// POINT (not per fragment): the 2x2 footprint is implied by the cell.  kept[i / 32] bit i % 32 = point i
// survived the cull (read by k_split).
__global__ void __launch_bounds__(kBinThreads) k_project_count(const float* __restrict__ pos, long long N,
                                                                Camera cam, uint32_t* __restrict__ cellcnt,
                                                                uint32_t* __restrict__ kept) {
    __shared__ __align__(16) float s_pos[kBinChunk * 3];
    for (long long base = (long long)blockIdx.x * kBinChunk; base < N; base += (long long)gridDim.x * kBinChunk) {
        __syncthreads();
        stage_positions(pos, base, N, s_pos);
        __syncthreads();
#pragma unroll
        for (int k = 0; k < kBinPPT; ++k) {
            const int l = k * kBinThreads + threadIdx.x;
            const long long i = base + l;                // a warp's lanes hold 32 consecutive, 32-aligned points
            int cell = -1;
            if (i < N) cell = project_point(cam, s_pos[3 * l], s_pos[3 * l + 1], s_pos[3 * l + 2]).cell;
            if (cell >= 0) atomicAdd(&cellcnt[cell], 1u);
            const uint32_t mask = __ballot_sync(0xffffffffu, cell >= 0);
            if ((threadIdx.x & 31) == 0 && i < N) kept[i >> 5] = mask;
        }
    }
}

// a1 (emission): re-project (bit-identical to the count pass), take the point's slot from a returning atomic
// on cursor[cell] (a copy of the exclusive cell offsets, so slots of a cell are handed out in arrival order;
// afterwards cursor[c] == celloff[c + 1]) and write ONE full 32-byte sector per point:
// { depth_bits, idx, tx, ty | opacity, cell, 0, 0 }.  (Anything narrower than a sector scattered by slot costs a
// DRAM read-modify-write: DESIGN.md section 10, round-1 facts.)  All of a thread's atomics and opacity loads are
// issued before the first store.
// SH (NEXT row f2, sh.cuh): the pass also evaluates every kept point's view-dependent feature from its 36 SH
// coefficients (read once, here, coalesced) and leaves it in shfeat[point] for the cell sort to pick up.
template <bool SH>
__global__ void __launch_bounds__(kBinThreads) k_scatter(const float* __restrict__ pos,
                                                          const float* __restrict__ opacity, long long N, Camera cam,
                                                          uint32_t* __restrict__ cursor, float4* __restrict__ A,
                                                          const float4* __restrict__ sh_coeff, ViewPoint view,
                                                          float4* __restrict__ shfeat) {
    __shared__ __align__(16) float s_pos[kBinChunk * 3];
    for (long long base = (long long)blockIdx.x * kBinChunk; base < N; base += (long long)gridDim.x * kBinChunk) {
        __syncthreads();
        stage_positions(pos, base, N, s_pos);
        __syncthreads();
        uint32_t slot[kBinPPT];
        float op[kBinPPT];
        Proj p[kBinPPT];
#pragma unroll
        for (int k = 0; k < kBinPPT; ++k) {
            const int l = k * kBinThreads + threadIdx.x;
            p[k] = project_point(cam, s_pos[3 * l], s_pos[3 * l + 1], s_pos[3 * l + 2]);   // padding -> culled
        }
#pragma unroll
        for (int k = 0; k < kBinPPT; ++k) {
            const bool live = p[k].cell >= 0;
            slot[k] = live ? atomicAdd(&cursor[p[k].cell], 1u) : 0u;
            op[k] = live ? __ldcs(&opacity[base + k * kBinThreads + threadIdx.x]) : 0.f;
        }
#pragma unroll
        for (int k = 0; k < kBinPPT; ++k) {
            if (p[k].cell < 0) continue;
            const long long i = base + k * kBinThreads + threadIdx.x;
            float4 a0, a1;
            a0.x = __uint_as_float(p[k].depth_bits);
            a0.y = __uint_as_float((uint32_t)i);
            a0.z = p[k].tx;
            a0.w = p[k].ty;
            a1.x = op[k];
            a1.y = __uint_as_float((uint32_t)p[k].cell);
            a1.z = 0.f; a1.w = 0.f;
            st_sector(A + 2 * (size_t)slot[k], a0, a1);         // one 256-bit store = the whole 32-byte sector
            if (SH) {
                const int l = k * kBinThreads + threadIdx.x;
                shfeat[i] = sh_feature(sh_coeff + (size_t)i * kShBasis, s_pos[3 * l] - view.cx, s_pos[3 * l + 1] - view.cy,
                                       s_pos[3 * l + 2] - view.cz);
            }
        }
    }
}

// ---- a2: device-wide exclusive scan, single pass with decoupled look-back ---------------------------
// data[0..n) -> exclusive prefix sums in place; data[n] = total.  status[] (one u64 per tile) and
// *tile_counter must be zero on entry.  Tiles are claimed through an atomic ticket so that a tile only
// ever waits on tiles that are already running (forward progress without co-residency assumptions).
constexpr int kScanThreads = 256;
constexpr int kScanItems   = 16;
constexpr int kScanTile    = kScanThreads * kScanItems;

__global__ void __launch_bounds__(kScanThreads) k_scan_u32(uint32_t* __restrict__ data, uint32_t n,
                                                            unsigned long long* __restrict__ status,
                                                            uint32_t* __restrict__ tile_counter,
                                                            uint32_t* __restrict__ total_out,
                                                            uint32_t* __restrict__ copy_out) {
    __shared__ uint32_t s_tile;
    __shared__ uint32_t s_warp[kScanThreads / 32];
    __shared__ uint32_t s_prefix;
    if (threadIdx.x == 0) s_tile = atomicAdd(tile_counter, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const uint32_t base = tile * kScanTile + threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
    if (base + kScanItems <= n) {
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q) {
            const uint4 t = reinterpret_cast<const uint4*>(data + base)[q];
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
    } else {
#pragma unroll
        for (int q = 0; q < kScanItems; ++q) v[q] = base + q < n ? data[base + q] : 0u;
    }
    uint32_t sum = 0;
#pragma unroll
    for (int q = 0; q < kScanItems; ++q) { const uint32_t t = v[q]; v[q] = sum; sum += t; }
    // block-wide exclusive scan of the per-thread sums
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t inc = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < kScanThreads / 32 ? s_warp[lane] : 0u;
#pragma unroll
        for (int d = 1; d < kScanThreads / 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, w, d); if (lane >= d) w += t; }
        if (lane < kScanThreads / 32) s_warp[lane] = w;                       // inclusive over warps
        const uint32_t aggregate = __shfl_sync(0xffffffffu, w, kScanThreads / 32 - 1);
        // publish the aggregate, then look back
        volatile unsigned long long* st = status;
        if (lane == 0) {
            const unsigned long long flag = tile == 0 ? 2ull : 1ull;
            st[tile] = (flag << 62) | aggregate;
            __threadfence();
        }
        uint32_t prefix = 0;
        if (tile > 0) {
            int look = (int)tile - 1;
            while (true) {                                                     // warp-wide window of 32 predecessors
                const int idx = look - lane;
                unsigned long long s = idx >= 0 ? st[idx] : (2ull << 62);
                while (__any_sync(0xffffffffu, (s >> 62) == 0ull)) { s = idx >= 0 ? st[idx] : (2ull << 62); }
                const uint32_t incl_mask = __ballot_sync(0xffffffffu, (s >> 62) == 2ull);
                const int first_incl = incl_mask ? __ffs(incl_mask) - 1 : 32;  // nearest tile with an inclusive prefix
                uint32_t contrib = lane <= first_incl ? (uint32_t)(s & 0xffffffffull) : 0u;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) contrib += __shfl_xor_sync(0xffffffffu, contrib, d);
                prefix += contrib;
                if (incl_mask) break;
                look -= 32;
            }
            if (lane == 0) {
                __threadfence();
                st[tile] = (2ull << 62) | (unsigned long long)(prefix + aggregate);
            }
        }
        if (lane == 0) {
            s_prefix = prefix;
            if ((tile + 1) * (unsigned long long)kScanTile >= n) {             // last tile: total
                data[n] = prefix + aggregate;
                if (total_out) *total_out = prefix + aggregate;
            }
        }
    }
    __syncthreads();
    const uint32_t off = s_prefix + (warp > 0 ? s_warp[warp - 1] : 0u) + (inc - sum);
    if (base + kScanItems <= n) {
#pragma unroll
        for (int q = 0; q < kScanItems / 4; ++q)
        {
            const uint4 o4 = make_uint4(v[4 * q] + off, v[4 * q + 1] + off, v[4 * q + 2] + off, v[4 * q + 3] + off);
            reinterpret_cast<uint4*>(data + base)[q] = o4;
            if (copy_out) reinterpret_cast<uint4*>(copy_out + base)[q] = o4;     // second copy (the scatter's slot cursors)
        }
    } else {
#pragma unroll
        for (int q = 0; q < kScanItems; ++q)
            if (base + q < n) { data[base + q] = v[q] + off; if (copy_out) copy_out[base + q] = v[q] + off; }
    }
}

// ---- a2: per-pixel fragment counts (2x2 box sum of the cell counts) ---------------------------------
__device__ __forceinline__ uint32_t pixel_count(const uint32_t* __restrict__ celloff, int W, int x, int y) {
    const uint32_t c0 = (uint32_t)y * (W + 1) + x, c1 = c0 + (W + 1);
    return (__ldg(&celloff[c0 + 2]) - __ldg(&celloff[c0])) + (__ldg(&celloff[c1 + 2]) - __ldg(&celloff[c1]));
}

// One thread per CELL index c = j (W+1) + i: the fragment count of pixel (i, j) when it is inside the
// image (total, optional count image) and the list of cells too large for the counting sort.
__global__ void __launch_bounds__(256) k_classify(const uint32_t* __restrict__ celloff, int W, int H,
                                                   Header* __restrict__ hdr, BigCell* __restrict__ bigcells,
                                                   uint32_t* __restrict__ pixcnt) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    const int C = (W + 1) * (H + 1);
    uint32_t n = 0;
    if (c < C) {
        const int j = c / (W + 1), i = c - j * (W + 1);
        if (i < W && j < H) {
            n = pixel_count(celloff, W, i, j);
            if (pixcnt) pixcnt[j * W + i] = n;
        }
        const uint32_t a = __ldg(&celloff[c]), m = __ldg(&celloff[c + 1]) - a;
        if (m > (uint32_t)kCellSmall) {
            BigCell e; e.cell = (uint32_t)c; e.start = a; e.n = m; e.pad = 0;
            bigcells[atomicAdd(&hdr->n_big_cells, 1u)] = e;
        }
    }
    // block reduction of n -> one 64-bit atomic per CTA
    unsigned long long s = n;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    __shared__ unsigned long long s_sum[8];
    if ((threadIdx.x & 31) == 0) s_sum[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long t = 0;
        for (int w = 0; w < 8; ++w) t += s_sum[w];
        if (t) atomicAdd(&hdr->n_fragments, t);
    }
}

__global__ void __launch_bounds__(256) k_counts_out(const uint32_t* __restrict__ celloff, int W, int H,
                                                     uint32_t* __restrict__ counts) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < W * H) { const int y = p / W; counts[p] = pixel_count(celloff, W, p - y * W, y); }
}

// Per-pixel blended fragment count = the four list positions at which the forward pass stopped (pcur).
__global__ void __launch_bounds__(256) k_blended_out(const uint4* __restrict__ pcur, uint32_t P, uint32_t* __restrict__ out) {
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p < P) { const uint4 c = pcur[p]; out[p] = c.x + c.y + c.z + c.w; }
}

// Records a tile item of tw x th pixels at (X, Y) stages into shared memory: each of its th+1 cell
// rows is one contiguous slot range, widened to multiples of 4 records (16-byte bulk copies of dk).
__device__ __forceinline__ uint32_t tile_padded_records(const uint32_t* __restrict__ celloff, int W, int H, int X,
                                                        int Y, int tw, int th) {
    uint32_t tot = 0;
    for (int r = 0; r <= th; ++r) {
        const int j = Y + r;
        if (j > H) break;
        const uint32_t rowbase = (uint32_t)j * (W + 1);
        const uint32_t a = __ldg(&celloff[rowbase + min(X, W + 1)]);
        const uint32_t b = __ldg(&celloff[rowbase + min(X + tw + 1, W + 1)]);
        if (b > a) tot += ((b + 3u) & ~3u) - (a & ~3u);
    }
    return tot;
}

// One thread per base tile: emit it if its records fit the shared-memory capacity, otherwise halve
// its larger side and retry.  A sub-tile of kMinTilePix pixels or fewer that still does not fit sends
// its pixels to the long-run list (they are merged straight from global memory, big.cuh).
// Bands: tile row r belongs to band min(r / rows_per_band, n_bands - 1); band b's items go to items + band_base[b].
struct BandPlan {
    int n_bands, rows_per_band;
    uint32_t item_base[kMaxBands];       // start of the band's item list inside items[]
};

// Two passes over the same DFS: the first counts what the thread's base tile will emit, the warp then reserves the
// slots of all its lanes with ONE atomic per list (thousands of single-slot atomics on one address serialise:
// 122 us on the stress workload), the second writes.
__global__ void __launch_bounds__(128) k_build_items(const uint32_t* __restrict__ celloff, int W, int H, int cap,
                                                      BandPlan plan, Header* __restrict__ hdr,
                                                      uint32_t* __restrict__ items_all, uint32_t* __restrict__ bigpix) {
    const int ntx = (W + kTileW - 1) / kTileW, nty = (H + kTileH - 1) / kTileH;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = t < ntx * nty;
    const int tt = live ? t : 0;
    const int X0 = (tt % ntx) * kTileW, Y0 = (tt / ntx) * kTileH;
    const int band = min((tt / ntx) / plan.rows_per_band, plan.n_bands - 1);
    uint32_t* items = items_all + plan.item_base[band];
    uint32_t n_it = 0, n_bp = 0, at_it = 0, at_bp = 0;
    unsigned long long n_bf = 0;
    const int lane = threadIdx.x & 31;
    for (int pass = 0; pass < 2; ++pass) {
        uint32_t stack[12];                              // binary DFS: depth <= 7, one sibling pending per level
        int sp = 0;
        if (live) stack[sp++] = encode_item(X0, Y0, kTileLW, kTileLH);
        while (sp > 0) {
            const uint32_t it = stack[--sp];
            const int X = it & 0xfff, Y = (it >> 12) & 0xfff, lw = (it >> 24) & 7, lh = (it >> 27) & 3;
            if (X >= W || Y >= H) continue;
            const int tw = 1 << lw, th = 1 << lh;
            const uint32_t n = tile_padded_records(celloff, W, H, X, Y, tw, th);
            if (n <= (uint32_t)cap) {                    // empty tiles too: their pixels must be zeroed
                if (pass == 0) ++n_it; else items[at_it++] = it;
                continue;
            }
            // a small sub-tile that still does not fit: its pixels go to the long-run path -- unless it misses the capacity by
            // less than half, in which case halving it further (down to one pixel) keeps its pixels in shared memory
            // (infer: 1784 such pixels cost 226 us as long runs, one thread each and every step a round trip to L2, and 7 us
            // as small tiles: forward 4.36 -> 4.12 ms; stress: a cluster pixel has 10^3..10^4 fragments of which the cut-off
            // keeps ~10^2, staging them all would be the waste, and the long-run path has 2 x 10^4 pixels to overlap)
            if (tw * th <= kMinTilePix && (n > (uint32_t)cap + (uint32_t)cap / 2u || tw * th == 1)) {
                for (int y = Y; y < min(Y + th, H); ++y)
                    for (int x = X; x < min(X + tw, W); ++x) {
                        if (pass == 0) { ++n_bp; n_bf += pixel_count(celloff, W, x, y); }
                        else bigpix[at_bp++] = (uint32_t)(y * W + x);
                    }
                continue;
            }
            if (lw >= lh + 1 || lh == 0) {               // split the wider side (tiles are kept ~2:1)
                stack[sp++] = encode_item(X + (tw >> 1), Y, lw - 1, lh);
                stack[sp++] = encode_item(X, Y, lw - 1, lh);
            } else {
                stack[sp++] = encode_item(X, Y + (th >> 1), lw, lh - 1);
                stack[sp++] = encode_item(X, Y, lw, lh - 1);
            }
        }
        if (pass == 0) {
            // warp-wide reservation; lanes of one warp may belong to different bands (a warp spans at most two tile rows
            // worth of base tiles only when ntx < 32): reserve per band among the lanes that share it
            const uint32_t peers = __match_any_sync(0xffffffffu, band);
            uint32_t inc_it = 0, inc_bp = 0, tot_it = 0, tot_bp = 0;
            unsigned long long tot_bf = 0;
            for (int l = 0; l < 32; ++l) {
                const uint32_t a = __shfl_sync(0xffffffffu, n_it, l), b = __shfl_sync(0xffffffffu, n_bp, l);
                const unsigned long long c = __shfl_sync(0xffffffffu, n_bf, l);
                if ((peers >> l) & 1u) {
                    if (l < lane) { inc_it += a; inc_bp += b; }
                    tot_it += a; tot_bp += b; tot_bf += c;
                }
            }
            const int leader = __ffs(peers) - 1;
            uint32_t base_it = 0, base_bp = 0;
            if (lane == leader) {
                if (tot_it) base_it = atomicAdd(&hdr->band_items[band], tot_it);
                if (tot_bp) { base_bp = atomicAdd(&hdr->n_big_pixels, tot_bp); atomicAdd(&hdr->n_big_fragments, tot_bf); }
            }
            at_it = __shfl_sync(0xffffffffu, base_it, leader) + inc_it;
            at_bp = __shfl_sync(0xffffffffu, base_bp, leader) + inc_bp;
        }
    }
}

}  // namespace inpc
