// cellsort.cuh -- step a3 of the hot path: the segmented (depth bits, point index) key sort.
//
// The segments are the CELLS of the (W+1) x (H+1) grid, not the pixels: every pixel's depth-ordered
// run is the merge of its four sorted cell lists (tile.cuh), so N points are sorted once instead of
// 4N fragments twice (forward and backward).  Two kernels:
//   k_cellsort      cells of up to kCellSmall points.  A CTA walks windows of whole cells
//                   (<= kCsWindow records), keeps each thread's records in registers and their 64-bit keys
//                   (depth_bits << 32 | point_idx, unique) in shared memory; a record's sorted position is
//                   the number of smaller keys in its own cell (rank by counting: cells are small, the
//                   loop is a broadcast shared-memory read).  The record is then written straight to its
//                   sorted slot together with its features, gathered from feat[idx] (the only gather of
//                   the whole path): dk[slot] = depth bits, R[slot] = { tx, ty, opacity, idx | feat }.
//   k_cellsort_big  one CTA per larger cell (depth-complexity stress): all-ascending bitonic network on
//                   (depth_bits << 32 | source slot) keys, ties resolved by point index; chunks of kBigChunk
//                   keys in shared memory, the long-distance stages on the L2-resident key slice.
#pragma once
#include "common.cuh"

namespace inpc {

constexpr int kCsThreads = 256;
constexpr int kCsPer     = 4;                            // records per thread per window
constexpr int kCsWindow  = kCsThreads * kCsPer;          // >= kCellSmall
constexpr int kCsCells   = 1024;                         // cells per CTA work unit

template <int D>
__device__ __forceinline__ void emit_sorted(const float4 a0, const float4 a1, uint32_t dst,
                                            const float* __restrict__ feat, uint32_t* __restrict__ dk,
                                            float4* __restrict__ Ra, float4* __restrict__ Rf) {
    constexpr int FV = D / 4;
    const uint32_t idx = __float_as_uint(a0.y);
    float4 f[D / 4];
#pragma unroll
    for (int q = 0; q < D / 4; ++q) f[q] = __ldg(reinterpret_cast<const float4*>(feat + (size_t)idx * D) + q);
    dk[dst] = __float_as_uint(a0.x);
    Ra[dst] = make_float4(a0.z, a0.w, a1.x, a0.y);       // tx, ty, opacity, idx
#pragma unroll
    for (int q = 0; q < FV; ++q) Rf[(size_t)dst * FV + q] = f[q];
}

template <int D>
__global__ void __launch_bounds__(kCsThreads) k_cellsort(const float4* __restrict__ A,
                                                          const uint32_t* __restrict__ celloff, uint32_t C,
                                                          uint32_t unit_begin, uint32_t unit_end,
                                                          const float* __restrict__ feat,
                                                          uint32_t* __restrict__ dk, float4* __restrict__ Ra, float4* __restrict__ Rf) {
    __shared__ uint32_t s_off[kCsCells + 1];
    __shared__ unsigned long long s_key[kCsWindow];
    const int tid = threadIdx.x;
    for (uint32_t unit = unit_begin + blockIdx.x; unit < unit_end; unit += gridDim.x) {   // this launch's band of units
        const uint32_t c0 = unit * kCsCells, nc = min((uint32_t)kCsCells, C - c0);
        __syncthreads();
        for (uint32_t c = tid; c <= nc; c += kCsThreads) s_off[c] = __ldg(&celloff[c0 + c]);
        __syncthreads();
        uint32_t wa = 0;                                 // first cell of the window (relative to c0)
        while (wa < nc) {
            // window = longest run of whole cells [wa, wb) with at most kCsWindow records (uniform search)
            const uint32_t s0 = s_off[wa];
            uint32_t lo = wa + 1, hi = nc;               // answer in [wa+1, nc]
            while (lo < hi) {
                const uint32_t mid = (lo + hi + 1) >> 1;
                if (s_off[mid] - s0 <= (uint32_t)kCsWindow) lo = mid; else hi = mid - 1;
            }
            const uint32_t wb = lo;
            const uint32_t nrec = s_off[wb] - s0;
            if (nrec > 0 && nrec <= (uint32_t)kCsWindow) {
                float4 a0[kCsPer], a1[kCsPer];
#pragma unroll
                for (int q = 0; q < kCsPer; ++q) {
                    const uint32_t l = q * kCsThreads + tid;
                    if (l < nrec) {
                        a0[q] = __ldcs(&A[2 * (size_t)(s0 + l)]);
                        a1[q] = __ldcs(&A[2 * (size_t)(s0 + l) + 1]);
                        s_key[l] = ((unsigned long long)__float_as_uint(a0[q].x) << 32) | __float_as_uint(a0[q].y);
                    }
                }
                __syncthreads();
#pragma unroll
                for (int q = 0; q < kCsPer; ++q) {
                    const uint32_t l = q * kCsThreads + tid;
                    if (l < nrec) {
                        const uint32_t cell = __float_as_uint(a1[q].y) - c0;
                        const uint32_t cs = s_off[cell] - s0, ce = s_off[cell + 1] - s0;
                        if (ce - cs <= (uint32_t)kCellSmall) {
                            const unsigned long long me = s_key[l];
                            uint32_t r = 0;
                            for (uint32_t j = cs; j < ce; ++j) r += s_key[j] < me ? 1u : 0u;
                            emit_sorted<D>(a0[q], a1[q], s0 + cs + r, feat, dk, Ra, Rf);
                        }
                    }
                }
                __syncthreads();
            }
            // nrec > kCsWindow only when [wa, wa+1) is a single oversized cell: k_cellsort_big's
            wa = wb;
        }
    }
}

// ---- large cells ------------------------------------------------------------------------------------
// key = depth_bits << 32 | source slot; equal depth bits (rare) are ordered by point index, read from A.
__device__ __forceinline__ bool bigcell_less(unsigned long long a, unsigned long long b, const float4* __restrict__ A) {
    const uint32_t da = (uint32_t)(a >> 32), db = (uint32_t)(b >> 32);
    if (da != db) return da < db;
    const uint32_t ia = __float_as_uint(__ldg(&A[2 * (size_t)(uint32_t)a]).y);
    const uint32_t ib = __float_as_uint(__ldg(&A[2 * (size_t)(uint32_t)b]).y);
    return ia < ib;
}

// One compare-exchange of the all-ascending network on shared-memory keys (equal depth bits: rare).
__device__ __forceinline__ void cex(unsigned long long* s, uint32_t i, uint32_t l, const float4* A) {
    const unsigned long long a = s[i], b = s[l];
    const uint32_t da = (uint32_t)(a >> 32), db = (uint32_t)(b >> 32);
    bool sw = db < da;
    if (da == db) sw = bigcell_less(b, a, A);
    if (sw) { s[i] = b; s[l] = a; }
}

// merge stages j = j0, j0/2, ..., 1 of the all-ascending network on s[0..m) (m <= kBigChunk); j0 a power of two.
// All index arithmetic is shifts: span, j are powers of two (lj = log2 j).
__device__ __forceinline__ void smem_merge_stages(unsigned long long* s, uint32_t m, uint32_t j0, const float4* A) {
    uint32_t span = 2; while (span < m) span <<= 1;
    for (uint32_t j = j0, lj = 31u - __clz(j0); j > 0; j >>= 1, --lj) {
        for (uint32_t c = threadIdx.x; c < (span >> 1); c += blockDim.x) {
            const uint32_t i = ((c >> lj) << (lj + 1)) + (c & (j - 1)), l = i + j;
            if (l < m) cex(s, i, l, A);
        }
        __syncthreads();
    }
}

__device__ __forceinline__ void smem_sort_full(unsigned long long* s, uint32_t m, const float4* A) {
    uint32_t span = 2; while (span < m) span <<= 1;
    for (uint32_t k = 2, lhk = 0; k <= span; k <<= 1, ++lhk) {          // hk = k / 2 = 1 << lhk
        const uint32_t hk = k >> 1;
        for (uint32_t c = threadIdx.x; c < (span >> 1); c += blockDim.x) {
            const uint32_t i = ((c >> lhk) << (lhk + 1)) + (c & (hk - 1)), l = i ^ (k - 1);
            if (l < m) cex(s, i, l, A);
        }
        __syncthreads();
        if (k >= 4) smem_merge_stages(s, m, k >> 2, A);
    }
}

// THREADS / CHUNK: CTA size and keys sorted in shared memory at a time.  Two instances run back to back: cells of
// up to 1024 points on 128-thread CTAs with 8 KB of shared memory (16 CTAs per SM: what bounds this kernel is the
// number of cells in flight, every bitonic stage being a CTA barrier), larger cells on 512-thread CTAs with 64 KB.
// A CTA takes every cell of the list in turn and skips those outside [n_lo, n_hi].
template <int D, int THREADS, int CHUNK>
__global__ void __launch_bounds__(THREADS) k_cellsort_big(const Header* __restrict__ hdr, uint32_t n_lo, uint32_t n_hi,
                                                               uint32_t* __restrict__ cursor,
                                                               const BigCell* __restrict__ bigcells,
                                                               const float4* __restrict__ A,
                                                               unsigned long long* __restrict__ keys_all,
                                                               const float* __restrict__ feat,
                                                               uint32_t* __restrict__ dk, float4* __restrict__ Ra, float4* __restrict__ Rf) {
    extern __shared__ __align__(16) unsigned char smem_big[];
    unsigned long long* s_keys = reinterpret_cast<unsigned long long*>(smem_big);
    __shared__ uint32_t s_b;
    const int tid = threadIdx.x;
    const uint32_t n_big = hdr->n_big_cells;
    while (true) {
        __syncthreads();
        if (tid == 0) s_b = atomicAdd(cursor, 1u);
        __syncthreads();
        const uint32_t b = s_b;
        if (b >= n_big) break;
        const BigCell e = bigcells[b];
        const uint32_t n = e.n, start = e.start;
        if (n < n_lo || n > n_hi) continue;               // the other instance's (uniform across the CTA)
        unsigned long long* keys = keys_all + start;     // scratch slice, indexed like the slots
        auto make_key = [&](uint32_t l) -> unsigned long long {
            const uint32_t depth = __float_as_uint(__ldg(&A[2 * (size_t)(start + l)]).x);
            return ((unsigned long long)depth << 32) | (unsigned long long)(start + l);
        };
        if (n <= (uint32_t)CHUNK) {
            for (uint32_t l = tid; l < n; l += THREADS) s_keys[l] = make_key(l);
            __syncthreads();
            smem_sort_full(s_keys, n, A);
            for (uint32_t l = tid; l < n; l += THREADS) __stcg(&keys[l], s_keys[l]);
        } else {
            for (uint32_t cb = 0; cb < n; cb += CHUNK) {
                const uint32_t m = min((uint32_t)CHUNK, n - cb);
                __syncthreads();
                for (uint32_t l = tid; l < m; l += THREADS) s_keys[l] = make_key(cb + l);
                __syncthreads();
                smem_sort_full(s_keys, m, A);
                for (uint32_t l = tid; l < m; l += THREADS) __stcg(&keys[cb + l], s_keys[l]);
            }
            __syncthreads();
            uint32_t np2 = CHUNK; while (np2 < n) np2 <<= 1;
            for (uint32_t k = 2u * CHUNK; k <= np2; k <<= 1) {
                const uint32_t hk = k >> 1;
                for (uint32_t c = tid; c < (np2 >> 1); c += THREADS) {          // flip stage, global
                    const uint32_t i = ((c / hk) * k) + (c & (hk - 1)), l = i ^ (k - 1);
                    if (l < n) {
                        const unsigned long long a = __ldcg(&keys[i]), bb = __ldcg(&keys[l]);
                        if (bigcell_less(bb, a, A)) { __stcg(&keys[i], bb); __stcg(&keys[l], a); }
                    }
                }
                __syncthreads();
                uint32_t j = k >> 2;
                for (; j >= (uint32_t)CHUNK; j >>= 1) {                          // long-distance stages, global
                    for (uint32_t c = tid; c < (np2 >> 1); c += THREADS) {
                        const uint32_t i = ((c / j) * (j << 1)) + (c & (j - 1)), l = i + j;
                        if (l < n) {
                            const unsigned long long a = __ldcg(&keys[i]), bb = __ldcg(&keys[l]);
                            if (bigcell_less(bb, a, A)) { __stcg(&keys[i], bb); __stcg(&keys[l], a); }
                        }
                    }
                    __syncthreads();
                }
                for (uint32_t cb = 0; cb < n; cb += CHUNK) {                     // j < chunk: in shared memory
                    const uint32_t m = min((uint32_t)CHUNK, n - cb);
                    for (uint32_t l = tid; l < m; l += THREADS) s_keys[l] = __ldcg(&keys[cb + l]);
                    __syncthreads();
                    smem_merge_stages(s_keys, m, CHUNK >> 1, A);
                    for (uint32_t l = tid; l < m; l += THREADS) __stcg(&keys[cb + l], s_keys[l]);
                    __syncthreads();
                }
            }
        }
        __syncthreads();
        // permute: sorted position l takes the record of source slot low32(keys[l])
        for (uint32_t l = tid; l < n; l += THREADS) {
            const uint32_t src = (uint32_t)__ldcg(&keys[l]);
            const float4 a0 = __ldg(&A[2 * (size_t)src]), a1 = __ldg(&A[2 * (size_t)src + 1]);
            emit_sorted<D>(a0, a1, start + l, feat, dk, Ra, Rf);
        }
    }
}

}  // namespace inpc
