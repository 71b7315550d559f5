// big.cuh -- the long-run path: pixels deeper than kPixMax fragments (depth-complexity stress,
// BASELINE.json config 5: up to tens of thousands of fragments in one pixel).
//
// One CTA per such pixel (persistent over the list k_classify_pixels built):
//   a3  the run's keys (depth bits << 32 | record << 2 | corner) are gathered into the pixel's slice of
//       `bigkeys` and sorted by (depth bits, point index) with an all-ascending bitonic network:
//       runs <= kBigChunk entirely in shared memory; longer runs chunk-wise in shared memory with the
//       few long-distance stages done on the (L2-resident) global slice.  Virtual +inf padding: a
//       comparator whose upper index is >= n is skipped, so no power-of-two padding is stored.
//   a4  warp 0 composites front to back straight from the sorted slice (same 32-wide prefix-product
//       step as the tile kernel), stops at the cut-off, and keeps the transmittance entering every
//       chunk in `bigtin` for the backward pass.
//   a5  backward: chunks walked back to front; per-fragment gradients are added with red.global.add
//       (these pixels are few; their points' other fragments are written by the tile kernel first).
#pragma once
#include "common.cuh"
#include "tile.cuh"

namespace inpc {

struct BigArgs {
    const Header* hdr;
    uint32_t* big_cursor;
    BigEntry* big;
    const uint32_t* celloff;
    const float4* rec;
    const float* rop;
    unsigned long long* bigkeys;
    double* bigtin;
    int W, H;
    float* out_feat;
    float* out_alpha;
    const uint32_t* pixoff;
    uint32_t* sorted_idx;
    uint32_t* sorted_depth;
    const float* g_feat;
    const float* g_alpha;
    float* d_feat;
    float* d_opacity;
    float* d_uv;
};

__device__ __forceinline__ bool big_less(unsigned long long a, unsigned long long b, const float4* __restrict__ rec, int RV) {
    const uint32_t da = (uint32_t)(a >> 32), db = (uint32_t)(b >> 32);
    if (da != db) return da < db;
    const uint32_t ia = __float_as_uint(__ldg(&rec[(size_t)(((uint32_t)a) >> 2) * RV]).y);
    const uint32_t ib = __float_as_uint(__ldg(&rec[(size_t)(((uint32_t)b) >> 2) * RV]).y);
    return ia < ib;
}

// Long runs carry the transmittance and the backward recurrence in fp64: an fp32 product of tens of
// thousands of (1 - a) factors drifts past the 1e-5 gradient floor.
__device__ __forceinline__ double warp_incl_prod_d(double v, int lane) {
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= d) v *= t;
    }
    return v;
}

// merge stages j = j0, j0/2, ..., 1 of the all-ascending network on s[0..m) (m <= kBigChunk)
__device__ __forceinline__ void smem_merge_stages(unsigned long long* s, uint32_t m, uint32_t j0, const float4* rec, int RV) {
    uint32_t span = 2; while (span < m) span <<= 1;
    for (uint32_t j = j0; j > 0; j >>= 1) {
        for (uint32_t c = threadIdx.x; c < (span >> 1); c += blockDim.x) {
            const uint32_t i = ((c / j) * (j << 1)) + (c & (j - 1)), l = i + j;
            if (l < m) {
                const unsigned long long a = s[i], b = s[l];
                if (big_less(b, a, rec, RV)) { s[i] = b; s[l] = a; }
            }
        }
        __syncthreads();
    }
}

__device__ __forceinline__ void smem_sort_full(unsigned long long* s, uint32_t m, const float4* rec, int RV) {
    uint32_t span = 2; while (span < m) span <<= 1;
    for (uint32_t k = 2; k <= span; k <<= 1) {
        const uint32_t hk = k >> 1;
        for (uint32_t c = threadIdx.x; c < (span >> 1); c += blockDim.x) {
            const uint32_t i = ((c / hk) * k) + (c & (hk - 1)), l = i ^ (k - 1);
            if (l < m) {
                const unsigned long long a = s[i], b = s[l];
                if (big_less(b, a, rec, RV)) { s[i] = b; s[l] = a; }
            }
        }
        __syncthreads();
        if (k >= 4) smem_merge_stages(s, m, k >> 2, rec, RV);
    }
}

template <int D, int MODE>
__global__ void __launch_bounds__(kBigThreads) k_big(BigArgs A) {
    constexpr int RV = 1 + D / 4;
    extern __shared__ __align__(16) unsigned char smem_big[];
    unsigned long long* s_keys = reinterpret_cast<unsigned long long*>(smem_big);
    __shared__ uint32_t s_b;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int W = A.W;
    const uint32_t n_big = (uint32_t)(A.hdr->big_packed >> 40);

    while (true) {
        __syncthreads();
        if (tid == 0) s_b = atomicAdd(A.big_cursor, 1u);
        __syncthreads();
        const uint32_t b = s_b;
        if (b >= n_big) break;
        const BigEntry e = A.big[b];
        const uint32_t n = e.n;
        const int y = e.pix / W, x = e.pix - y * W;
        unsigned long long* keys = A.bigkeys + e.start;
        double* tin = A.bigtin + e.tin_base;

        if (MODE != kBwd) {
            const uint32_t c0 = (uint32_t)y * (W + 1) + x, c1 = c0 + (W + 1);
            const uint32_t o00 = __ldg(&A.celloff[c0]), o01 = __ldg(&A.celloff[c0 + 1]), o02 = __ldg(&A.celloff[c0 + 2]);
            const uint32_t o10 = __ldg(&A.celloff[c1]), o11 = __ldg(&A.celloff[c1 + 1]);
            const uint32_t n0 = o02 - o00;
            auto make_key = [&](uint32_t l) -> unsigned long long {
                uint32_t g, dy, dx;
                if (l < n0) { g = o00 + l; dy = 1u; dx = g < o01 ? 1u : 0u; }
                else        { g = o10 + (l - n0); dy = 0u; dx = g < o11 ? 1u : 0u; }
                const uint32_t depth = __float_as_uint(__ldg(&A.rec[(size_t)g * RV]).x);
                return ((unsigned long long)depth << 32) | (unsigned long long)((g << 2) | (dy << 1) | dx);
            };
            // ---------------------------------------------------------------- a3: sort
            if (n <= (uint32_t)kBigChunk) {
                for (uint32_t l = tid; l < n; l += kBigThreads) s_keys[l] = make_key(l);
                __syncthreads();
                smem_sort_full(s_keys, n, A.rec, RV);
                for (uint32_t l = tid; l < n; l += kBigThreads) __stcg(&keys[l], s_keys[l]);
            } else {
                for (uint32_t cb = 0; cb < n; cb += kBigChunk) {
                    const uint32_t m = min((uint32_t)kBigChunk, n - cb);
                    __syncthreads();
                    for (uint32_t l = tid; l < m; l += kBigThreads) s_keys[l] = make_key(cb + l);
                    __syncthreads();
                    smem_sort_full(s_keys, m, A.rec, RV);
                    for (uint32_t l = tid; l < m; l += kBigThreads) __stcg(&keys[cb + l], s_keys[l]);
                }
                __syncthreads();
                uint32_t np2 = kBigChunk; while (np2 < n) np2 <<= 1;
                for (uint32_t k = 2u * kBigChunk; k <= np2; k <<= 1) {
                    const uint32_t hk = k >> 1;
                    for (uint32_t c = tid; c < (np2 >> 1); c += kBigThreads) {          // flip stage, global
                        const uint32_t i = ((c / hk) * k) + (c & (hk - 1)), l = i ^ (k - 1);
                        if (l < n) {
                            const unsigned long long a = __ldcg(&keys[i]), bb = __ldcg(&keys[l]);
                            if (big_less(bb, a, A.rec, RV)) { __stcg(&keys[i], bb); __stcg(&keys[l], a); }
                        }
                    }
                    __syncthreads();
                    uint32_t j = k >> 2;
                    for (; j >= (uint32_t)kBigChunk; j >>= 1) {                          // long-distance stages, global
                        for (uint32_t c = tid; c < (np2 >> 1); c += kBigThreads) {
                            const uint32_t i = ((c / j) * (j << 1)) + (c & (j - 1)), l = i + j;
                            if (l < n) {
                                const unsigned long long a = __ldcg(&keys[i]), bb = __ldcg(&keys[l]);
                                if (big_less(bb, a, A.rec, RV)) { __stcg(&keys[i], bb); __stcg(&keys[l], a); }
                            }
                        }
                        __syncthreads();
                    }
                    for (uint32_t cb = 0; cb < n; cb += kBigChunk) {                     // j < chunk: in shared memory
                        const uint32_t m = min((uint32_t)kBigChunk, n - cb);
                        for (uint32_t l = tid; l < m; l += kBigThreads) s_keys[l] = __ldcg(&keys[cb + l]);
                        __syncthreads();
                        smem_merge_stages(s_keys, m, kBigChunk >> 1, A.rec, RV);
                        for (uint32_t l = tid; l < m; l += kBigThreads) __stcg(&keys[cb + l], s_keys[l]);
                        __syncthreads();
                    }
                }
            }
            __syncthreads();
            if (MODE == kFwdDump) {
                const uint32_t ob = A.pixoff[e.pix];
                for (uint32_t l = tid; l < n; l += kBigThreads) {
                    const unsigned long long key = __ldcg(&keys[l]);
                    const float4 k4 = __ldg(&A.rec[(size_t)(((uint32_t)key) >> 2) * RV]);
                    A.sorted_idx[ob + l] = __float_as_uint(k4.y);
                    A.sorted_depth[ob + l] = __float_as_uint(k4.x);
                }
            }
        }

        // per-lane fragment fetch from the sorted global slice
        auto fetch = [&](uint32_t cb, uint32_t& g, uint32_t& corner, float& a, float& op, float4& k4) -> bool {
            const uint32_t kk = cb + lane;
            const bool valid = kk < n;
            g = 0; corner = 0; a = 0.f; op = 0.f; k4 = make_float4(0.f, 0.f, 0.f, 0.f);
            if (valid) {
                const unsigned long long key = __ldcg(&keys[kk]);
                g = ((uint32_t)key) >> 2; corner = ((uint32_t)key) & 3u;
                k4 = __ldg(&A.rec[(size_t)g * RV]);
                op = __ldg(&A.rop[g]);
                const float wx = (corner & 1u) ? k4.z : 1.f - k4.z;
                const float wy = (corner & 2u) ? k4.w : 1.f - k4.w;
                a = op * (wx * wy);
            }
            return valid;
        };

        if (warp == 0 && MODE != kBwd) {
            // -------------------------------------------------------------------- a4: blend
            float acc[D]; float accA = 0.f;
#pragma unroll
            for (int d = 0; d < D; ++d) acc[d] = 0.f;
            double T_in = 1.0;
            uint32_t nchunk_blended = 0;
            for (uint32_t cb = 0; cb < n; cb += 32) {
                if (T_in < (double)kTMin) break;
                if (lane == 0) tin[cb >> 5] = T_in;
                nchunk_blended = (cb >> 5) + 1;
                uint32_t g, corner; float a, op; float4 k4;
                const bool valid = fetch(cb, g, corner, a, op, k4);
                const double incl = warp_incl_prod_d(1.0 - (double)a, lane);
                double excl = __shfl_up_sync(0xffffffffu, incl, 1);
                if (lane == 0) excl = 1.0;
                const double T = T_in * excl;
                if (valid && T >= (double)kTMin) {
                    const float c = (float)(T * (double)a);
                    accA += c;
#pragma unroll
                    for (int v = 0; v < D / 4; ++v) {
                        const float4 f = __ldg(&A.rec[(size_t)g * RV + 1 + v]);
                        acc[4 * v] += c * f.x; acc[4 * v + 1] += c * f.y; acc[4 * v + 2] += c * f.z; acc[4 * v + 3] += c * f.w;
                    }
                }
                T_in *= __shfl_sync(0xffffffffu, incl, 31);
            }
#pragma unroll
            for (int s = 16; s > 0; s >>= 1) {
                accA += __shfl_xor_sync(0xffffffffu, accA, s);
#pragma unroll
                for (int d = 0; d < D; ++d) acc[d] += __shfl_xor_sync(0xffffffffu, acc[d], s);
            }
            if (lane == 0) {
                const size_t pix = e.pix;
#pragma unroll
                for (int v = 0; v < D / 4; ++v)
                    reinterpret_cast<float4*>(A.out_feat + pix * D)[v] = make_float4(acc[4 * v], acc[4 * v + 1], acc[4 * v + 2], acc[4 * v + 3]);
                A.out_alpha[pix] = accA;
                A.big[b].nb = nchunk_blended;      // chunks that hold blended fragments
            }
        }

        if (warp == 0 && MODE == kBwd) {
            // -------------------------------------------------------------------- a5: backward
            const size_t pix = e.pix;
            float gf[D];
#pragma unroll
            for (int v = 0; v < D / 4; ++v) {
                const float4 t = __ldg(reinterpret_cast<const float4*>(A.g_feat + pix * D) + v);
                gf[4 * v] = t.x; gf[4 * v + 1] = t.y; gf[4 * v + 2] = t.z; gf[4 * v + 3] = t.w;
            }
            const float gA = A.g_alpha ? __ldg(A.g_alpha + pix) : 0.f;
            double B_in = 0.0;
            for (int c = (int)e.nb - 1; c >= 0; --c) {
                const double Tc = __ldcg(&tin[c]);
                uint32_t g, corner; float a, op; float4 k4;
                const bool valid = fetch((uint32_t)c << 5, g, corner, a, op, k4);
                const double incl = warp_incl_prod_d(1.0 - (double)a, lane);
                double excl = __shfl_up_sync(0xffffffffu, incl, 1);
                if (lane == 0) excl = 1.0;
                const double T = Tc * excl;
                const bool bl = valid && T >= (double)kTMin;
                float G = gA;
                if (bl) {
#pragma unroll
                    for (int v = 0; v < D / 4; ++v) {
                        const float4 f = __ldg(&A.rec[(size_t)g * RV + 1 + v]);
                        G += f.x * gf[4 * v] + f.y * gf[4 * v + 1] + f.z * gf[4 * v + 2] + f.w * gf[4 * v + 3];
                    }
                }
                double M = bl ? 1.0 - (double)a : 1.0, C = bl ? (double)a * (double)G : 0.0;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const double M2 = __shfl_down_sync(0xffffffffu, M, d);
                    const double C2 = __shfl_down_sync(0xffffffffu, C, d);
                    if (lane + d < 32) { C = C + M * C2; M = M * M2; }
                }
                const double Mn = __shfl_down_sync(0xffffffffu, M, 1), Cn = __shfl_down_sync(0xffffffffu, C, 1);
                const double B = lane < 31 ? Cn + Mn * B_in : B_in;
                if (bl) {
                    const float Ta = (float)(T * (double)a), dLda = (float)(T * ((double)G - B));
                    const uint32_t idx = __float_as_uint(k4.y);
                    const int dx = corner & 1, dy = corner >> 1;
                    const float wx = dx ? k4.z : 1.f - k4.z, wy = dy ? k4.w : 1.f - k4.w;
                    float* pf = A.d_feat + (size_t)idx * D;
#pragma unroll
                    for (int v = 0; v < D / 4; ++v)
                        red_add_v4(pf + 4 * v, Ta * gf[4 * v], Ta * gf[4 * v + 1], Ta * gf[4 * v + 2], Ta * gf[4 * v + 3]);
                    red_add(A.d_opacity + idx, wx * wy * dLda);
                    red_add_v2(A.d_uv + 2 * (size_t)idx, op * (dx ? wy : -wy) * dLda, op * (dy ? wx : -wx) * dLda);
                }
                B_in = __shfl_sync(0xffffffffu, C, 0) + __shfl_sync(0xffffffffu, M, 0) * B_in;
            }
        }
    }
}

}  // namespace inpc
