// sampler.cuh -- NEXT row f4, the rasterizer's upstream neighbour: viewpoint-specific sampling of the implicit point
// cloud (Sec. 3.2 Eq. 4; depth Eq. 9; frustum re-sampling; "sampling an
// implicit point cloud takes up more than half of the rendering time during inference").
//
//   per leaf i (centre c_i, level l_i, probability p_i, side = root_side / 2^l_i):
//     p^_i = 1_visible * p_i / (d_i * 2^(l_i * lambda_l)),  lambda_l = 0.5                                  (Eq. 4)
//     d_i  = max(|z_view - near| / (far - near), 1e-8)                                                      (Eq. 9)
//     visible <=> the leaf's cube can intersect the view frustum (reading R19): its centre or one of its eight corners
//                 lies inside the frustum, OR no frustum plane has all eight corners on its outer side (the conservative
//                 box-against-planes test: it never misses a cube the frustum enters through a face or an edge, nor
//                 the one that contains the camera; it may admit a few cubes next to a frustum edge, whose samples the
//                 re-draw then rejects)
//   multinomial sampling WITH replacement: N independent draws from the distribution p^ / sum p^, by inverse CDF;
//   every draw is offset uniformly inside its leaf's cube; a position outside the frustum is drawn again (up to
//   kSampleAttempts times; what still fails is returned as NaN / leaf -1 and culled by the rasterizer).
//
// So that the result is REPRODUCIBLE BIT FOR BIT by an independent implementation (the oracle), everything that
// decides an integer is integer or individually rounded IEEE arithmetic (R19):
//   * z_view, u, v: the rasterizer's canonical fp32 projection (common.cuh project ops);
//   * p^ in fp64 with one rounded operation per step; the CDF is INTEGER: w_i = floor(p^_i / max p^ * 2^32), prefix sums
//     in u64 (exact, whatever the order of the parallel scan), draw = floor(r * total / 2^64) by 64x64 -> 128-bit multiply;
//   * random numbers: the counter-based SplitMix64 (seed + (counter + 1) * golden gamma, Stafford mix 13), four per
//     attempt: counter = ((sample * kSampleAttempts + attempt) * 4 + k), k = 0 leaf draw, 1..3 jitter (top 24 bits).
#pragma once
#include "common.cuh"

namespace inpc {

constexpr int kSampleAttempts = 8;
constexpr int kMaxLeafLevel = 30;        // leaf_level outside [0, 30] is treated as "never sampled" (the paper's octree stops at 8: 256^3)
constexpr int kScan64Threads = 256, kScan64Items = 8, kScan64Tile = kScan64Threads * kScan64Items;

__host__ __device__ __forceinline__ unsigned long long splitmix64(unsigned long long seed, unsigned long long counter) {
    unsigned long long z = seed + (counter + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// canonical fp32 camera-space position and image coordinates (the same operation sequence as project_point)
__device__ __forceinline__ bool in_frustum(const Camera& c, float x, float y, float z, float* zc_out = nullptr) {
    const float xc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[0], x), __fmul_rn(c.R[1], y)), __fmul_rn(c.R[2], z)), c.t[0]);
    const float yc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[3], x), __fmul_rn(c.R[4], y)), __fmul_rn(c.R[5], z)), c.t[1]);
    const float zc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[6], x), __fmul_rn(c.R[7], y)), __fmul_rn(c.R[8], z)), c.t[2]);
    if (zc_out) *zc_out = zc;
    if (!(zc > c.near_z && zc < c.far_z)) return false;
    const float u = __fadd_rn(__fdiv_rn(__fmul_rn(c.fx, xc), zc), c.cx);
    const float v = __fadd_rn(__fdiv_rn(__fmul_rn(c.fy, yc), zc), c.cy);
    return u >= 0.f && u < (float)c.W && v >= 0.f && v < (float)c.H;
}

// Which of the six frustum planes the point lies OUTSIDE of (bit set), in camera space, every operation rounded on its
// own: near / far on z_c, the four side planes through the camera centre written without the division
// (u >= 0 <=> fx x_c + cx z_c >= 0 for z_c > 0, and the plane form stays meaningful for z_c <= 0, where u does not).
// Each test is the negation of "inside", so a NaN coordinate counts as outside of every plane.
__device__ __forceinline__ unsigned outside_planes(const Camera& c, float x, float y, float z) {
    const float xc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[0], x), __fmul_rn(c.R[1], y)), __fmul_rn(c.R[2], z)), c.t[0]);
    const float yc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[3], x), __fmul_rn(c.R[4], y)), __fmul_rn(c.R[5], z)), c.t[1]);
    const float zc = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.R[6], x), __fmul_rn(c.R[7], y)), __fmul_rn(c.R[8], z)), c.t[2]);
    const float fxx = __fmul_rn(c.fx, xc), fyy = __fmul_rn(c.fy, yc);
    const float left = __fadd_rn(fxx, __fmul_rn(c.cx, zc)), right = __fadd_rn(fxx, __fmul_rn(__fsub_rn(c.cx, (float)c.W), zc));
    const float top = __fadd_rn(fyy, __fmul_rn(c.cy, zc)), bottom = __fadd_rn(fyy, __fmul_rn(__fsub_rn(c.cy, (float)c.H), zc));
    return (!(zc > c.near_z) ? 1u : 0u) | (!(zc < c.far_z) ? 2u : 0u) | (!(left >= 0.f) ? 4u : 0u) | (!(right < 0.f) ? 8u : 0u) |
           (!(top >= 0.f) ? 16u : 0u) | (!(bottom < 0.f) ? 32u : 0u);
}

// Eq. 4 / Eq. 9 per leaf; the maximum of p^ (positive doubles order like their bit patterns) by one atomic per CTA.
__global__ void __launch_bounds__(256) k_leaf_weight(const float* __restrict__ centre, const int32_t* __restrict__ level,
                                                      const float* __restrict__ prob, uint32_t L, float root_side, Camera cam,
                                                      double* __restrict__ phat, unsigned long long* __restrict__ max_bits) {
    double mx = 0.0;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < L; i += gridDim.x * blockDim.x) {
        const float x = centre[3 * i], y = centre[3 * i + 1], z = centre[3 * i + 2];
        const int l = level[i];
        const bool level_ok = l >= 0 && l <= kMaxLeafLevel;        // outside of it 2^-l is not a normal fp32: such a leaf gets p^ = 0
        const float h = __fmul_rn(0.5f, __fmul_rn(root_side, __int_as_float((127 - (level_ok ? l : 0)) << 23)));   // half side, exact
        float zc;
        bool vis = in_frustum(cam, x, y, z, &zc);
        unsigned all_out = 63u;                                    // planes that have every corner so far on their outer side
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const float qx = __fadd_rn(x, (k & 1) ? h : -h), qy = __fadd_rn(y, (k & 2) ? h : -h), qz = __fadd_rn(z, (k & 4) ? h : -h);
            vis = vis || in_frustum(cam, qx, qy, qz);
            all_out &= outside_planes(cam, qx, qy, qz);
        }
        vis = vis || all_out == 0u;
        double p = 0.0;
        if (vis && level_ok) {
            const double d = fmax(__ddiv_rn(fabs(__dsub_rn((double)zc, (double)cam.near_z)),
                                            __dsub_rn((double)cam.far_z, (double)cam.near_z)), 1e-8);
            const double f = ldexp((l & 1) ? 1.4142135623730951 : 1.0, l >> 1);                  // 2^(l / 2)
            p = __ddiv_rn((double)prob[i], __dmul_rn(d, f));
            if (!(p > 0.0) || !(p < 1.7976931348623157e308)) p = 0.0;                            // NaN / inf / negative inputs
        }
        phat[i] = p;
        mx = fmax(mx, p);
    }
    __shared__ double s_mx[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0) s_mx[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) mx = fmax(mx, s_mx[w]);
        atomicMax(max_bits, (unsigned long long)__double_as_longlong(mx));
    }
}

// integer weights + tile-local inclusive scan; tile sums for the second level
__global__ void __launch_bounds__(kScan64Threads) k_cdf_local(const double* __restrict__ phat, uint32_t L,
                                                               const unsigned long long* __restrict__ max_bits,
                                                               unsigned long long* __restrict__ cdf,
                                                               unsigned long long* __restrict__ tile_sum) {
    __shared__ unsigned long long s_warp[kScan64Threads / 32];
    const double m = __longlong_as_double((long long)*max_bits);
    const uint32_t base = blockIdx.x * kScan64Tile + threadIdx.x * kScan64Items;
    unsigned long long v[kScan64Items], run = 0;
#pragma unroll
    for (int q = 0; q < kScan64Items; ++q) {
        unsigned long long w = 0;
        if (base + q < L && m > 0.0) w = (unsigned long long)floor(__dmul_rn(__ddiv_rn(phat[base + q], m), 4294967296.0));
        run += w; v[q] = run;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned long long inc = run;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    unsigned long long off = inc - run;
    for (int w = 0; w < warp; ++w) off += s_warp[w];
#pragma unroll
    for (int q = 0; q < kScan64Items; ++q) if (base + q < L) cdf[base + q] = v[q] + off;
    if (threadIdx.x == kScan64Threads - 1) tile_sum[blockIdx.x] = off + run;
}

// exclusive scan of the tile sums by ONE CTA (n_tiles <= 8192 => L <= 16.7 M leaves, 256^3 = the paper's cap)
__global__ void __launch_bounds__(1024) k_cdf_tiles(unsigned long long* __restrict__ tile_sum, uint32_t n_tiles,
                                                     unsigned long long* __restrict__ total) {
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (uint32_t b = 0; b < n_tiles; b += 1024) {
        const uint32_t i = b + threadIdx.x;
        const unsigned long long x = i < n_tiles ? tile_sum[i] : 0ull;
        unsigned long long inc = x;
        const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += t; }
        if (lane == 31) s_warp[warp] = inc;
        __syncthreads();
        unsigned long long off = s_carry;
        for (int w = 0; w < warp; ++w) off += s_warp[w];
        if (i < n_tiles) tile_sum[i] = off + inc - x;                  // exclusive
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = off + inc;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = s_carry;
}

__global__ void __launch_bounds__(kScan64Threads) k_cdf_add(unsigned long long* __restrict__ cdf, uint32_t L,
                                                             const unsigned long long* __restrict__ tile_sum) {
    const unsigned long long off = tile_sum[blockIdx.x];
    const uint32_t base = blockIdx.x * kScan64Tile;
    for (uint32_t q = threadIdx.x; q < kScan64Tile; q += kScan64Threads) if (base + q < L) cdf[base + q] += off;
}

// Guide table of the inverse CDF: the top kGuideBits bits b of the 64-bit random number confine the draw
// r = floor(rng * total / 2^64) to [lo_b, lo_{b+1}] with lo_b = floor((b << (64 - kGuideBits)) * total / 2^64) (mulhi is
// monotone in rng), so the drawn leaf -- the first i with cdf[i] > r -- lies in [guide[b], guide[b + 1]] where
// guide[b] = first i with cdf[i] > lo_b and guide[2^kGuideBits] = L - 1.  The search inside that range finds the SAME
// leaf as a search over the whole CDF (it is the unique first i with cdf[i] > r), in ~4 probes instead of 20 for 2^20 leaves.
constexpr int kGuideBits = 16;
constexpr uint32_t kGuide = 1u << kGuideBits;

__global__ void __launch_bounds__(256) k_cdf_guide(const unsigned long long* __restrict__ cdf, uint32_t L,
                                                    const unsigned long long* __restrict__ total_p,
                                                    uint32_t* __restrict__ guide) {
    const uint32_t b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b > kGuide) return;
    const unsigned long long total = *total_p;
    uint32_t lo = 0, hi = L - 1;
    if (b < kGuide && total > 0) {
        const unsigned long long r = __umul64hi((unsigned long long)b << (64 - kGuideBits), total);   // < total
        while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (__ldg(&cdf[mid]) > r) hi = mid; else lo = mid + 1; }
    } else {
        lo = L - 1;
    }
    guide[b] = lo;
}

// one thread per sample: draw a leaf (inverse CDF: guide table, then binary search), jitter inside it, re-draw while outside the frustum
__global__ void __launch_bounds__(256) k_sample(const unsigned long long* __restrict__ cdf, uint32_t L,
                                                 const unsigned long long* __restrict__ total_p,
                                                 const float* __restrict__ centre, const int32_t* __restrict__ level,
                                                 float root_side, Camera cam, unsigned long long seed, long long N,
                                                 float* __restrict__ pos, int32_t* __restrict__ leaf_out,
                                                 unsigned long long* __restrict__ n_valid, int attempts,
                                                 const uint32_t* __restrict__ guide) {
    const unsigned long long total = *total_p;
    unsigned int ok = 0;
    for (long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x; j < N; j += (long long)gridDim.x * blockDim.x) {
        float px = __int_as_float(0x7fc00000), py = px, pz = px;
        int32_t leaf = -1;
        for (int a = 0; a < attempts && total > 0; ++a) {      // attempts = kSampleAttempts, or 1 (INPC_SAMPLE_NO_RESAMPLE); same counters
            const unsigned long long c0 = ((unsigned long long)j * kSampleAttempts + a) * 4ull;
            const unsigned long long rng0 = splitmix64(seed, c0);
            const unsigned long long r = __umul64hi(rng0, total);                         // floor(rng * total / 2^64)
            const uint32_t gb = (uint32_t)(rng0 >> (64 - kGuideBits));
            uint32_t lo = __ldg(&guide[gb]), hi = __ldg(&guide[gb + 1]);                  // first i with cdf[i] > r lies in [lo, hi]
            while (lo < hi) { const uint32_t mid = (lo + hi) >> 1; if (__ldg(&cdf[mid]) > r) hi = mid; else lo = mid + 1; }
            const int l = level[lo];
            const float side = __fmul_rn(root_side, __int_as_float((127 - l) << 23));
            float q[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const float u = __fmul_rn((float)(uint32_t)(splitmix64(seed, c0 + 1 + k) >> 40), 5.9604644775390625e-08f);   // 2^-24
                q[k] = __fadd_rn(centre[3 * lo + k], __fmul_rn(__fsub_rn(u, 0.5f), side));
            }
            if (in_frustum(cam, q[0], q[1], q[2])) { px = q[0]; py = q[1]; pz = q[2]; leaf = (int32_t)lo; break; }
        }
        pos[3 * j] = px; pos[3 * j + 1] = py; pos[3 * j + 2] = pz;
        leaf_out[j] = leaf;
        ok += leaf >= 0 ? 1u : 0u;
    }
    __shared__ unsigned int s_ok[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ok += __shfl_xor_sync(0xffffffffu, ok, o);
    if ((threadIdx.x & 31) == 0) s_ok[threadIdx.x >> 5] = ok;
    __syncthreads();
    if (threadIdx.x == 0) {                                   // one atomic per (persistent) CTA
        unsigned long long t = 0;
        for (int w = 0; w < 8; ++w) t += s_ok[w];
        if (t) atomicAdd(n_valid, t);
    }
}

}  // namespace inpc
