// sh.cuh -- NEXT row f2: spherical-harmonics evaluation fused into the rasterizer ("The remaining M
// features are used as coefficients for SH evaluations to produce a view-dependent feature for each point ... SH of
// degree 2 and 4D view-dependent output features, resulting in M = 36 SH coefficients per point"; PAPER.md:370:
// "the spherical harmonics computations are fused into this pipeline"; ablation "SH PyTorch" 4.5 vs 5.8 fps, :413).
//
//   feature[d] = sum_{b=0..8} Y_b(dir) * coeff[4 b + d],   dir = (p_world - camera centre) / |.|,   d = 0..3
// Y_0..Y_8 = the real SH basis of degree 0..2 (Condon-Shortley phase, the convention of the common graphics code
// bases; reading R18).  Coefficients are stored basis-major (nine float4 per point) so that a feature is
// nine vector multiply-adds.
//
// Where it is fused (B200 reading of "fused"): into the EMISSION pass k_scatter<SH>, which already streams every
// point's position -- the 144 bytes of coefficients are read once, coalesced, and only the 16-byte feature goes on
// into the pipeline (the cell sort gathers features by point index: gathering 144-byte rows there would cost 4.5
// random sectors per point instead of one).  Backward: k_split<SH> writes dL/dcoeff[4 b + d] = Y_b * dL/dfeature[d].
#pragma once
#include "common.cuh"

namespace inpc {

constexpr int kShBasis = 9;
constexpr int kShCoeffs = 4 * kShBasis;       // M = 36

struct ViewPoint { float cx, cy, cz; };       // camera centre in world space, -R^T t

__device__ __forceinline__ void sh_basis9(float x, float y, float z, float (&Y)[kShBasis]) {
    const float n2 = x * x + y * y + z * z;
    const float inv = n2 > 0.f ? rsqrtf(n2) : 0.f;          // a point ON the camera centre sees the constant term only
    x *= inv; y *= inv; z *= inv;
    Y[0] = 0.28209479177387814f;
    Y[1] = -0.4886025119029199f * y;
    Y[2] = 0.4886025119029199f * z;
    Y[3] = -0.4886025119029199f * x;
    Y[4] = 1.0925484305920792f * x * y;
    Y[5] = -1.0925484305920792f * y * z;
    Y[6] = 0.31539156525252005f * (2.f * z * z - x * x - y * y);
    Y[7] = -1.0925484305920792f * x * z;
    Y[8] = 0.5462742152960396f * (x * x - y * y);
}

// feature of one point from its 36 coefficients (nine float4, basis-major)
__device__ __forceinline__ float4 sh_feature(const float4* __restrict__ c, float x, float y, float z) {
    float Y[kShBasis];
    sh_basis9(x, y, z, Y);
    float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int b = 0; b < kShBasis; ++b) {
        const float4 q = __ldcs(&c[b]);
        f.x += Y[b] * q.x; f.y += Y[b] * q.y; f.z += Y[b] * q.z; f.w += Y[b] * q.w;
    }
    return f;
}

}  // namespace inpc
