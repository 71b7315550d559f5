// tile.cuh -- per-pixel merge routines of the LONG-RUN path (big.cuh), steps a4/a5 of the hot path.
//
// The tile kernels k_blend (blend.cuh) and k_back (back.cuh) carry their own software-pipelined, shared-memory
// versions of these loops; what is left here is the plain form, read straight from global memory, that
// k_big uses for the pixels whose neighbourhood does not fit a shared-memory tile:
//   blend_pixel     a4: the pixel's four cell lists are sorted by (depth bits, point index), so its blend order
//                   is their merge: keep the four head keys in registers, take the minimum (equal depth bits:
//                   the smaller point index), composite that fragment (Eq. 1), advance that list.
//                   The loop ends at the cut-off T < 1e-4 -- nothing behind it is even read (unless DUMP asks
//                   for the whole order).  With INPC_SAVE_FOR_BACKWARD the transmittance in front of every
//                   blended fragment goes to gT[(slot, corner)] and the four list positions at the stop to
//                   pcur[pixel].
//   backward_pixel  a5: start from pcur and merge the four lists BACKWARDS (maximum first),
//                   reading T from gT; division-free recurrence
//                   dL/da_k = T_k (G_k - B_k),  B_{k-1} = a_k G_k + (1 - a_k) B_k.
//                   dL/da goes to gD[(slot, corner)]; grad.cuh combines the four corners of every record.
#pragma once
#include "common.cuh"

namespace inpc {

enum TileMode { kFwd = 0, kFwdDump = 1, kBwd = 2 };

// The four lists of one pixel as cursors into dk / R (shared-memory indices in the tile kernel, global
// slots in the long-run path).  Lists 0, 1 lie in cell row y, lists 2, 3 in cell row y+1.
struct PixLists { uint32_t c0, e0, c1, e1, c2, e2, c3, e3; };

// Forward merge + blend of one pixel.  gofs_top / gofs_bot: global slot = cursor + gofs (per cell row).
// TT = float in the tile kernel, double in the long-run path (thousands of factors).
template <int D, bool DUMP, typename TT>
__device__ __forceinline__ void blend_pixel(const uint32_t* dk, const float4* Ra, const float4* Rf, PixLists L, uint32_t gofs_top,
                                            uint32_t gofs_bot, float* __restrict__ gT, float (&acc)[D], float& accA,
                                            uint4& consumed, uint32_t* __restrict__ sorted_idx,
                                            uint32_t* __restrict__ sorted_depth, float* __restrict__ sorted_T,
                                            uint32_t obase) {
    constexpr int FV = D / 4;
    const uint32_t s0 = L.c0, s1 = L.c1, s2 = L.c2, s3 = L.c3;
    uint32_t c0 = L.c0, c1 = L.c1, c2 = L.c2, c3 = L.c3;
    uint32_t h0 = c0 < L.e0 ? dk[c0] : kSentHi, h1 = c1 < L.e1 ? dk[c1] : kSentHi;
    uint32_t h2 = c2 < L.e2 ? dk[c2] : kSentHi, h3 = c3 < L.e3 ? dk[c3] : kSentHi;
#pragma unroll
    for (int d = 0; d < D; ++d) acc[d] = 0.f;
    accA = 0.f;
    TT T = (TT)1;
    bool blending = true;
    uint32_t k = 0;
    while (true) {
        const uint32_t m = min(min(h0, h1), min(h2, h3));
        if (m == kSentHi) break;
        if (blending && T < (TT)kTMin) {                 // fragment k is blended iff T_k >= 1e-4
            blending = false;
            consumed = make_uint4(c0 - s0, c1 - s1, c2 - s2, c3 - s3);
            if (!DUMP) break;
        }
        int j = h0 == m ? 0 : (h1 == m ? 1 : (h2 == m ? 2 : 3));
        if ((int)(h0 == m) + (int)(h1 == m) + (int)(h2 == m) + (int)(h3 == m) > 1) {
            uint32_t best = 0xFFFFFFFFu;                 // equal depth bits: ascending point index
            if (h0 == m) { const uint32_t i = __float_as_uint(Ra[c0].w); if (i < best) { best = i; j = 0; } }
            if (h1 == m) { const uint32_t i = __float_as_uint(Ra[c1].w); if (i < best) { best = i; j = 1; } }
            if (h2 == m) { const uint32_t i = __float_as_uint(Ra[c2].w); if (i < best) { best = i; j = 2; } }
            if (h3 == m) { const uint32_t i = __float_as_uint(Ra[c3].w); if (i < best) { best = i; j = 3; } }
        }
        const uint32_t ref = j == 0 ? c0 : (j == 1 ? c1 : (j == 2 ? c2 : c3));
        const uint32_t end = j == 0 ? L.e0 : (j == 1 ? L.e1 : (j == 2 ? L.e2 : L.e3));
        const float4 r0 = Ra[ref];                   // tx, ty, opacity, idx
        if (blending) {
            const float wx = (j & 1) ? 1.f - r0.x : r0.x;       // lists 0, 2: corner dx = 1 (weight tx)
            const float wy = (j & 2) ? 1.f - r0.y : r0.y;       // lists 0, 1: corner dy = 1 (weight ty)
            const float a = r0.z * (wx * wy);                     // Eq. 7
            const float c = (float)T * a;
            accA += c;
#pragma unroll
            for (int v = 0; v < D / 4; ++v) {
                const float4 f = Rf[ref * FV + v];
                acc[4 * v] += c * f.x; acc[4 * v + 1] += c * f.y; acc[4 * v + 2] += c * f.z; acc[4 * v + 3] += c * f.w;
            }
            if (gT) gT[(size_t)(ref + ((j & 2) ? gofs_bot : gofs_top)) * 4 + (3 - j)] = (float)T;
            if (DUMP) sorted_T[obase + k] = (float)T;
            T *= (TT)(1.f - a);
        } else if (DUMP) {
            sorted_T[obase + k] = -1.f;                  // behind the cut-off: recorded, not blended
        }
        if (DUMP) {
            sorted_idx[obase + k] = __float_as_uint(r0.w);
            sorted_depth[obase + k] = m;
            ++k;
        }
        const uint32_t nx = ref + 1;
        const uint32_t nh = nx < end ? dk[nx] : kSentHi;
        if (j == 0) { c0 = nx; h0 = nh; } else if (j == 1) { c1 = nx; h1 = nh; }
        else if (j == 2) { c2 = nx; h2 = nh; } else { c3 = nx; h3 = nh; }
    }
    if (blending) consumed = make_uint4(c0 - s0, c1 - s1, c2 - s2, c3 - s3);
}

// Backward of one pixel: lists hold [start, start + consumed); gTa is indexed like dk (cursor * 4 + corner).
template <int D, typename TT>
__device__ __forceinline__ void backward_pixel(const uint32_t* dk, const float4* Ra, const float4* Rf, const float* gTa, PixLists L,
                                               uint32_t gofs_top, uint32_t gofs_bot, const float (&g)[D], float gA,
                                               float* __restrict__ gD) {
    constexpr int FV = D / 4;
    // c_j = one past the last blended record of list j; L.c_j = its start
    uint32_t c0 = L.e0, c1 = L.e1, c2 = L.e2, c3 = L.e3;
    uint32_t t0 = c0 > L.c0 ? dk[c0 - 1] : 0u, t1 = c1 > L.c1 ? dk[c1 - 1] : 0u;
    uint32_t t2 = c2 > L.c2 ? dk[c2 - 1] : 0u, t3 = c3 > L.c3 ? dk[c3 - 1] : 0u;
    TT B = (TT)0;
    while (true) {
        const uint32_t m = max(max(t0, t1), max(t2, t3));
        if (m == 0u) break;                              // depth bits are > 0 (z_c > near_z >= 0)
        int j = t0 == m ? 0 : (t1 == m ? 1 : (t2 == m ? 2 : 3));
        if ((int)(t0 == m) + (int)(t1 == m) + (int)(t2 == m) + (int)(t3 == m) > 1) {
            uint32_t best = 0u;                          // reverse order: descending point index
            if (t0 == m) { const uint32_t i = __float_as_uint(Ra[c0 - 1].w); if (i >= best) { best = i; j = 0; } }
            if (t1 == m) { const uint32_t i = __float_as_uint(Ra[c1 - 1].w); if (i >= best) { best = i; j = 1; } }
            if (t2 == m) { const uint32_t i = __float_as_uint(Ra[c2 - 1].w); if (i >= best) { best = i; j = 2; } }
            if (t3 == m) { const uint32_t i = __float_as_uint(Ra[c3 - 1].w); if (i >= best) { best = i; j = 3; } }
        }
        const uint32_t ref = (j == 0 ? c0 : (j == 1 ? c1 : (j == 2 ? c2 : c3))) - 1u;
        const uint32_t start = j == 0 ? L.c0 : (j == 1 ? L.c1 : (j == 2 ? L.c2 : L.c3));
        const float4 r0 = Ra[ref];
        const float T = gTa[(size_t)ref * 4 + (3 - j)];
        const float wx = (j & 1) ? 1.f - r0.x : r0.x;
        const float wy = (j & 2) ? 1.f - r0.y : r0.y;
        const float a = r0.z * (wx * wy);
        float G = gA;
#pragma unroll
        for (int v = 0; v < D / 4; ++v) {
            const float4 f = Rf[ref * FV + v];
            G += f.x * g[4 * v] + f.y * g[4 * v + 1] + f.z * g[4 * v + 2] + f.w * g[4 * v + 3];
        }
        gD[(size_t)(ref + ((j & 2) ? gofs_bot : gofs_top)) * 4 + (3 - j)] = (float)((TT)T * ((TT)G - B));
        B = (TT)a * (TT)G + (TT)(1.f - a) * B;
        const uint32_t nt = ref > start ? dk[ref - 1] : 0u;
        if (j == 0) { c0 = ref; t0 = nt; } else if (j == 1) { c1 = ref; t1 = nt; }
        else if (j == 2) { c2 = ref; t2 = nt; } else { c3 = ref; t3 = nt; }
    }
}

}  // namespace inpc
