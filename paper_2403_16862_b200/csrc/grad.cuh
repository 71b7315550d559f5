// grad.cuh -- the last stage of step a5: "the per-point gradient [is computed] by combining its four splat
// gradients in a weighted sum according to the ... bilinear interpolation weights".
//
//   k_combine  one thread per RECORD (slot order, coalesced): reads the record's four (T, dL/da) pairs
//              from gT / gD, decides per corner whether that fragment was blended (its position in the
//              cell list < the pixel's stop position pcur; the four corner pixels' limits and image gradients
//              are staged once per CELL in shared memory), and forms
//                 dL/dfeat    = sum_c T_c a_c g_img[pixel_c]            (S5)
//                 dL/dopacity = sum_c w_c dL/da_c                        (S6)
//                 dL/d(u, v)  = opacity * sum_c (dw_c/du, dw_c/dv) dL/da_c
//              and, in the same pass, the point's BLENDING WEIGHT  b = max_c T_c a_c  over its blended
//              fragments (Eq. 3's update input; "fused into this pipeline"),
//              and writes them as ONE (D = 4) or TWO (D = 8) full 32-byte sectors to gpt[point_idx]: the
//              only scattered write of the backward pass, and never narrower than a sector.  No atomics:
//              every fragment has exactly one writer, so gradients are bit-reproducible run to run.
//   k_split    one thread per POINT: gpt -> grad_feat[N][D], grad_opacity[N], grad_uv[N][2] and, when asked for,
//              blend_weight[N] (coalesced); culled points (their bit of the kept mask is 0) get exact zeros.
#pragma once
#include "common.cuh"
#include "sh.cuh"

namespace inpc {

constexpr int kGradThreads = 256;
constexpr int kGradCells   = 128;      // cells per work unit
constexpr int kGradPart    = 4096;     // a unit with more records than this is cut into parts of this many (see k_combine)

template <int D> __host__ __device__ constexpr int gpt_floats() { return D == 4 ? 8 : 16; }

template <int D>
__global__ void __launch_bounds__(kGradThreads) k_combine(Header* __restrict__ hdr,
                                                           const uint32_t* __restrict__ celloff, uint32_t C,
                                                           uint32_t unit_begin, uint32_t unit_end, int W,
                                                           int H, const float4* __restrict__ Ra,
                                                           const float4* __restrict__ gT, const float4* __restrict__ gD,
                                                           const uint4* __restrict__ pcur,
                                                           const float* __restrict__ g_feat, ImageIO io,
                                                           float* __restrict__ gpt, unsigned long long* __restrict__ queue) {
    constexpr int GP = gpt_floats<D>();
    constexpr int FV = D / 4;
    __shared__ uint32_t s_off[kGradCells + 1];
    // per (cell of the unit, corner): how many records of the cell the corner's pixel blended (0: pixel outside the
    // image) and that pixel's image gradient, loaded ONCE per cell -- every record of a cell needs the same four pixels
    __shared__ uint32_t s_lim[kGradCells][4];
    __shared__ float4   s_g[kGradCells][4][FV];
    __shared__ uint32_t s_unit, s_part;
    const int tid = threadIdx.x;
    if (!hdr->bwd_ok) return;
    const uint32_t n_units = unit_end - unit_begin;
    // Units (kGradCells cells) are handed out dynamically.  Their record counts differ by orders of magnitude (a cell
    // holds anything from 0 to tens of thousands of records), so a unit with more than kGradPart records is cut into
    // parts: the CTA that draws the unit takes part 0 and queues the others (queue[]: unit | part << 32); a CTA that
    // finds no unit left takes parts from the queue.  A CTA that queues parts keeps drawing work itself afterwards, so
    // every queued part is taken by someone.
    while (true) {
        __syncthreads();
        if (tid == 0) {
            uint32_t u = atomicAdd(&hdr->combine_cursor, 1u), part = 0u;
            if (u >= n_units) {
                // take a ticket; it is good once the queue has grown past it, and void once every unit has been drawn and
                // has queued what it was going to queue (combine_done == n_units: the tail is final)
                u = 0xFFFFFFFFu;
                const uint32_t t = atomicAdd(&hdr->combine_q_head, 1u);
                while (true) {
                    const bool final = *reinterpret_cast<volatile uint32_t*>(&hdr->combine_done) >= n_units;
                    __threadfence();
                    if (t < *reinterpret_cast<volatile uint32_t*>(&hdr->combine_q_tail)) {
                        unsigned long long e;                                                      // (queue[] starts out as all ones)
                        while ((e = *reinterpret_cast<volatile unsigned long long*>(&queue[t])) == ~0ull) { }   // its writer is about to store it
                        u = (uint32_t)e; part = (uint32_t)(e >> 32);
                        break;
                    }
                    if (final) break;
                }
            }
            s_unit = u; s_part = part;
        }
        __syncthreads();
        if (s_unit == 0xFFFFFFFFu) break;
        const uint32_t unit = unit_begin + s_unit, part = s_part;
        const uint32_t c0 = unit * kGradCells, nc = min((uint32_t)kGradCells, C - c0);
        for (uint32_t c = tid; c <= nc; c += kGradThreads) s_off[c] = __ldg(&celloff[c0 + c]);
        for (uint32_t e = tid; e < nc * 4u; e += kGradThreads) {
            const uint32_t cl = e >> 2, c = e & 3u;
            const uint32_t cell = c0 + cl;
            const int j = cell / (W + 1), i = cell - j * (W + 1);
            const int px = i - 1 + (int)(c & 1u), py = j - 1 + (int)(c >> 1);
            uint32_t lim = 0;
            float4 g[FV];
#pragma unroll
            for (int v = 0; v < FV; ++v) g[v] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (px >= 0 && px < W && py >= 0 && py < H) {                    // else: the fragment does not exist
                const size_t pp = (size_t)py * W + px;
                const uint4 cur = __ldg(&pcur[pp]);
                lim = c == 3 ? cur.x : (c == 2 ? cur.y : (c == 1 ? cur.z : cur.w));   // the cell is the pixel's list 3 - c
#pragma unroll
                for (int v = 0; v < FV; ++v) {
                    if (!io.planar) g[v] = __ldg(reinterpret_cast<const float4*>(g_feat + pp * D) + v);
                    else g[v] = make_float4(__ldg(g_feat + (size_t)(4 * v) * io.P + pp), __ldg(g_feat + (size_t)(4 * v + 1) * io.P + pp),
                                            __ldg(g_feat + (size_t)(4 * v + 2) * io.P + pp), __ldg(g_feat + (size_t)(4 * v + 3) * io.P + pp));
                }
            }
            s_lim[cl][c] = lim;
#pragma unroll
            for (int v = 0; v < FV; ++v) s_g[cl][c][v] = g[v];
        }
        __syncthreads();
        const uint32_t S0 = s_off[0], E0 = s_off[nc];
        const uint32_t n_parts = (E0 - S0 + kGradPart - 1) / kGradPart;
        if (part == 0u && tid == 0) {                            // queue the other parts of a large unit
            if (n_parts > 1u) {
                const uint32_t at = atomicAdd(&hdr->combine_q_tail, n_parts - 1u);
                for (uint32_t q = 1; q < n_parts; ++q)
                    *reinterpret_cast<volatile unsigned long long*>(&queue[at + q - 1u]) = (unsigned long long)s_unit | ((unsigned long long)q << 32);
            }
            __threadfence();
            atomicAdd(&hdr->combine_done, 1u);
        }
        const uint32_t S = S0 + part * kGradPart, E = min(E0, S + (uint32_t)kGradPart);
        uint32_t lo = 0;                                         // a thread's slots ascend: the search resumes at its last cell
        for (uint32_t slot = S + tid; slot < E; slot += kGradThreads) {
            // the record's own (coalesced) loads first: they do not depend on the cell search
            const float4 r0 = __ldg(&Ra[slot]);                   // tx, ty, opacity, idx
            const float4 t4 = __ldcs(&gT[slot]), d4 = __ldcs(&gD[slot]);
            // cell of this slot: the last c with s_off[c] <= slot (empty cells repeat offsets)
            uint32_t hi = nc - 1;
            while (lo < hi) {
                const uint32_t mid = (lo + hi + 1) >> 1;
                if (s_off[mid] <= slot) lo = mid; else hi = mid - 1;
            }
            const uint32_t r = slot - s_off[lo];
            const float tc[4] = {t4.x, t4.y, t4.z, t4.w}, dc[4] = {d4.x, d4.y, d4.z, d4.w};
            float df[D];
#pragma unroll
            for (int d = 0; d < D; ++d) df[d] = 0.f;
            float dop = 0.f, du = 0.f, dv = 0.f, bw = 0.f;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int dx = c & 1, dy = c >> 1;
                if (r >= s_lim[lo][c]) continue;                           // behind the cut-off or outside the image: exactly 0
                const float wx = dx ? r0.x : 1.f - r0.x, wy = dy ? r0.y : 1.f - r0.y;
                const float Ta = tc[c] * (r0.z * (wx * wy));
                const float dl = dc[c];
                bw = fmaxf(bw, Ta);                                        // b = alpha T of this fragment (Eq. 3)
                dop += wx * wy * dl;
                du += (dx ? wy : -wy) * dl;
                dv += (dy ? wx : -wx) * dl;
                const float Tg = io.scale * Ta;                            // the gradient image's scale, applied once (1: exact)
#pragma unroll
                for (int v = 0; v < FV; ++v) {
                    const float4 t = s_g[lo][c][v];
                    df[4 * v] += Tg * t.x; df[4 * v + 1] += Tg * t.y; df[4 * v + 2] += Tg * t.z; df[4 * v + 3] += Tg * t.w;
                }
            }
            du *= r0.z; dv *= r0.z;
            float4* out = reinterpret_cast<float4*>(gpt + (size_t)__float_as_uint(r0.w) * GP);
            if (D == 4) {
                st_sector(out, make_float4(df[0], df[1], df[2], df[3]), make_float4(dop, du, dv, bw));
            } else {
                st_sector(out, make_float4(df[0], df[1], df[2], df[3]), make_float4(df[4], df[5], df[6], df[7]));
                st_sector(out + 2, make_float4(dop, du, dv, bw), make_float4(0.f, 0.f, 0.f, 0.f));
            }
        }
    }
}

// SH (NEXT row f2): d_feat is dL/dcoeff[N][36] = Y_b(dir) dL/dfeature[d] instead of dL/dfeature[N][4]; pos / view give
// the direction (no gradient flows into the position through it: the paper's positions are sampled, not optimised).
template <int D, bool SH>
__global__ void __launch_bounds__(256) k_split(const Header* __restrict__ hdr, const float* __restrict__ gpt,
                                                const uint32_t* __restrict__ kept,
                                                long long N, float* __restrict__ d_feat, float* __restrict__ d_opacity,
                                                float* __restrict__ d_uv, float* __restrict__ blend_weight,
                                                const float* __restrict__ pos, ViewPoint view) {
    constexpr int GP = gpt_floats<D>();
    if (!hdr->bwd_ok) return;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        float4 f[D / 4], o = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int v = 0; v < D / 4; ++v) f[v] = make_float4(0.f, 0.f, 0.f, 0.f);
        if ((__ldg(&kept[i >> 5]) >> (i & 31)) & 1u) {
            const float4* in = reinterpret_cast<const float4*>(gpt + (size_t)i * GP);
#pragma unroll
            for (int v = 0; v < D / 4; ++v) f[v] = __ldcs(&in[v]);
            o = __ldcs(&in[D / 4]);
        }
        if (SH && d_feat) {
            float Y[kShBasis];
            sh_basis9(__ldg(&pos[3 * i]) - view.cx, __ldg(&pos[3 * i + 1]) - view.cy, __ldg(&pos[3 * i + 2]) - view.cz, Y);
#pragma unroll
            for (int b = 0; b < kShBasis; ++b)
                __stcs(reinterpret_cast<float4*>(d_feat + (size_t)i * kShCoeffs) + b,
                       make_float4(Y[b] * f[0].x, Y[b] * f[0].y, Y[b] * f[0].z, Y[b] * f[0].w));
        } else if (d_feat) {
#pragma unroll
            for (int v = 0; v < D / 4; ++v) __stcs(reinterpret_cast<float4*>(d_feat + (size_t)i * D) + v, f[v]);
        }
        if (d_opacity) __stcs(&d_opacity[i], o.x);          // any of the outputs may be NULL: its stores are skipped
        if (d_uv) __stcs(reinterpret_cast<float2*>(d_uv) + i, make_float2(o.y, o.z));
        if (blend_weight) __stcs(&blend_weight[i], o.w);
    }
}

}  // namespace inpc
