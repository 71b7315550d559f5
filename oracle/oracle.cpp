// ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, single-threaded CPU implementation of INPC's differentiable bilinear point
// rasterizer (arXiv 2403.16862, Sec. 3.4 + App. A.6), written from the paper as the plain
// definition of what the hot path computes: Eq. 1 applied, per pixel, to the
// depth-sorted multiset of Eq. 7 fragments of the Eq. 6 projections
// (PAPER.md:118-120).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// `--impl reference` leg may build, load or call this file.  It shares no code, header, table or
// helper with paper_2403_16862_b200/csrc (the CUDA path) and neither includes the other.
//
// Structure (deliberately unlike the GPU pipeline): one std::vector<Frag> bucket per pixel,
// std::sort per bucket, sequential fp64 compositing, sequential reverse traversal for gradients.
// All arithmetic is fp64 EXCEPT step S1 (the projection that decides the discrete quantities:
// cull, pixel index, depth key), which is BY SPECIFICATION a fixed sequence of individually
// rounded fp32 operations (reading R1) so that "bit-exact per-pixel counts and
// sorted order" is well defined.  Build with -ffp-contract=off (no FMA contraction).
//
// Readings of the paper taken here (DESIGN.md section 3 lists them all):
//   pixel centres at (i+0.5, j+0.5); pinhole divide; camera-space z orders fragments, ties broken
//   by ascending point index; per-FRAGMENT in-image test; near < z < far strict; zero-weight
//   fragments kept and counted; fragment k blended iff the transmittance before it is >= t_min
//   (1e-4 in BASELINE.json's north_star; not in the paper); premultiplied features; alpha output.
//
// Threads: none.  The `#pragma omp` lines below are inert in the build every test uses (no -fopenmp);
// bench.py's all-cores baseline leg builds the SAME source a second time with -fopenmp (liboracle_omp.so,
// SURVEY.md section 8d "Oracle timed beside it" (2)): pixels are independent in S3 / S4, and in the backward
// pass the per-point sums become `omp atomic` updates.  The arithmetic is untouched.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): closed forms, invariants, brute force, the adjoint
// of torch grid_sample, central finite differences, an independent torch-autograd restatement.
// No function here is "parity unpinned".
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Frag {
    uint32_t depth_bits;   // raw bits of the fp32 camera-space z (positive => unsigned order = numeric order)
    int64_t  idx;          // point index (tie-break, A8)
    double   w;            // bilinear weight, Eq. 7
    double   dwdu, dwdv;   // d w / d u, d w / d v  (A10)
    double   T;            // transmittance in front of this fragment (filled by blend)
    double   a;            // opacity * w (filled by blend)
};

struct Camera {
    float fx, fy, cx, cy;
    float R[9], t[3];
    float near_z, far_z;
    int32_t width, height;
};

struct State {
    int W = 0, H = 0, D = 0;
    int64_t N = 0;
    std::vector<std::vector<Frag>> bucket;   // one per pixel, row-major [H][W]
    std::vector<uint32_t> nb;                // blended count per pixel (valid after blend)
    std::vector<float>  opacity;             // copies of the inputs
    std::vector<float>  feat;
    int64_t kept = 0;                        // points that passed the depth / finiteness / range cull
    int64_t border_dropped = 0;              // fragments of kept points that fell outside the image
    bool blended = false;
};

// S2: the (up to) four fragments of one projected point.  fu = u - 0.5, fv = v - 0.5 and
// x0 = floor(fu), y0 = floor(fv) are given; tx, ty in [0,1).  Eq. 7 with centres at x0+0.5:
// 1-|u-u_i| = 1-tx for the left pixel, tx for the right one.
void emit(State& s, double fu, double fv, double x0, double y0, uint32_t depth_bits, int64_t i) {
    const double tx = fu - x0, ty = fv - y0;
    s.kept++;
    for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx) {
            const long px = (long)x0 + dx, py = (long)y0 + dy;
            if (px < 0 || px >= s.W || py < 0 || py >= s.H) { s.border_dropped++; continue; }
            const double wx = dx ? tx : 1.0 - tx;
            const double wy = dy ? ty : 1.0 - ty;
            Frag f;
            f.depth_bits = depth_bits;
            f.idx = i;
            f.w = wx * wy;
            f.dwdu = (dx ? 1.0 : -1.0) * wy;
            f.dwdv = (dy ? 1.0 : -1.0) * wx;
            f.T = 0.0; f.a = 0.0;
            s.bucket[(size_t)py * s.W + px].push_back(f);
        }
}

// S3: ascending (depth_bits, idx).
void sort_buckets(State& s) {
    const long P = (long)s.bucket.size();
#pragma omp parallel for schedule(dynamic, 256)
    for (long p = 0; p < P; ++p) {
        auto& b = s.bucket[p];
        std::sort(b.begin(), b.end(), [](const Frag& x, const Frag& y) {
            if (x.depth_bits != y.depth_bits) return x.depth_bits < y.depth_bits;
            return x.idx < y.idx;
        });
    }
}

State* new_state(int64_t N, int D, int W, int H, const float* opacity, const float* feat) {
    State* s = new State;
    s->W = W; s->H = H; s->D = D; s->N = N;
    s->bucket.resize((size_t)W * H);
    s->nb.assign((size_t)W * H, 0);
    s->opacity.assign(opacity, opacity + N);
    s->feat.assign(feat, feat + (size_t)N * D);
    return s;
}

}  // namespace

extern "C" {

// S1 + S2 + S3 from world-space points.  The projection is the canonical fp32 sequence:
// every operation below is one IEEE fp32 operation, in this order, never fused.
// Follows Eq. 6 with the pinhole divide (reading A2), near/far of PAPER.md:310.
void* oracle_create(const float* pos, const float* opacity, const float* feat, int64_t N, int32_t D,
                    const Camera* cam) {
    State* s = new_state(N, D, cam->width, cam->height, opacity, feat);
    const float* R = cam->R;
    const float Wm1 = (float)(cam->width - 1), Hm1 = (float)(cam->height - 1);
    for (int64_t i = 0; i < N; ++i) {
        const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        float m0, m1, m2, acc;
        m0 = R[0] * x; m1 = R[1] * y; acc = m0 + m1; m2 = R[2] * z; acc = acc + m2; const float xc = acc + cam->t[0];
        m0 = R[3] * x; m1 = R[4] * y; acc = m0 + m1; m2 = R[5] * z; acc = acc + m2; const float yc = acc + cam->t[1];
        m0 = R[6] * x; m1 = R[7] * y; acc = m0 + m1; m2 = R[8] * z; acc = acc + m2; const float zc = acc + cam->t[2];
        if (!(zc > cam->near_z && zc < cam->far_z)) continue;            // strict; false for NaN
        float nu = cam->fx * xc; nu = nu / zc; const float u = nu + cam->cx;
        float nv = cam->fy * yc; nv = nv / zc; const float v = nv + cam->cy;
        if (!std::isfinite(u) || !std::isfinite(v)) continue;
        const float fu = u - 0.5f, fv = v - 0.5f;
        const float x0 = std::floor(fu), y0 = std::floor(fv);
        // a point whose four pixels are all outside the image emits nothing (range-checked as floats)
        if (!(x0 >= -1.0f && x0 <= Wm1 && y0 >= -1.0f && y0 <= Hm1)) continue;
        uint32_t bits; std::memcpy(&bits, &zc, 4);
        emit(*s, (double)fu, (double)fv, (double)x0, (double)y0, bits, i);   // fu - x0 is exact in fp64
    }
    sort_buckets(*s);
    return s;
}

// Same pipeline from already-projected image coordinates in fp64 (no camera, no cull except the
// image range): lets tests perturb u, v for finite differences and pin the weights in isolation.
void* oracle_create_uv(const double* u, const double* v, const float* depth, const float* opacity,
                       const float* feat, int64_t N, int32_t D, int32_t W, int32_t H) {
    State* s = new_state(N, D, W, H, opacity, feat);
    for (int64_t i = 0; i < N; ++i) {
        const double fu = u[i] - 0.5, fv = v[i] - 0.5;
        const double x0 = std::floor(fu), y0 = std::floor(fv);
        if (!(x0 >= -1.0 && x0 <= W - 1 && y0 >= -1.0 && y0 <= H - 1)) continue;
        uint32_t bits; std::memcpy(&bits, &depth[i], 4);
        emit(*s, fu, fv, x0, y0, bits, i);
    }
    sort_buckets(*s);
    return s;
}

void oracle_free(void* h) { delete (State*)h; }

int64_t oracle_total(void* h) {
    State* s = (State*)h; int64_t t = 0;
    for (auto& b : s->bucket) t += (int64_t)b.size();
    return t;
}
int64_t oracle_kept(void* h) { return ((State*)h)->kept; }
// threads the build can use: 1 unless compiled with -fopenmp (bench.py's all-cores leg)
int oracle_threads(void) {
#ifdef _OPENMP
    int n = 1;
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
    return n;
#else
    return 1;
#endif
}
int64_t oracle_border_dropped(void* h) { return ((State*)h)->border_dropped; }

void oracle_counts(void* h, uint32_t* counts) {
    State* s = (State*)h;
    for (size_t p = 0; p < s->bucket.size(); ++p) counts[p] = (uint32_t)s->bucket[p].size();
}

// offsets[P+1] (exclusive sum of counts), then per fragment in pixel-major sorted order:
// point index, depth bits, bilinear weight.
void oracle_sorted(void* h, int64_t* offsets, int64_t* point_idx, uint32_t* depth_bits, double* weight) {
    State* s = (State*)h; int64_t o = 0;
    for (size_t p = 0; p < s->bucket.size(); ++p) {
        offsets[p] = o;
        for (auto& f : s->bucket[p]) {
            point_idx[o] = f.idx; depth_bits[o] = f.depth_bits;
            if (weight) weight[o] = f.w;
            ++o;
        }
    }
    offsets[s->bucket.size()] = o;
}

// S4: front-to-back compositing, Eq. 1 (product index read as j < i).
// Fragment k is blended iff T_k >= t_min (t_min = 1e-4: north_star; t_min <= 0 disables the cut-off).
// Outputs: img[H][W][D] premultiplied, alpha[H][W] = sum of blended T*a,
// nb[H][W] blended count, margin[H][W] = min_k |T_k - t_min| / t_min over every T the termination
// test looked at (harness rule for threshold-ambiguous pixels; +inf when t_min <= 0).
// force_nb (harness aid for those pixels, reading R7; NULL = off): where force_nb[p] is not
// 0xFFFFFFFF the termination test is replaced by "blend exactly the first force_nb[p] fragments" -- the
// compositing arithmetic is the same; margin[p] is +inf there.
void oracle_blend(void* h, double t_min, const uint32_t* force_nb, double* img, double* alpha, uint32_t* nb,
                  double* margin) {
    State* s = (State*)h; const int D = s->D;
    const long P = (long)s->bucket.size();
#pragma omp parallel for schedule(dynamic, 256)
    for (long p = 0; p < P; ++p) {
        double T = 1.0, A = 0.0, m = INFINITY;
        double* C = img + p * D;
        for (int d = 0; d < D; ++d) C[d] = 0.0;
        uint32_t n = 0;
        const bool forced = force_nb && force_nb[p] != 0xFFFFFFFFu;
        for (auto& f : s->bucket[p]) {
            if (forced) {
                if (n >= force_nb[p]) break;
            } else {
                if (t_min > 0.0) m = std::min(m, std::fabs(T - t_min) / t_min);
                if (T < t_min) break;
            }
            const double a = (double)s->opacity[f.idx] * f.w;
            const float* F = &s->feat[(size_t)f.idx * D];
            for (int d = 0; d < D; ++d) C[d] += T * a * (double)F[d];
            A += T * a;
            f.T = T; f.a = a;
            T *= (1.0 - a);
            ++n;
        }
        alpha[p] = A;
        s->nb[p] = n;
        if (nb) nb[p] = n;
        if (margin) margin[p] = m;
    }
    s->blended = true;
}

// Per fragment, in the order of oracle_sorted: the transmittance T_k in front of it if the last
// oracle_blend composited it, -1 otherwise.
int oracle_sorted_T(void* h, double* T) {
    State* s = (State*)h;
    if (!s->blended) return -1;
    int64_t o = 0;
    for (size_t p = 0; p < s->bucket.size(); ++p) {
        uint32_t k = 0;
        for (auto& f : s->bucket[p]) { T[o++] = k < s->nb[p] ? f.T : -1.0; ++k; }
    }
    return 0;
}

// NEXT row f1 -- per-point blending weight, the input of the octree's probability update (Eq. 3,
// PAPER.md:75-78): "we use the transmitted blending weight b_j = alpha_j T_j (Eq. (1)) for the updates".
// A point has up to four fragments (Eq. 7); its weight is the largest alpha T among those the last
// oracle_blend composited (reading: a point "generated using the i-th leaf" contributes through whichever
// of its splats is most visible; the max over the points of a leaf is the sampler's).  Points without a
// blended fragment (culled, outside the image, or entirely behind the cut-off) get 0.
int oracle_blend_weights(void* h, double* bw) {
    State* s = (State*)h;
    if (!s->blended) return -1;
    for (int64_t i = 0; i < s->N; ++i) bw[i] = 0.0;
    for (size_t p = 0; p < s->bucket.size(); ++p)
        for (uint32_t k = 0; k < s->nb[p]; ++k) {
            const Frag& f = s->bucket[p][k];
            bw[f.idx] = std::max(bw[f.idx], f.a * f.T);
        }
    return 0;
}

// S5 + S6: gradients of  L = <g_img, img> + <g_alpha, alpha>  w.r.t. features, opacities and the
// projected position (u, v) of every point (per-splat gradients in forward order,
// four splat gradients combined with the bilinear weights).  Division-free reverse recurrence:
// with G_k = sum_d feat[i_k][d] g[p][d] + gA[p],
//   dL/da_k = T_k (G_k - B_k),   B_{k-1} = a_k G_k + (1 - a_k) B_k,   B_{nb-1} = 0,
// because d/da_k sum_j T_j a_j G_j = T_k G_k - sum_{j>k} T_j a_j G_j / (1 - a_k) and
// B_k = sum_{j>k} a_j G_j prod_{k<m<j} (1 - a_m).  No gradient through the sort or the cut-off.
int oracle_backward(void* h, const double* g_img, const double* g_alpha,
                    double* d_feat, double* d_opacity, double* d_uv) {
    State* s = (State*)h; const int D = s->D;
    if (!s->blended) return -1;
    for (int64_t i = 0; i < s->N * D; ++i) d_feat[i] = 0.0;
    for (int64_t i = 0; i < s->N; ++i) { d_opacity[i] = 0.0; d_uv[2 * i] = 0.0; d_uv[2 * i + 1] = 0.0; }
    const long P = (long)s->bucket.size();
#pragma omp parallel for schedule(dynamic, 256)
    for (long p = 0; p < P; ++p) {
        const double* g = g_img + p * D;
        const double gA = g_alpha ? g_alpha[p] : 0.0;
        auto& b = s->bucket[p];
        double B = 0.0;
        for (int64_t k = (int64_t)s->nb[p] - 1; k >= 0; --k) {
            const Frag& f = b[k];
            const float* F = &s->feat[(size_t)f.idx * D];
            double G = gA;
            for (int d = 0; d < D; ++d) G += (double)F[d] * g[d];
            const double dLda = f.T * (G - B);
            B = f.a * G + (1.0 - f.a) * B;
            for (int d = 0; d < D; ++d) {
#pragma omp atomic
                d_feat[(size_t)f.idx * D + d] += f.T * f.a * g[d];
            }
            const double op = (double)s->opacity[f.idx];
#pragma omp atomic
            d_opacity[f.idx] += f.w * dLda;
#pragma omp atomic
            d_uv[2 * f.idx]     += op * f.dwdu * dLda;
#pragma omp atomic
            d_uv[2 * f.idx + 1] += op * f.dwdv * dLda;
        }
    }
    return 0;
}

// Diagnostic only (never gated): how many points would change pixel or cull status if S1 were
// evaluated in fp64 instead of the canonical fp32 sequence.
int64_t oracle_count_fp64_projection_changes(const float* pos, int64_t N, const Camera* cam) {
    int64_t changed = 0;
    const float* R = cam->R;
    for (int64_t i = 0; i < N; ++i) {
        const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        float m0, m1, m2, acc;
        m0 = R[0] * x; m1 = R[1] * y; acc = m0 + m1; m2 = R[2] * z; acc = acc + m2; const float xc = acc + cam->t[0];
        m0 = R[3] * x; m1 = R[4] * y; acc = m0 + m1; m2 = R[5] * z; acc = acc + m2; const float yc = acc + cam->t[1];
        m0 = R[6] * x; m1 = R[7] * y; acc = m0 + m1; m2 = R[8] * z; acc = acc + m2; const float zc = acc + cam->t[2];
        const bool keep32 = (zc > cam->near_z && zc < cam->far_z);
        float nu = cam->fx * xc; nu = nu / zc; const float u = nu + cam->cx;
        float nv = cam->fy * yc; nv = nv / zc; const float v = nv + cam->cy;
        const double X = (double)R[0] * x + (double)R[1] * y + (double)R[2] * z + cam->t[0];
        const double Y = (double)R[3] * x + (double)R[4] * y + (double)R[5] * z + cam->t[1];
        const double Z = (double)R[6] * x + (double)R[7] * y + (double)R[8] * z + cam->t[2];
        const bool keep64 = (Z > cam->near_z && Z < cam->far_z);
        if (keep32 != keep64) { changed++; continue; }
        if (!keep32) continue;
        const double U = cam->fx * X / Z + cam->cx, V = cam->fy * Y / Z + cam->cy;
        if (std::floor((double)(u - 0.5f)) != std::floor(U - 0.5) ||
            std::floor((double)(v - 0.5f)) != std::floor(V - 0.5)) changed++;
    }
    return changed;
}

}  // extern "C"
