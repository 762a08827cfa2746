// noit_resolve_common.cuh -- argument block and the composite epilogue (S5) shared by the
// resolve kernels (general thread-per-pixel kernel and the staged ring kernel).
#pragma once
#include "noit_internal.cuh"

struct ResolveArgs {
    uint32_t P, F;
    int32_t W, H;
    const uint32_t* offsets;
    const float* depth;
    const void* rgba;
    float bg[3];
    const float* bg_image;         // per-pixel background [P][4] or NULL (NEXT-4)
    float* out_trans;
    float* out_final;
    float* out_depth1;
    float* features10;             // NEXT-4 (DFAOIT mode): optional [P][10] inspection output
    // S9
    const uint32_t* pixel_list;
    const uint32_t* pixel_count;
    // S7 / frame-global LOD (O7g)
    const float* pass_scales;      // device {w, s_2, s_3}: frame-global pass-2 / pass-3 lod
    const uint8_t* cell_level;
    const uint8_t* tile_lod;        // per-tile mode: bit 0 mixed, bit 1 depth-only, per 32-pixel tile
    uint8_t level_to_lod[4];
    const float* coarse_g[2];      // G[10] per coarse pixel, lod 1 (half) and lod 2 (quarter)
    int32_t coarse_w[2], coarse_h[2];
    // staged kernel
    const float4* mlp_packed;      // per-lane MMA fragments of the weights (NOIT_MLP_BF16)
    uint32_t num_tiles;
    // [1] finished warps; [64 + 32 c] ticket counter c < 2^NOIT_TICKET_COUNTERS_LOG2; self-resetting
    uint32_t* tile_counter;
};

// ADAPTIVE = per-tile lods from cell_level (S7); GLOBAL = frame-global lods from pass_scales (O7g):
// separate instantiations, so neither carries the other's state in registers
enum { NOIT_RESOLVE_ALL = 0, NOIT_RESOLVE_LIST = 1, NOIT_RESOLVE_ADAPTIVE = 2, NOIT_RESOLVE_GLOBAL = 3 };

#ifdef __CUDACC__
// lod > 0 pixel of S7 (O7): bilinear sample of G = [a2*C2 (3), a2, C_acc (3), A_tail, T_tail, N]
// at the full-res pixel centre, taps clamped to the coarse texels of the pixel's own leaf and to
// the image (A19).  lerp(a,b,w) = a + w(b-a), x first then y; the weights are dyadic.
// G is stored as 12 floats (three float4) per coarse pixel: [a2*C2 (3), a2, C_acc (3), A_tail,
// T_tail, N, pad, pad].  r = 1 << lod; the leaf side is 1 << leaf_shift pixels (both powers of two:
// shifts, no integer divisions).
#define NOIT_G_STRIDE 12
__device__ __forceinline__ void sample_coarse_g(const float* __restrict__ G, int cw, int ch, int lod,
                                                int leaf_shift, int x, int y, float out[10])
{
    const float inv_r = lod == 1 ? 0.5f : 0.25f;
    const float u = ((float)x + 0.5f) * inv_r - 0.5f, v = ((float)y + 0.5f) * inv_r - 0.5f;
    const float fu = floorf(u), fv = floorf(v);
    const int i0 = (int)fu, j0 = (int)fv;
    const float wx = u - fu, wy = v - fv;
    const int lx0 = (x >> leaf_shift) << leaf_shift, ly0 = (y >> leaf_shift) << leaf_shift;
    const int leaf_last = (1 << leaf_shift) - 1;
    const int tx_lo = lx0 >> lod, ty_lo = ly0 >> lod;
    const int tx_hi = min((lx0 + leaf_last) >> lod, cw - 1);
    const int ty_hi = min((ly0 + leaf_last) >> lod, ch - 1);
    const int xa = min(max(i0, tx_lo), tx_hi), xb = min(max(i0 + 1, tx_lo), tx_hi);
    const int ya = min(max(j0, ty_lo), ty_hi), yb = min(max(j0 + 1, ty_lo), ty_hi);
    const float4* g00 = reinterpret_cast<const float4*>(G) + 3 * ((size_t)ya * cw + xa);
    const float4* g10 = reinterpret_cast<const float4*>(G) + 3 * ((size_t)ya * cw + xb);
    const float4* g01 = reinterpret_cast<const float4*>(G) + 3 * ((size_t)yb * cw + xa);
    const float4* g11 = reinterpret_cast<const float4*>(G) + 3 * ((size_t)yb * cw + xb);
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        const float4 A4 = __ldg(g00 + q), B4 = __ldg(g10 + q), C4 = __ldg(g01 + q), D4 = __ldg(g11 + q);
        const float a[4] = {A4.x, A4.y, A4.z, A4.w}, b[4] = {B4.x, B4.y, B4.z, B4.w};
        const float c[4] = {C4.x, C4.y, C4.z, C4.w}, d[4] = {D4.x, D4.y, D4.z, D4.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (4 * q + k >= 10) continue;
            const float top = fmaf(wx, b[k] - a[k], a[k]), bot = fmaf(wx, d[k] - c[k], c[k]);
            out[4 * q + k] = fmaf(wy, bot - top, top);
        }
    }
}
// O5 / Eq. 4.  c1 = straight RGBA of layer 1; l2 = PREMULTIPLIED layer 2
// (a2*C2, a2); absent layers are all-zero (A10).  f is ignored when has_tail is false (A2).
__device__ __forceinline__ void composite_store(const ResolveArgs& A, uint32_t p, float4 c1,
                                                float4 l2, float d1, bool has_tail,
                                                const float f[3], float t_tail)
{
    const float t1 = 1.f - c1.w;
    const float t2 = t1 * (1.f - l2.w);                       // T_2
    const float g = has_tail ? t2 : 0.f;
    const float ct_r = fmaf(g, f[0], fmaf(t1, l2.x, c1.w * c1.x));
    const float ct_g = fmaf(g, f[1], fmaf(t1, l2.y, c1.w * c1.y));
    const float ct_b = fmaf(g, f[2], fmaf(t1, l2.z, c1.w * c1.z));
    const float t_tot = t2 * t_tail;
    if (A.out_trans)
        __stcs(reinterpret_cast<float4*>(A.out_trans) + p, make_float4(ct_r, ct_g, ct_b, t_tot));
    if (A.out_final) {
        float4 bg = make_float4(A.bg[0], A.bg[1], A.bg[2], 0.f);
        if (A.bg_image) bg = __ldcs(reinterpret_cast<const float4*>(A.bg_image) + p);
        __stcs(reinterpret_cast<float4*>(A.out_final) + p,
               make_float4(fmaf(t_tot, bg.x, ct_r), fmaf(t_tot, bg.y, ct_g), fmaf(t_tot, bg.z, ct_b),
                           1.f - t_tot));
    }
    if (A.out_depth1) __stcs(A.out_depth1 + p, d1);
}
#endif
