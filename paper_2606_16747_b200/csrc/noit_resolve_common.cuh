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
    float* out_trans;
    float* out_final;
    float* out_depth1;
    // S9
    const uint32_t* pixel_list;
    const uint32_t* pixel_count;
    // S7
    const uint8_t* cell_level;
    uint8_t level_to_lod[4];
    const float* coarse_g[2];      // G[10] per coarse pixel, lod 1 (half) and lod 2 (quarter)
    int32_t coarse_w[2], coarse_h[2];
    // staged kernel
    const float4* mlp_packed;      // per-lane MMA fragments of the weights (NOIT_MLP_BF16)
    uint32_t num_tiles;
    uint32_t* tile_counter;        // [0] next tile, [1] finished warps; self-resetting
};

#ifdef __CUDACC__
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
    if (A.out_final)
        __stcs(reinterpret_cast<float4*>(A.out_final) + p,
               make_float4(fmaf(t_tot, A.bg[0], ct_r), fmaf(t_tot, A.bg[1], ct_g),
                           fmaf(t_tot, A.bg[2], ct_b), 1.f - t_tot));
    if (A.out_depth1) __stcs(A.out_depth1 + p, d1);
}
#endif
