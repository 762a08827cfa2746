// noit_features.cu -- noit_build_features (S1-S3) and noit_infer (S4 alone).
// These two entry points materialise intermediates the fused resolve never writes; they exist
// for inspection, for parity of the selection / counts (bit-exact class) and as the un-fused
// reference arrangement of the path.  One pixel (row) per thread.
#include "noit_internal.cuh"

template <typename ColorT>
__global__ void __launch_bounds__(256)
build_features_kernel(uint32_t P, const uint32_t* __restrict__ offsets,
                      const float* __restrict__ depth, const ColorT* __restrict__ rgba,
                      noit_layers out)
{
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const uint32_t b = __ldg(offsets + p), e = __ldg(offsets + p + 1);
    PixelState<true> s;
    s.init();
    for (uint32_t j = b; j < e; ++j) s.push(__ldg(depth + j), load_rgba(rgba, j), j);
    const uint32_t n = e - b;
    if (out.idx1) out.idx1[p] = n >= 1 ? s.i1 - b : NOIT_ABSENT;
    if (out.idx2) out.idx2[p] = n >= 2 ? s.i2 - b : NOIT_ABSENT;
    if (out.count) out.count[p] = n;
    if (out.layer1) reinterpret_cast<float4*>(out.layer1)[p] = s.c1;
    if (out.layer2) reinterpret_cast<float4*>(out.layer2)[p] = s.c2;
    if (out.depth1) out.depth1[p] = n >= 1 ? s.d1 : 1.0f;
    if (out.tail_raw) {
        float* t = out.tail_raw + 5 * (size_t)p;
        t[0] = s.acc_r; t[1] = s.acc_g; t[2] = s.acc_b; t[3] = s.a_tail; t[4] = s.t_tail;
    }
    if (out.features) {
        float x[5];
        make_features((float)n, s.t_tail, s.acc_r, s.acc_g, s.acc_b, s.a_tail, x);
        float* f = out.features + 5 * (size_t)p;
#pragma unroll
        for (int k = 0; k < 5; ++k) f[k] = x[k];
    }
}

__global__ void __launch_bounds__(128)
infer_kernel(const __grid_constant__ MlpWeights W, const float* __restrict__ features, uint32_t n,
             float* __restrict__ tail_rgb)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    float x[5], f[3];
#pragma unroll
    for (int k = 0; k < 5; ++k) x[k] = __ldg(features + 5 * (size_t)r + k);
    mlp_forward(W, x, f);
#pragma unroll
    for (int k = 0; k < 3; ++k) tail_rgb[3 * (size_t)r + k] = f[k];
}

extern "C" {

noit_status noit_build_features(noit_ctx* ctx, const noit_fragbuf* fb, const noit_layers* out,
                                void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_build_features: ctx is NULL");
    NOIT_TRY(noit_check_fragbuf(ctx, fb, "noit_build_features"));
    if (!out) return noit_fail(ctx, NOIT_ERR_NULL, "noit_build_features: out is NULL");
    if (!out->idx1 && !out->idx2 && !out->count && !out->layer1 && !out->layer2 && !out->depth1 &&
        !out->tail_raw && !out->features)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_build_features: every output is NULL");
    if (!noit_aligned(out->layer1, 16) || !noit_aligned(out->layer2, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_build_features: layer1/2 need 16-byte alignment");
    const uint32_t P = (uint32_t)fb->width * (uint32_t)fb->height;
    const dim3 grid((P + 255) / 256), block(256);
    cudaStream_t st = (cudaStream_t)stream;
    if (fb->color_fmt == NOIT_RGBA_F16)
        build_features_kernel<__half><<<grid, block, 0, st>>>(
            P, fb->offsets, fb->depth, (const __half*)fb->rgba, *out);
    else
        build_features_kernel<float><<<grid, block, 0, st>>>(
            P, fb->offsets, fb->depth, (const float*)fb->rgba, *out);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

noit_status noit_infer(noit_ctx* ctx, const float* features, uint32_t n, float* tail_rgb,
                       void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_infer: ctx is NULL");
    if (!ctx->has_weights) return noit_fail(ctx, NOIT_ERR_NO_WEIGHTS, "noit_infer: no weights set");
    if (n == 0) return NOIT_OK;
    if (!features || !tail_rgb) return noit_fail(ctx, NOIT_ERR_NULL, "noit_infer: NULL buffer");
    infer_kernel<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(ctx->w, features, n, tail_rgb);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

}  // extern "C"
