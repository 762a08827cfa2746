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

// S4 alone on the tensor cores (bf16-rounded weights, exact in TF32): the two-pass TF32 split of
// noit_internal.cuh, 32 rows per warp, 8 warps per CTA.  Rows are read and written coalesced
// through the warp's shared-memory scratch (160 + 96 floats per 32 rows); a grid-stride loop keeps
// the packed weights (10 float4 per lane) in registers across tiles.
constexpr int kInferWarps = 8;
__global__ void __launch_bounds__(kInferWarps * 32)
infer_mma_kernel(const float4* __restrict__ mlp_packed, const float* __restrict__ features, uint32_t n,
                 float* __restrict__ tail_rgb)
{
    __shared__ __align__(16) float scratch_s[kInferWarps][32 * 12];
    __shared__ __align__(16) float io_s[kInferWarps][32 * 5];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* const scratch = scratch_s[warp];
    float* const io = io_s[warp];
    float4 wv[NOIT_MMA_CHUNKS];
#pragma unroll
    for (int v = 0; v < NOIT_MMA_CHUNKS; ++v) wv[v] = __ldg(mlp_packed + v * 32 + lane);
    const uint32_t tiles = (n + 31u) / 32u, stride = gridDim.x * kInferWarps;
    for (uint32_t t = blockIdx.x * kInferWarps + warp; t < tiles; t += stride) {
        const size_t r0 = (size_t)t * 32;
        const uint32_t rows = min(32u, n - (uint32_t)r0);
        __syncwarp();
        for (uint32_t i = lane; i < rows * 5u; i += 32u) io[i] = __ldcs(features + 5 * r0 + i);   // coalesced
        __syncwarp();
        float x[5], f[3];
#pragma unroll
        for (int k = 0; k < 5; ++k) x[k] = (uint32_t)lane < rows ? io[5 * lane + k] : 0.f;
        mlp_forward_mma(MmaWeightsReg{wv}, scratch, lane, x, f);
        __syncwarp();
#pragma unroll
        for (int k = 0; k < 3; ++k) io[3 * lane + k] = f[k];
        __syncwarp();
        for (uint32_t i = lane; i < rows * 3u; i += 32u) __stcs(tail_rgb + 3 * r0 + i, io[i]);
    }
}

// NEXT-4: the comparison system's network, 10 -> 32 -> 16 -> 3 with a sigmoid output (
// 931 parameters).  Same shape of kernel as infer_kernel: one row per thread, weights as
// constant-bank operands of the FFMAs, dot products from the bias in input-index order.
struct MlpWeights10 {
    float w1[32][10];
    float b1[32];
    float w2[16][32];
    float b2[16];
    float w3[3][16];
    float b3[3];
};
static_assert(sizeof(MlpWeights10) == NOIT_DFAOIT_PARAMS * 4, "931 parameters");

__global__ void __launch_bounds__(128)
infer10_kernel(const __grid_constant__ MlpWeights10 W, const float* __restrict__ features, uint32_t n,
               float* __restrict__ rgb)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    float x[10], h1[32], h2[16];
#pragma unroll
    for (int k = 0; k < 10; ++k) x[k] = __ldg(features + 10 * (size_t)r + k);
#pragma unroll
    for (int o = 0; o < 32; ++o) {
        float a = W.b1[o];
#pragma unroll
        for (int i = 0; i < 10; ++i) a = fmaf(W.w1[o][i], x[i], a);
        h1[o] = fmaxf(a, 0.f);
    }
#pragma unroll
    for (int o = 0; o < 16; ++o) {
        float a = W.b2[o];
#pragma unroll
        for (int i = 0; i < 32; ++i) a = fmaf(W.w2[o][i], h1[i], a);
        h2[o] = fmaxf(a, 0.f);
    }
#pragma unroll
    for (int o = 0; o < 3; ++o) {
        float a = W.b3[o];
#pragma unroll
        for (int i = 0; i < 16; ++i) a = fmaf(W.w3[o][i], h2[i], a);
        rgb[3 * (size_t)r + o] = 1.0f / (1.0f + expf(-a));
    }
}

extern "C" {

noit_status noit_infer_dfaoit(noit_ctx* ctx, const float* host_w, int32_t count, const float* features,
                              uint32_t n, float* rgb, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_infer_dfaoit: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_infer_dfaoit"));
    if (!host_w) return noit_fail(ctx, NOIT_ERR_NULL, "noit_infer_dfaoit: host_w is NULL");
    if (count != NOIT_DFAOIT_PARAMS)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_infer_dfaoit: count %d != 931 (P:97-104)", count);
    if (n == 0) return NOIT_OK;
    if (!features || !rgb) return noit_fail(ctx, NOIT_ERR_NULL, "noit_infer_dfaoit: NULL buffer");
    MlpWeights10 w;
    memcpy(&w, host_w, sizeof w);
    infer10_kernel<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(w, features, n, rgb);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

noit_status noit_build_features(noit_ctx* ctx, const noit_fragbuf* fb, const noit_layers* out,
                                void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_build_features: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_build_features"));
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
    NOIT_TRY(noit_check_device(ctx, "noit_infer"));
    if (!ctx->has_weights) return noit_fail(ctx, NOIT_ERR_NO_WEIGHTS, "noit_infer: no weights set");
    if (n == 0) return NOIT_OK;
    if (!features || !tail_rgb) return noit_fail(ctx, NOIT_ERR_NULL, "noit_infer: NULL buffer");
    if (ctx->precision == NOIT_MLP_BF16 && ctx->d_mlp) {       // weights exact in TF32: tensor cores
        const uint32_t tiles = (n + 31u) / 32u;
        const uint32_t grid = min((tiles + kInferWarps - 1) / kInferWarps, (uint32_t)ctx->num_sms * 8u);
        infer_mma_kernel<<<grid, kInferWarps * 32, 0, (cudaStream_t)stream>>>(
            static_cast<const float4*>(ctx->d_mlp), features, n, tail_rgb);
    } else {
        infer_kernel<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(ctx->w, features, n, tail_rgb);
    }
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

}  // extern "C"

// ---- noit_validate_fragbuf: the CSR preconditions the hot kernels rely on ---------------------
__global__ void validate_offsets_kernel(const uint32_t* __restrict__ offsets, uint32_t P, uint32_t F,
                                        uint32_t* __restrict__ first_bad)
{
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p > P) return;
    bool bad = false;
    if (p == 0) bad = offsets[0] != 0u;
    if (p == P) bad = bad || offsets[P] != F;
    if (p < P) bad = bad || offsets[p + 1] < offsets[p];
    if (bad) atomicMin(first_bad, p);
}

extern "C" noit_status noit_validate_fragbuf(noit_ctx* ctx, const noit_fragbuf* fb, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_validate_fragbuf: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_validate_fragbuf"));
    NOIT_TRY(noit_check_fragbuf(ctx, fb, "noit_validate_fragbuf"));
    cudaStream_t st = (cudaStream_t)stream;
    const uint32_t P = (uint32_t)fb->width * (uint32_t)fb->height;
    uint32_t* flag = ctx->d_counters + 20;
    const uint32_t none = 0xFFFFFFFFu;
    NOIT_CUDA(ctx, cudaMemcpyAsync(flag, &none, sizeof none, cudaMemcpyHostToDevice, st));
    validate_offsets_kernel<<<(P + 1 + 255) / 256, 256, 0, st>>>(fb->offsets, P, fb->num_fragments, flag);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    uint32_t bad = none;
    NOIT_CUDA(ctx, cudaMemcpyAsync(&bad, flag, sizeof bad, cudaMemcpyDeviceToHost, st));
    NOIT_CUDA(ctx, cudaStreamSynchronize(st));
    if (bad != none)
        return noit_fail(ctx, NOIT_ERR_FORMAT,
                         "noit_validate_fragbuf: offsets are not a CSR of %u fragments (first violation at pixel %u)",
                         fb->num_fragments, bad);
    return NOIT_OK;
}
