// noit_api.cu -- context, weights, error reporting and argument checks of libnoit.so.
#include <stdarg.h>

#include <new>

#include "noit_internal.cuh"

static char g_err[512] = "no error";

noit_status noit_fail(noit_ctx* ctx, noit_status st, const char* fmt, ...)
{
    char* dst = ctx ? ctx->err : g_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return st;
}

noit_status noit_cuda_check(noit_ctx* ctx, cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return NOIT_OK;
    return noit_fail(ctx, NOIT_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

noit_status noit_check_device(noit_ctx* ctx, const char* who)
{
    int dev = -1;
    const cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noit_cuda_check(ctx, e, "cudaGetDevice");
    if (dev != ctx->device)
        return noit_fail(ctx, NOIT_ERR_CUDA, "%s: the context was created on device %d, the current device is %d",
                         who, ctx->device, dev);
    return NOIT_OK;
}

noit_status noit_check_fragbuf(noit_ctx* ctx, const noit_fragbuf* fb, const char* name)
{
    if (!fb) return noit_fail(ctx, NOIT_ERR_NULL, "%s: fragment buffer is NULL", name);
    if (fb->width <= 0 || fb->height <= 0)
        return noit_fail(ctx, NOIT_ERR_SIZE, "%s: width/height must be > 0", name);
    const uint64_t P = (uint64_t)fb->width * (uint64_t)fb->height;
    if (P + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "%s: P+1 overflows u32", name);
    if (fb->color_fmt != NOIT_RGBA_F16 && fb->color_fmt != NOIT_RGBA_F32)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: unknown color_fmt %d", name, fb->color_fmt);
    if (!fb->offsets) return noit_fail(ctx, NOIT_ERR_NULL, "%s: offsets is NULL", name);
    if (fb->num_fragments > 0 && (!fb->depth || !fb->rgba))
        return noit_fail(ctx, NOIT_ERR_NULL, "%s: depth/rgba is NULL with F > 0", name);
    if (!noit_aligned(fb->offsets, 4) || !noit_aligned(fb->depth, 16) ||
        !noit_aligned(fb->rgba, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT,
                         "%s: offsets need 4-byte, depth/rgba 16-byte alignment", name);
    return NOIT_OK;
}

extern "C" {

noit_status noit_create(noit_ctx** out)
{
    if (!out) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_create: out is NULL");
    *out = nullptr;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noit_cuda_check(nullptr, e, "cudaGetDevice");
    noit_ctx* c = new (std::nothrow) noit_ctx();
    if (!c) return noit_fail(nullptr, NOIT_ERR_CUDA, "noit_create: out of host memory");
    c->device = dev;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
        c->num_sms = sms;
    e = cudaMalloc(&c->d_counters, NOIT_COUNTER_WORDS * sizeof(uint32_t));
    if (e == cudaSuccess) e = cudaMemset(c->d_counters, 0, NOIT_COUNTER_WORDS * sizeof(uint32_t));
    if (e != cudaSuccess) {
        noit_cuda_check(nullptr, e, "noit_create scratch");
        delete c;
        return NOIT_ERR_CUDA;
    }
    snprintf(c->err, sizeof c->err, "no error");
    *out = c;
    return NOIT_OK;
}

void noit_destroy(noit_ctx* ctx)
{
    if (!ctx) return;
    cudaFree(ctx->d_counters);
    cudaFree(ctx->d_mlp);
    cudaFree(ctx->d_tile_lod);
    cudaFree(ctx->d_coarse_g[0]);
    cudaFree(ctx->d_coarse_g[1]);
    cudaFree(ctx->d_stage);
    if (ctx->h2d_stream) cudaStreamDestroy(ctx->h2d_stream);
    if (ctx->d2h_stream) cudaStreamDestroy(ctx->d2h_stream);
    for (cudaEvent_t e : ctx->host_ev)
        if (e) cudaEventDestroy(e);
    cudaFree(ctx->d_tile_depth);
    delete ctx;
}

// bf16 round-to-nearest-even of a finite fp32, widened back (A6).
static float round_bf16(float v)
{
    uint32_t u;
    memcpy(&u, &v, 4);
    if ((u & 0x7F800000u) != 0x7F800000u) u += 0x7FFFu + ((u >> 16) & 1u);
    u &= 0xFFFF0000u;
    memcpy(&v, &u, 4);
    return v;
}

noit_status noit_set_weights(noit_ctx* ctx, const float* host_w, int32_t count, int32_t precision)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_set_weights: ctx is NULL");
    if (!host_w) return noit_fail(ctx, NOIT_ERR_NULL, "noit_set_weights: host_w is NULL");
    if (count != NOIT_MLP_PARAMS)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_set_weights: count %d != 771 (P:97)", count);
    if (precision != NOIT_MLP_FP32 && precision != NOIT_MLP_BF16)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_set_weights: unknown precision %d", precision);
    float* dst = reinterpret_cast<float*>(&ctx->w);
    for (int i = 0; i < NOIT_MLP_PARAMS; ++i)
        dst[i] = precision == NOIT_MLP_BF16 ? round_bf16(host_w[i]) : host_w[i];
    memset(&ctx->wt, 0, sizeof ctx->wt);
    for (int o = 0; o < 32; ++o) {
        for (int i = 0; i < 5; ++i) ctx->wt.w1t[i][o] = ctx->w.w1[o][i];
        ctx->wt.b1[o] = ctx->w.b1[o];
    }
    for (int o = 0; o < 16; ++o) {
        for (int i = 0; i < 32; ++i) ctx->wt.w2t[i][o] = ctx->w.w2[o][i];
        ctx->wt.b2[o] = ctx->w.b2[o];
    }
    for (int o = 0; o < 3; ++o) {
        for (int i = 0; i < 16; ++i) ctx->wt.w3t[i][o] = ctx->w.w3[o][i];
        ctx->wt.b3[o] = ctx->w.b3[o];
    }
    // packed per-lane MMA fragments (layout: mlp_forward_mma in noit_internal.cuh)
    {
        float pk[NOIT_MMA_CHUNKS * 32 * 4];
        memset(pk, 0, sizeof pk);
        const MlpWeights& w = ctx->w;
        for (int lane = 0; lane < 32; ++lane) {
            const int g = lane >> 2, t = lane & 3;
            auto at = [&](int idx) -> float& { return pk[((idx >> 2) * 32 + lane) * 4 + (idx & 3)]; };
            for (int j = 0; j < 4; ++j) {
                at(2 * j) = w.w1[8 * j + g][t];
                at(2 * j + 1) = t == 0 ? w.w1[8 * j + g][4] : (t == 1 ? w.b1[8 * j + g] : 0.f);
            }
            for (int j = 0; j < 2; ++j) {
                for (int sidx = 0; sidx < 4; ++sidx) {
                    at(8 + 2 * (4 * j + sidx)) = w.w2[8 * j + g][8 * sidx + 2 * t];
                    at(8 + 2 * (4 * j + sidx) + 1) = w.w2[8 * j + g][8 * sidx + 2 * t + 1];
                }
                for (int h = 0; h < 2; ++h) {
                    at(24 + 4 * j + 2 * h) = w.b2[8 * j + 2 * t];
                    at(24 + 4 * j + 2 * h + 1) = w.b2[8 * j + 2 * t + 1];
                }
            }
            for (int sidx = 0; sidx < 2; ++sidx) {
                at(32 + 2 * sidx) = g < 3 ? w.w3[g][8 * sidx + 2 * t] : 0.f;
                at(32 + 2 * sidx + 1) = g < 3 ? w.w3[g][8 * sidx + 2 * t + 1] : 0.f;
            }
            for (int h = 0; h < 2; ++h) {
                at(36 + 2 * h) = 2 * t < 3 ? w.b3[2 * t] : 0.f;
                at(36 + 2 * h + 1) = 2 * t + 1 < 3 ? w.b3[2 * t + 1] : 0.f;
            }
        }
        if (!ctx->d_mlp) NOIT_CUDA(ctx, cudaMalloc(&ctx->d_mlp, sizeof pk));
        NOIT_CUDA(ctx, cudaMemcpy(ctx->d_mlp, pk, sizeof pk, cudaMemcpyHostToDevice));
    }
    ctx->precision = precision;
    ctx->has_weights = true;
    return NOIT_OK;
}

noit_status noit_get_weights(const noit_ctx* ctx, float* host_out, int32_t count)
{
    noit_ctx* c = const_cast<noit_ctx*>(ctx);
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_get_weights: ctx is NULL");
    if (!host_out) return noit_fail(c, NOIT_ERR_NULL, "noit_get_weights: host_out is NULL");
    if (count != NOIT_MLP_PARAMS) return noit_fail(c, NOIT_ERR_SIZE, "noit_get_weights: count != 771");
    if (!ctx->has_weights) return noit_fail(c, NOIT_ERR_NO_WEIGHTS, "noit_get_weights: no weights set");
    memcpy(host_out, &ctx->w, sizeof(MlpWeights));
    return NOIT_OK;
}

const char* noit_last_error(const noit_ctx* ctx) { return ctx ? ctx->err : g_err; }

uint64_t noit_launch_count(const noit_ctx* ctx) { return ctx ? ctx->launches : 0; }

noit_status noit_debug_bounds_violations(noit_ctx* ctx, uint32_t* host_count)
{
    if (!ctx || !host_count) return noit_fail(ctx, NOIT_ERR_NULL, "noit_debug_bounds_violations: NULL argument");
    NOIT_TRY(noit_check_device(ctx, "noit_debug_bounds_violations"));
    NOIT_CUDA(ctx, cudaDeviceSynchronize());
    NOIT_CUDA(ctx, cudaMemcpy(host_count, ctx->d_counters + NOIT_DEBUG_COUNTER, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    return NOIT_OK;
}

}  // extern "C"
