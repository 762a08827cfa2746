// noit_reproject.cu -- S8: depth-based temporal reprojection with a disocclusion test
// ("reprojecting pixels using the nearest available depth and the previous
// view-projection matrix"; O8, A21-A23), and its bilinear-filtered variant (NEXT-4, O8b, A28).
// The accept mask must be bit-exact, so the arithmetic is fp32 in ONE fixed order: every
// multiply-add is an explicit __fmaf_rn, everything else an explicit _rn intrinsic (never
// contracted by the compiler); the file is also compiled with -fmad=false.
#include "noit_internal.cuh"

struct ReprojArgs {
    int32_t W, H;
    float M[16];
    float thr;
    float inv_w, inv_h;            // 1.0f / W, 1.0f / H (IEEE fp32, formed once on the host)
    float bg[3];
    const float* prev_trans; const float* prev_depth; const float* cur_depth;
    float* out_trans; float* out_depth; float* out_final;
    uint8_t* accept; uint32_t* reject_list; uint32_t* reject_count;
};

template <bool kBilinear>
__global__ void __launch_bounds__(256)
reproject_kernel(const __grid_constant__ ReprojArgs A)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x, y = blockIdx.y;
    const bool inside = x < A.W;
    bool ok = false;
    uint32_t p = 0;
    if (inside) {
        p = (uint32_t)y * (uint32_t)A.W + (uint32_t)x;
        const float fW = (float)A.W, fH = (float)A.H;
        const float xn = __fmaf_rn(__fmul_rn(2.0f, __fadd_rn((float)x, 0.5f)), A.inv_w, -1.0f);
        const float yn = __fmaf_rn(__fmul_rn(2.0f, __fadd_rn((float)y, 0.5f)), A.inv_h, -1.0f);
        const float d = __ldcs(A.cur_depth + p);
        float c[4];
#pragma unroll
        for (int k = 0; k < 4; ++k)
            c[k] = __fmaf_rn(A.M[4 * k + 0], xn,
                             __fmaf_rn(A.M[4 * k + 1], yn, __fmaf_rn(A.M[4 * k + 2], d, A.M[4 * k + 3])));
        ok = c[3] > 0.0f;
        if (ok) {
            const float xp = __fdiv_rn(c[0], c[3]), yp = __fdiv_rn(c[1], c[3]);
            const float d_e = __fdiv_rn(c[2], c[3]);
            const float u = __fmul_rn(__fmul_rn(__fadd_rn(xp, 1.0f), 0.5f), fW);
            const float v = __fmul_rn(__fmul_rn(__fadd_rn(yp, 1.0f), 0.5f), fH);
            const float fx = floorf(u), fy = floorf(v);
            ok = (fx >= 0.0f) && (fx < fW) && (fy >= 0.0f) && (fy < fH);   // NaN rejects here
            if (ok) {
                const uint32_t q = (uint32_t)(int)fy * (uint32_t)A.W + (uint32_t)(int)fx;
                ok = fabsf(__fsub_rn(__ldg(A.prev_depth + q), d_e)) <= A.thr;
                if (ok) {
                    float4 t = __ldg(reinterpret_cast<const float4*>(A.prev_trans) + q);
                    if (kBilinear) {
                        // O8b / A28: 2x2 footprint around (u - 0.5, v - 0.5), used only if all four
                        // taps pass the disocclusion test (no blending across a depth edge)
                        const float ub = __fsub_rn(u, 0.5f), vb = __fsub_rn(v, 0.5f);
                        const float x0f = floorf(ub), y0f = floorf(vb);
                        const float wx = __fsub_rn(ub, x0f), wy = __fsub_rn(vb, y0f);
                        const int x0 = max((int)x0f, 0), x1 = min((int)x0f + 1, A.W - 1);
                        const int y0 = max((int)y0f, 0), y1 = min((int)y0f + 1, A.H - 1);
                        const uint32_t q00 = (uint32_t)y0 * (uint32_t)A.W + (uint32_t)x0,
                                       q01 = (uint32_t)y0 * (uint32_t)A.W + (uint32_t)x1,
                                       q10 = (uint32_t)y1 * (uint32_t)A.W + (uint32_t)x0,
                                       q11 = (uint32_t)y1 * (uint32_t)A.W + (uint32_t)x1;
                        const float e00 = __ldg(A.prev_depth + q00), e01 = __ldg(A.prev_depth + q01);
                        const float e10 = __ldg(A.prev_depth + q10), e11 = __ldg(A.prev_depth + q11);
                        const bool all4 = fabsf(__fsub_rn(e00, d_e)) <= A.thr && fabsf(__fsub_rn(e01, d_e)) <= A.thr &&
                                          fabsf(__fsub_rn(e10, d_e)) <= A.thr && fabsf(__fsub_rn(e11, d_e)) <= A.thr;
                        if (all4) {
                            const float4* T = reinterpret_cast<const float4*>(A.prev_trans);
                            const float4 t00 = __ldg(T + q00), t01 = __ldg(T + q01);
                            const float4 t10 = __ldg(T + q10), t11 = __ldg(T + q11);
                            auto lerp2 = [&](float a00, float a01, float a10, float a11) -> float {
                                const float top = __fmaf_rn(wx, __fsub_rn(a01, a00), a00);
                                const float bot = __fmaf_rn(wx, __fsub_rn(a11, a10), a10);
                                return __fmaf_rn(wy, __fsub_rn(bot, top), top);
                            };
                            t = make_float4(lerp2(t00.x, t01.x, t10.x, t11.x), lerp2(t00.y, t01.y, t10.y, t11.y),
                                            lerp2(t00.z, t01.z, t10.z, t11.z), lerp2(t00.w, t01.w, t10.w, t11.w));
                        }
                    }
                    __stcs(reinterpret_cast<float4*>(A.out_trans) + p, t);      // nearest: bit copy
                    if (A.out_depth) __stcs(A.out_depth + p, d_e);
                    if (A.out_final)
                        __stcs(reinterpret_cast<float4*>(A.out_final) + p,
                               make_float4(__fmaf_rn(t.w, A.bg[0], t.x), __fmaf_rn(t.w, A.bg[1], t.y),
                                           __fmaf_rn(t.w, A.bg[2], t.z), __fsub_rn(1.0f, t.w)));
                }
            }
        }
        if (A.accept) A.accept[p] = ok ? 1 : 0;
    }
    // rejected pixels -> list, one atomic per warp (list order is unspecified, O8)
    const bool rej = inside && !ok;
    const uint32_t m = __ballot_sync(0xffffffffu, rej);
    if (m) {
        const int lane = threadIdx.x & 31;
        uint32_t base = 0;
        if (lane == __ffs(m) - 1) base = atomicAdd(A.reject_count, (uint32_t)__popc(m));
        base = __shfl_sync(0xffffffffu, base, __ffs(m) - 1);
        if (rej && A.reject_list) A.reject_list[base + __popc(m & ((1u << lane) - 1))] = p;
    }
}

extern "C" noit_status noit_reproject(noit_ctx* ctx, const noit_reproject_desc* d, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_reproject: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_reproject"));
    if (!d) return noit_fail(ctx, NOIT_ERR_NULL, "noit_reproject: desc is NULL");
    if (!d->prev_trans || !d->prev_depth || !d->cur_depth || !d->out_trans || !d->reject_count)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_reproject: a required pointer is NULL");
    if (d->width <= 0 || d->height <= 0 || (uint64_t)d->width * (uint64_t)d->height + 1 > 0xFFFFFFFFull ||
        d->height > 65535)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_reproject: bad width/height");
    if (d->filter != NOIT_REPROJECT_NEAREST && d->filter != NOIT_REPROJECT_BILINEAR)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_reproject: unknown filter %d", d->filter);
    if (!noit_aligned(d->prev_trans, 16) || !noit_aligned(d->out_trans, 16) ||
        !noit_aligned(d->out_final, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_reproject: f32x4 images need 16-byte alignment");
    ReprojArgs A;
    A.W = d->width; A.H = d->height;
    memcpy(A.M, d->M, sizeof A.M);
    A.thr = d->depth_threshold;
    A.inv_w = 1.0f / (float)d->width;      // same correctly rounded fp32 quotient as O8's 1.0f/W
    A.inv_h = 1.0f / (float)d->height;
    memcpy(A.bg, d->background, sizeof A.bg);
    A.prev_trans = d->prev_trans; A.prev_depth = d->prev_depth; A.cur_depth = d->cur_depth;
    A.out_trans = d->out_trans; A.out_depth = d->out_depth; A.out_final = d->out_final;
    A.accept = d->accept; A.reject_list = d->reject_list; A.reject_count = d->reject_count;
    cudaStream_t st = (cudaStream_t)stream;
    NOIT_CUDA(ctx, cudaMemsetAsync(d->reject_count, 0, sizeof(uint32_t), st));
    const dim3 grid((d->width + 255) / 256, d->height);
    if (d->filter == NOIT_REPROJECT_BILINEAR) reproject_kernel<true><<<grid, 256, 0, st>>>(A);
    else reproject_kernel<false><<<grid, 256, 0, st>>>(A);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}
