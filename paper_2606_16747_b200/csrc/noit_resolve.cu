// noit_resolve.cu -- noit_resolve / noit_resolve_host: host-side checks and dispatch, and the S7
// pre-pass (coarse_g_kernel).  Every resolve (plain frame, S7 adaptive, S9 pixel list) runs in
// the staged kernel (noit_resolve_staged.cu).
#include <algorithm>

#include "noit_resolve_common.cuh"

noit_status noit_launch_resolve_staged(noit_ctx* ctx, const ResolveArgs& A, int color_fmt, int mode,
                                       cudaStream_t st);
noit_status noit_launch_resolve_dfaoit(noit_ctx* ctx, const ResolveArgs& A, int color_fmt,
                                       const MlpWeights10T& w10, cudaStream_t st);

// S7 pre-pass: G (10 values in 12 floats) of every coarse pixel whose leaf is resolved at that lod (self-contained
// O1-O2 on the coarse buffer, A19).  Coarse pixels of other leaves are never sampled: skipped.
// One launch covers both coarse levels: blocks [0, blocks1) the half-res buffer (lod 1), blocks
// [blocks1, blocks12) the quarter-res buffer (lod 2).  In the per-tile mode the blocks from
// blocks12 on write the lod summary of the staged kernel's 32-pixel tiles (one thread per tile):
// bit 0 = some pixel of the tile has lod > 0, bit 1 = every pixel does (pixels past the frame
// count as coarse), so the tile loop reads one byte instead of a level per lane and two votes.
struct CoarseLevel {
    int cw, ch;
    const uint32_t* offsets;
    const float* depth;
    const void* rgba;
    float* G;
};
constexpr int kPreBlock = 256;     // threads per block of the pre-pass
template <typename ColorT>
__global__ void __launch_bounds__(kPreBlock)
coarse_g_kernel(CoarseLevel lv1, CoarseLevel lv2, uint32_t blocks1, uint32_t blocks12, int full_w,
                const uint8_t* __restrict__ cell_level, uchar4 level_to_lod, uint8_t* __restrict__ tile_lod,
                uint32_t num_tiles, uint32_t P, const float* __restrict__ pass_scales)
{
    if (blockIdx.x >= blocks12) {                         // lod summary of tile t (per-tile mode)
        const uint32_t t = (blockIdx.x - blocks12) * blockDim.x + threadIdx.x;
        if (t >= num_tiles) return;
        const uint8_t l2l[4] = {level_to_lod.x, level_to_lod.y, level_to_lod.z, level_to_lod.w};
        const uint32_t W = (uint32_t)full_w, cw8 = (W + 7u) >> 3;
        uint32_t p = t * 32u;
        const uint32_t end = min(p + 32u, P);
        bool any = false, all = true;
        while (p < end) {                                 // one step per 8x8 cell the tile crosses
            const uint32_t y = p / W, x = p - y * W;
            const int lod = l2l[cell_level[(size_t)(y >> 3) * cw8 + (x >> 3)] & 3];
            any = any || lod > 0;
            all = all && lod > 0;
            p += min(8u - (x & 7u), W - x);
        }
        tile_lod[t] = (uint8_t)((any ? 1u : 0u) | ((any && all) ? 2u : 0u));
        return;
    }
    const bool second = blockIdx.x >= blocks1;
    const CoarseLevel lv = second ? lv2 : lv1;
    const int lod = second ? 2 : 1, r = 1 << lod;
    const uint32_t q = (blockIdx.x - (second ? blocks1 : 0u)) * blockDim.x + threadIdx.x;
    if (q >= (uint32_t)lv.cw * (uint32_t)lv.ch) return;
    if (pass_scales) {                                    // frame-global control (O7g, A27): a coarse
        const float s2 = __ldg(pass_scales + 1), s3 = __ldg(pass_scales + 2);   // buffer neither pass
        const int l2 = s2 > 0.70710678f ? 0 : (s2 > 0.35355339f ? 1 : 2);       // uses is not scanned
        const int l3 = s3 > 0.70710678f ? 0 : (s3 > 0.35355339f ? 1 : 2);
        if (l2 != lod && l3 != lod) return;
    }
    const int Y = q / lv.cw, X = q - Y * lv.cw;
    if (cell_level) {                                     // NULL: frame-global lod, every pixel
        const int level = cell_level[(size_t)((Y * r) >> 3) * ((full_w + 7) >> 3) + ((X * r) >> 3)] & 3;
        const uint8_t l2l[4] = {level_to_lod.x, level_to_lod.y, level_to_lod.z, level_to_lod.w};
        if (l2l[level] != lod) return;
    }
    const ColorT* __restrict__ rgba = static_cast<const ColorT*>(lv.rgba);
    const uint32_t b = __ldg(lv.offsets + q), e = __ldg(lv.offsets + q + 1);
    PixelState<false> s;
    s.init();
    for (uint32_t j = b; j < e; ++j) s.push(__ldg(lv.depth + j), load_rgba(rgba, j), j);
    float4* g = reinterpret_cast<float4*>(lv.G) + 3 * (size_t)q;
    g[0] = make_float4(s.c2.w * s.c2.x, s.c2.w * s.c2.y, s.c2.w * s.c2.z, s.c2.w);
    g[1] = make_float4(s.acc_r, s.acc_g, s.acc_b, s.a_tail);
    g[2] = make_float4(s.t_tail, (float)(e - b), 0.f, 0.f);
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
static noit_status check_desc(noit_ctx* ctx, const noit_resolve_desc* d, const char* who)
{
    if (!d) return noit_fail(ctx, NOIT_ERR_NULL, "%s: desc is NULL", who);
    NOIT_TRY(noit_check_fragbuf(ctx, &d->full, who));
    if (!ctx->has_weights) return noit_fail(ctx, NOIT_ERR_NO_WEIGHTS, "%s: no weights set", who);
    if (!d->out_trans && !d->out_final && !d->out_depth1)
        return noit_fail(ctx, NOIT_ERR_NULL, "%s: every output is NULL", who);
    if (!noit_aligned(d->out_trans, 16) || !noit_aligned(d->out_final, 16) ||
        !noit_aligned(d->out_depth1, 4))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: out_trans/out_final need 16-byte alignment", who);
    if (!noit_aligned(d->background_image, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: background_image needs 16-byte alignment", who);
    if ((d->pixel_list != nullptr) != (d->pixel_count != nullptr))
        return noit_fail(ctx, NOIT_ERR_NULL, "%s: pixel_list and pixel_count go together", who);
    if (d->pixel_list && d->cell_level)
        return noit_fail(ctx, NOIT_ERR_UNSUPPORTED, "%s: pixel_list with cell_level", who);
    if (d->pass_scales) {                                  // frame-global lod (O7g)
        if (d->cell_level || d->pixel_list)
            return noit_fail(ctx, NOIT_ERR_UNSUPPORTED, "%s: pass_scales with cell_level / pixel_list", who);
        if (!noit_aligned(d->pass_scales, 4))
            return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: pass_scales needs 4-byte alignment", who);
        for (int lod = 1; lod <= 2; ++lod) {
            const noit_fragbuf* cb = lod == 1 ? d->half : d->quarter;
            if (!cb) return noit_fail(ctx, NOIT_ERR_NULL, "%s: pass_scales needs half and quarter", who);
            NOIT_TRY(noit_check_fragbuf(ctx, cb, who));
            const int r = 1 << lod;
            if (cb->width != (d->full.width + r - 1) / r || cb->height != (d->full.height + r - 1) / r)
                return noit_fail(ctx, NOIT_ERR_SIZE, "%s: lod %d buffer is not ceil(W/%d) x ceil(H/%d)",
                                 who, lod, r, r);
            if (cb->color_fmt != d->full.color_fmt)
                return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: coarse buffers must share color_fmt", who);
        }
    }
    if (d->cell_level) {
        for (int l = 0; l < 4; ++l) {
            const int lod = d->level_to_lod[l];
            if (lod > 2) return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: level_to_lod[%d] > 2", who, l);
            const noit_fragbuf* cb = lod == 1 ? d->half : (lod == 2 ? d->quarter : nullptr);
            if (lod == 0) continue;
            if (!cb) return noit_fail(ctx, NOIT_ERR_NULL, "%s: lod %d buffer is NULL", who, lod);
            NOIT_TRY(noit_check_fragbuf(ctx, cb, who));
            const int r = 1 << lod;
            if (cb->width != (d->full.width + r - 1) / r || cb->height != (d->full.height + r - 1) / r)
                return noit_fail(ctx, NOIT_ERR_SIZE, "%s: lod %d buffer is not ceil(W/%d) x ceil(H/%d)",
                                 who, lod, r, r);
            if (cb->color_fmt != d->full.color_fmt)
                return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: coarse buffers must share color_fmt", who);
        }
    }
    return NOIT_OK;
}

static noit_status resolve_device(noit_ctx* ctx, const noit_resolve_desc* d, cudaStream_t st)
{
    ResolveArgs A;
    memset(&A, 0, sizeof A);
    A.W = d->full.width;
    A.H = d->full.height;
    A.P = (uint32_t)A.W * (uint32_t)A.H;
    A.F = d->full.num_fragments;
    A.offsets = d->full.offsets;
    A.depth = d->full.depth;
    A.rgba = d->full.rgba;
    memcpy(A.bg, d->background, sizeof A.bg);
    A.bg_image = d->background_image;
    A.out_trans = d->out_trans;
    A.out_final = d->out_final;
    A.out_depth1 = d->out_depth1;
    A.pixel_list = d->pixel_list;
    A.pixel_count = d->pixel_count;
    A.cell_level = d->cell_level;
    const int fmt = d->full.color_fmt;

    if (d->pixel_list)                                     // S9: staged kernel, list mode
        return noit_launch_resolve_staged(ctx, A, fmt, NOIT_RESOLVE_LIST, st);
    if (d->cell_level || d->pass_scales) {                 // S7 / frame-global lod
        A.pass_scales = d->pass_scales;
        memcpy(A.level_to_lod, d->level_to_lod, 4);
        const uchar4 l2l = make_uchar4(d->level_to_lod[0], d->level_to_lod[1], d->level_to_lod[2],
                                       d->level_to_lod[3]);
        CoarseLevel lv[2];
        memset(lv, 0, sizeof lv);
        uint32_t blocks[2] = {0, 0};
        for (int lod = 1; lod <= 2; ++lod) {
            bool used = d->pass_scales != nullptr;         // global: the lods are decided on the device
            for (int l = 0; l < 4; ++l) used |= d->level_to_lod[l] == lod;
            if (!used) continue;
            const noit_fragbuf* cb = lod == 1 ? d->half : d->quarter;
            const size_t cp = (size_t)cb->width * cb->height;
            if (ctx->coarse_g_cap[lod - 1] < cp) {
                if (ctx->d_coarse_g[lod - 1]) {
                    NOIT_CUDA(ctx, cudaStreamSynchronize(st));
                    NOIT_CUDA(ctx, cudaFree(ctx->d_coarse_g[lod - 1]));
                    ctx->d_coarse_g[lod - 1] = nullptr;
                    ctx->coarse_g_cap[lod - 1] = 0;
                }
                NOIT_CUDA(ctx, cudaMalloc(&ctx->d_coarse_g[lod - 1], cp * NOIT_G_STRIDE * sizeof(float)));
                ctx->coarse_g_cap[lod - 1] = cp;
            }
            A.coarse_g[lod - 1] = ctx->d_coarse_g[lod - 1];
            A.coarse_w[lod - 1] = cb->width;
            A.coarse_h[lod - 1] = cb->height;
            lv[lod - 1] = CoarseLevel{cb->width, cb->height, cb->offsets, cb->depth, cb->rgba,
                                      ctx->d_coarse_g[lod - 1]};
            blocks[lod - 1] = (uint32_t)((cp + kPreBlock - 1) / kPreBlock);
        }
        // per-tile mode with no level mapped to a coarse lod: the frame is a plain resolve
        if (d->cell_level && blocks[0] + blocks[1] == 0)
            return noit_launch_resolve_staged(ctx, A, fmt, NOIT_RESOLVE_ALL, st);
        const uint32_t num_tiles = (A.P + 31u) / 32u;
        uint32_t blocks_s = 0;
        if (d->cell_level) {
            if (ctx->tile_lod_cap < num_tiles) {
                if (ctx->d_tile_lod) {
                    NOIT_CUDA(ctx, cudaStreamSynchronize(st));
                    NOIT_CUDA(ctx, cudaFree(ctx->d_tile_lod));
                    ctx->d_tile_lod = nullptr;
                    ctx->tile_lod_cap = 0;
                }
                NOIT_CUDA(ctx, cudaMalloc(&ctx->d_tile_lod, num_tiles));
                ctx->tile_lod_cap = num_tiles;
            }
            A.tile_lod = ctx->d_tile_lod;
            blocks_s = (num_tiles + kPreBlock - 1u) / kPreBlock;
        }
        if (blocks[0] + blocks[1] + blocks_s) {
            const uint32_t b12 = blocks[0] + blocks[1];
            if (fmt == NOIT_RGBA_F16)
                coarse_g_kernel<__half><<<b12 + blocks_s, kPreBlock, 0, st>>>(
                    lv[0], lv[1], blocks[0], b12, A.W, d->cell_level, l2l, ctx->d_tile_lod, num_tiles, A.P, d->pass_scales);
            else
                coarse_g_kernel<float><<<b12 + blocks_s, kPreBlock, 0, st>>>(
                    lv[0], lv[1], blocks[0], b12, A.W, d->cell_level, l2l, ctx->d_tile_lod, num_tiles, A.P, d->pass_scales);
            ctx->launches += 1;
            NOIT_CUDA(ctx, cudaGetLastError());
        }
        return noit_launch_resolve_staged(ctx, A, fmt, d->pass_scales ? NOIT_RESOLVE_GLOBAL : NOIT_RESOLVE_ADAPTIVE, st);
    }
    return noit_launch_resolve_staged(ctx, A, fmt, NOIT_RESOLVE_ALL, st);
}

extern "C" {

noit_status noit_resolve(noit_ctx* ctx, const noit_resolve_desc* d, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_resolve: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_resolve"));
    NOIT_TRY(check_desc(ctx, d, "noit_resolve"));
    return resolve_device(ctx, d, (cudaStream_t)stream);
}

noit_status noit_resolve_host(noit_ctx* ctx, const noit_resolve_desc* h, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_resolve_host: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_resolve_host"));
    if (h && (h->cell_level || h->pixel_list || h->half || h->quarter || h->pass_scales ||
              h->background_image))
        return noit_fail(ctx, NOIT_ERR_UNSUPPORTED, "noit_resolve_host: plain resolve only");
    NOIT_TRY(check_desc(ctx, h, "noit_resolve_host"));
    cudaStream_t st = (cudaStream_t)stream;
    const size_t P = (size_t)h->full.width * h->full.height, F = h->full.num_fragments;
    const size_t cb = h->full.color_fmt == NOIT_RGBA_F16 ? 8 : 16;
    auto up = [](size_t v) { return (v + 255) & ~(size_t)255; };
    const size_t o_off = 0, o_depth = o_off + up(4 * (P + 1)), o_rgba = o_depth + up(4 * F);
    const size_t o_trans = o_rgba + up(cb * F), o_final = o_trans + up(16 * P);
    const size_t o_d1 = o_final + up(16 * P), total = o_d1 + up(4 * P);
    if (ctx->stage_cap < total) {
        if (ctx->d_stage) {
            NOIT_CUDA(ctx, cudaStreamSynchronize(st));
            NOIT_CUDA(ctx, cudaFree(ctx->d_stage));
            ctx->d_stage = nullptr;
            ctx->stage_cap = 0;
        }
        NOIT_CUDA(ctx, cudaMalloc(&ctx->d_stage, total));
        ctx->stage_cap = total;
    }
    char* base = static_cast<char*>(ctx->d_stage);
    // Bands of whole 32-pixel tiles, pipelined over three streams: band b+1 is copied in while band
    // b is resolved and band b-1 is copied out (the CSR lists of a pixel range are one contiguous
    // fragment range, so a band is three contiguous H2D copies).  The link is full duplex, so the
    // outputs travel while the inputs still arrive; the kernels (19 us per band at 1080p) hide
    // entirely.  Small frames go in one band.
    if (!ctx->h2d_stream) {
        NOIT_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->h2d_stream, cudaStreamNonBlocking));
        NOIT_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->d2h_stream, cudaStreamNonBlocking));
        for (cudaEvent_t& e : ctx->host_ev) NOIT_CUDA(ctx, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    const uint32_t* hoff = h->full.offsets;               // HOST memory
    const size_t in_bytes = 4 * (P + 1) + (4 + cb) * F;
    const size_t nb = std::min<size_t>(NOIT_HOST_BANDS, std::max<size_t>(1, in_bytes >> 24));
    const size_t band_px = (((P + nb - 1) / nb) + 31) & ~(size_t)31;
    cudaEvent_t* ev_h2d = ctx->host_ev;
    cudaEvent_t* ev_k = ctx->host_ev + NOIT_HOST_BANDS;
    cudaEvent_t ev_start = ctx->host_ev[2 * NOIT_HOST_BANDS], ev_done = ctx->host_ev[2 * NOIT_HOST_BANDS + 1];
    // every band boundary is checked BEFORE anything is enqueued: a malformed CSR leaves the
    // caller's buffers untouched
    for (size_t p0 = 0; p0 < P; p0 += band_px) {
        const size_t p1 = std::min(P, p0 + band_px);
        if (hoff[p1] < hoff[p0] || hoff[p1] > F || (p0 == 0 && hoff[0] != 0))
            return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_resolve_host: offsets are not a CSR of F fragments");
    }
    // From here on copies and kernels are in flight on three streams and target the caller's host
    // buffers: an error inside the loop must not return before they have drained.
    const noit_status rc = [&]() -> noit_status {
    // the staging area is reused between calls: the copies start after the caller's earlier work
    NOIT_CUDA(ctx, cudaEventRecord(ev_start, st));
    NOIT_CUDA(ctx, cudaStreamWaitEvent(ctx->h2d_stream, ev_start, 0));
    NOIT_CUDA(ctx, cudaStreamWaitEvent(ctx->d2h_stream, ev_start, 0));
    uint32_t* d_off = reinterpret_cast<uint32_t*>(base + o_off);
    float* d_depth = reinterpret_cast<float*>(base + o_depth);
    char* d_rgba = base + o_rgba;
    float* d_trans = h->out_trans ? reinterpret_cast<float*>(base + o_trans) : nullptr;
    float* d_final = h->out_final ? reinterpret_cast<float*>(base + o_final) : nullptr;
    float* d_d1 = h->out_depth1 ? reinterpret_cast<float*>(base + o_d1) : nullptr;
    size_t band = 0;
    for (size_t p0 = 0; p0 < P; p0 += band_px, ++band) {
        const size_t p1 = std::min(P, p0 + band_px), np = p1 - p0;
        const size_t f0 = hoff[p0], f1 = hoff[p1];
        NOIT_CUDA(ctx, cudaMemcpyAsync(d_off + p0, hoff + p0, 4 * (np + 1), cudaMemcpyHostToDevice, ctx->h2d_stream));
        if (f1 > f0) {
            NOIT_CUDA(ctx, cudaMemcpyAsync(d_depth + f0, h->full.depth + f0, 4 * (f1 - f0), cudaMemcpyHostToDevice,
                                           ctx->h2d_stream));
            NOIT_CUDA(ctx, cudaMemcpyAsync(d_rgba + cb * f0, static_cast<const char*>(h->full.rgba) + cb * f0,
                                           cb * (f1 - f0), cudaMemcpyHostToDevice, ctx->h2d_stream));
        }
        NOIT_CUDA(ctx, cudaEventRecord(ev_h2d[band], ctx->h2d_stream));
        NOIT_CUDA(ctx, cudaStreamWaitEvent(st, ev_h2d[band], 0));
        // the band as a frame of its own: np pixels whose lists index the whole fragment arrays
        // (a tile's copy is rounded to 4 fragments, so it may read up to 3 fragments of the
        // neighbouring bands -- staged, never scanned)
        ResolveArgs A;
        memset(&A, 0, sizeof A);
        A.W = h->full.width;
        A.H = h->full.height;
        A.P = (uint32_t)np;
        A.F = (uint32_t)F;
        A.offsets = d_off + p0;
        A.depth = d_depth;
        A.rgba = d_rgba;
        memcpy(A.bg, h->background, sizeof A.bg);
        A.out_trans = d_trans ? d_trans + 4 * p0 : nullptr;
        A.out_final = d_final ? d_final + 4 * p0 : nullptr;
        A.out_depth1 = d_d1 ? d_d1 + p0 : nullptr;
        NOIT_TRY(noit_launch_resolve_staged(ctx, A, h->full.color_fmt, NOIT_RESOLVE_ALL, st));
        NOIT_CUDA(ctx, cudaEventRecord(ev_k[band], st));
        NOIT_CUDA(ctx, cudaStreamWaitEvent(ctx->d2h_stream, ev_k[band], 0));
        if (h->out_trans)
            NOIT_CUDA(ctx, cudaMemcpyAsync(h->out_trans + 4 * p0, d_trans + 4 * p0, 16 * np, cudaMemcpyDeviceToHost,
                                           ctx->d2h_stream));
        if (h->out_final)
            NOIT_CUDA(ctx, cudaMemcpyAsync(h->out_final + 4 * p0, d_final + 4 * p0, 16 * np, cudaMemcpyDeviceToHost,
                                           ctx->d2h_stream));
        if (h->out_depth1)
            NOIT_CUDA(ctx, cudaMemcpyAsync(h->out_depth1 + p0, d_d1 + p0, 4 * np, cudaMemcpyDeviceToHost,
                                           ctx->d2h_stream));
    }
    NOIT_CUDA(ctx, cudaEventRecord(ev_done, ctx->d2h_stream));
    NOIT_CUDA(ctx, cudaStreamWaitEvent(st, ev_done, 0));
    NOIT_CUDA(ctx, cudaStreamSynchronize(st));
    return NOIT_OK;
    }();
    if (rc != NOIT_OK) {                                  // drain what was enqueued, keep the first error text
        cudaStreamSynchronize(ctx->h2d_stream);
        cudaStreamSynchronize(st);
        cudaStreamSynchronize(ctx->d2h_stream);
    }
    return rc;
}

}  // extern "C"

// NEXT-4 (O12): the DFAOIT resolve, the comparison variant of P:99-104
extern "C" noit_status noit_resolve_dfaoit(noit_ctx* ctx, const noit_fragbuf* fb, const float* host_w,
                                           int32_t count, const float* background, float* out_trans,
                                           float* out_final, float* out_depth1, float* features10,
                                           void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_resolve_dfaoit: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_resolve_dfaoit"));
    NOIT_TRY(noit_check_fragbuf(ctx, fb, "noit_resolve_dfaoit"));
    if (!host_w || !background) return noit_fail(ctx, NOIT_ERR_NULL, "noit_resolve_dfaoit: host_w / background is NULL");
    if (count != NOIT_DFAOIT_PARAMS)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_resolve_dfaoit: count %d != 931 (P:97-104)", count);
    if (!out_trans && !out_final && !out_depth1)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_resolve_dfaoit: every output is NULL");
    if (!noit_aligned(out_trans, 16) || !noit_aligned(out_final, 16) || !noit_aligned(features10, 8))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_resolve_dfaoit: out_trans/out_final need 16-byte, features10 8-byte alignment");
    // input-major, padded copy of W1[32][10], b1, W2[16][32], b2, W3[3][16], b3 for the FFMA2 network
    MlpWeights10T w;
    memset(&w, 0, sizeof w);
    const float* W1 = host_w, *b1 = W1 + 320, *W2 = b1 + 32, *b2 = W2 + 512, *W3 = b2 + 16, *b3 = W3 + 48;
    for (int o = 0; o < 32; ++o) {
        for (int i = 0; i < 10; ++i) w.w1t[i][o] = W1[o * 10 + i];
        w.b1[o] = b1[o];
    }
    for (int o = 0; o < 16; ++o) {
        for (int i = 0; i < 32; ++i) w.w2t[i][o] = W2[o * 32 + i];
        w.b2[o] = b2[o];
    }
    for (int o = 0; o < 3; ++o) {
        for (int i = 0; i < 16; ++i) w.w3t[i][o] = W3[o * 16 + i];
        w.b3[o] = b3[o];
    }
    ResolveArgs A;
    memset(&A, 0, sizeof A);
    A.W = fb->width;
    A.H = fb->height;
    A.P = (uint32_t)A.W * (uint32_t)A.H;
    A.F = fb->num_fragments;
    A.offsets = fb->offsets;
    A.depth = fb->depth;
    A.rgba = fb->rgba;
    memcpy(A.bg, background, sizeof A.bg);
    A.out_trans = out_trans;
    A.out_final = out_final;
    A.out_depth1 = out_depth1;
    A.features10 = features10;
    return noit_launch_resolve_dfaoit(ctx, A, fb->color_fmt, w, (cudaStream_t)stream);
}
