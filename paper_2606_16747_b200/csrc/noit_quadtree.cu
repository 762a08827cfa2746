// noit_quadtree.cu -- S6: colour-variance / corner-metric quadtree split (O6).
// One CTA of 256 threads per 64x64 base tile.  Each warp reduces eight 8x8 cells (64 pixels =
// 2 per lane, loaded as 128-byte row segments) to exact integer moments with redux.sync; the
// 16 + 4 + 1 ancestors are sums of children, so the whole tree costs one read of the tile.
#include "noit_internal.cuh"

// q = rint(255 * clamp(c, 0, 1)): single fp32 multiply, round-half-even (O6, A16).
__device__ __forceinline__ uint32_t quant8(float c)
{
    const float cl = fminf(fmaxf(c, 0.f), 1.f);
    return __float2uint_rn(__fmul_rn(255.0f, cl));
}

struct Moments { uint32_t n, s1[3], s2[3]; };

__device__ __forceinline__ bool variance_splits(const Moments& m, uint32_t thr)
{
    if (m.n == 0) return false;                       // wholly outside the image (A17)
    const uint64_t n = m.n;
    uint64_t lhs = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) lhs += n * (uint64_t)m.s2[c] - (uint64_t)m.s1[c] * (uint64_t)m.s1[c];
    return lhs > (uint64_t)thr * n * n;
}

// Corner metric D (A14): mean pairwise Euclidean RGB distance of the 4 corner pixels
// of the node's in-image rectangle; fp32, pairs (01,02,03,12,13,23), nothing contracted.
__device__ bool corner_splits(const float* __restrict__ image, int W, int H, int x0, int y0, int side,
                              float thr)
{
    const int x1 = min(x0 + side, W), y1 = min(y0 + side, H);
    if (x0 >= x1 || y0 >= y1) return false;
    const int xs[4] = {x0, x1 - 1, x0, x1 - 1}, ys[4] = {y0, y0, y1 - 1, y1 - 1};
    float4 c[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
        c[k] = __ldg(reinterpret_cast<const float4*>(image) + (size_t)ys[k] * W + xs[k]);
    const int pa[6] = {0, 0, 0, 1, 1, 2}, pb[6] = {1, 2, 3, 2, 3, 3};
    float sum = 0.f;
#pragma unroll
    for (int k = 0; k < 6; ++k) {
        const float dr = __fsub_rn(c[pa[k]].x, c[pb[k]].x), dg = __fsub_rn(c[pa[k]].y, c[pb[k]].y),
                    db = __fsub_rn(c[pa[k]].z, c[pb[k]].z);
        float s = __fmul_rn(dr, dr);
        s = __fadd_rn(s, __fmul_rn(dg, dg));
        s = __fadd_rn(s, __fmul_rn(db, db));
        const float root = __fsqrt_rn(s);
        sum = k == 0 ? root : __fadd_rn(sum, root);
    }
    return __fmul_rn(sum, 1.0f / 6.0f) > thr;
}

__global__ void __launch_bounds__(256)
quadtree_kernel(const float* __restrict__ image, int W, int H, int metric, uint32_t var_thr,
                float corner_thr, uint32_t* __restrict__ tile_mask, uint8_t* __restrict__ cell_level,
                uint32_t* __restrict__ hist)
{
    __shared__ Moments cell[64];          // 8x8 cells, index cy*8 + cx
    __shared__ uint8_t split[21];         // node split flags: 0 root, 1..4 level 1, 5..20 level 2
    __shared__ uint8_t lvl[64];
    const int Tx = (W + 63) >> 6;
    const int tile = blockIdx.x, tx = tile % Tx, ty = tile / Tx;
    const int X = tx << 6, Y = ty << 6;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (metric == NOIT_QT_VARIANCE) {
        // warp w owns cell row w (cells 8w..8w+7).  Lane l covers pixel (l&7, l>>3) and
        // (l&7, 4 + (l>>3)) of a cell: each load instruction reads four 128-byte row segments.
        float4 px[16];
        bool ok[16];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int x = X + i * 8 + (lane & 7), y = Y + warp * 8 + h * 4 + (lane >> 3);
                ok[i * 2 + h] = x < W && y < H;
                px[i * 2 + h] = ok[i * 2 + h]
                                    ? __ldcs(reinterpret_cast<const float4*>(image) + (size_t)y * W + x)
                                    : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            uint32_t n = 0, s1[3] = {0, 0, 0}, s2[3] = {0, 0, 0};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (!ok[i * 2 + h]) continue;
                const uint32_t q[3] = {quant8(px[i * 2 + h].x), quant8(px[i * 2 + h].y),
                                       quant8(px[i * 2 + h].z)};
                n += 1;
#pragma unroll
                for (int c = 0; c < 3; ++c) { s1[c] += q[c]; s2[c] += q[c] * q[c]; }
            }
            n = __reduce_add_sync(0xffffffffu, n);
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                s1[c] = __reduce_add_sync(0xffffffffu, s1[c]);
                s2[c] = __reduce_add_sync(0xffffffffu, s2[c]);
            }
            if (lane == 0) {
                Moments m;
                m.n = n;
#pragma unroll
                for (int c = 0; c < 3; ++c) { m.s1[c] = s1[c]; m.s2[c] = s2[c]; }
                cell[warp * 8 + i] = m;
            }
        }
        __syncthreads();
        if (threadIdx.x < 21) {
            // node -> rectangle of cells: level 0: 8x8 cells, level 1: 4x4, level 2: 2x2
            int cx0, cy0, span;
            const int t = threadIdx.x;
            if (t == 0) { cx0 = 0; cy0 = 0; span = 8; }
            else if (t < 5) { const int c = t - 1; cx0 = 4 * (c & 1); cy0 = 4 * (c >> 1); span = 4; }
            else {
                const int c = (t - 5) >> 2, g = (t - 5) & 3;
                cx0 = 4 * (c & 1) + 2 * (g & 1); cy0 = 4 * (c >> 1) + 2 * (g >> 1); span = 2;
            }
            Moments m = {0, {0, 0, 0}, {0, 0, 0}};
            for (int v = 0; v < span; ++v)
                for (int u = 0; u < span; ++u) {
                    const Moments& q = cell[(cy0 + v) * 8 + cx0 + u];
                    m.n += q.n;
                    for (int c = 0; c < 3; ++c) { m.s1[c] += q.s1[c]; m.s2[c] += q.s2[c]; }
                }
            split[t] = variance_splits(m, var_thr);
        }
    } else {
        if (threadIdx.x < 21) {
            int x0, y0, side;
            const int t = threadIdx.x;
            if (t == 0) { x0 = X; y0 = Y; side = 64; }
            else if (t < 5) { const int c = t - 1; x0 = X + 32 * (c & 1); y0 = Y + 32 * (c >> 1); side = 32; }
            else {
                const int c = (t - 5) >> 2, g = (t - 5) & 3;
                x0 = X + 32 * (c & 1) + 16 * (g & 1); y0 = Y + 32 * (c >> 1) + 16 * (g >> 1); side = 16;
            }
            split[t] = corner_splits(image, W, H, x0, y0, side, corner_thr);
        }
    }
    __syncthreads();
    // top-down: a node's flag counts only if its parent split.  Thread c (8x8 cell c).
    if (threadIdx.x < 64) {
        const int cx = threadIdx.x & 7, cy = threadIdx.x >> 3;
        const int c = (cx >> 2) + 2 * (cy >> 2), g = ((cx >> 1) & 1) + 2 * ((cy >> 1) & 1);
        int level = 0;
        if (split[0]) {
            level = 1;
            if (split[1 + c]) level = split[5 + 4 * c + g] ? 3 : 2;
        }
        lvl[threadIdx.x] = (uint8_t)level;
        const int gx = (X >> 3) + cx, gy = (Y >> 3) + cy;
        if (cell_level && gx < ((W + 7) >> 3) && gy < ((H + 7) >> 3))
            cell_level[(size_t)gy * ((W + 7) >> 3) + gx] = (uint8_t)level;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t mask = 0;
        if (split[0]) {
            mask |= 1u;
            for (int c = 0; c < 4; ++c)
                if (split[1 + c]) {
                    mask |= 1u << (1 + c);
                    for (int g = 0; g < 4; ++g)
                        if (split[5 + 4 * c + g]) mask |= 1u << (5 + 4 * c + g);
                }
        }
        if (tile_mask) tile_mask[tile] = mask;
        if (hist) {
            // leaves with >= 1 in-image pixel: a leaf at level l is counted at its first cell
            uint32_t h[4] = {0, 0, 0, 0};
            for (int level = 0; level < 4; ++level) {
                const int side = 64 >> level, per = 1 << level, cs = side >> 3;
                for (int ny = 0; ny < per; ++ny)
                    for (int nx = 0; nx < per; ++nx) {
                        if (X + nx * side >= W || Y + ny * side >= H) continue;
                        if (lvl[(ny * cs) * 8 + nx * cs] == level) h[level] += 1;
                    }
            }
            for (int level = 0; level < 4; ++level)
                if (h[level]) atomicAdd(hist + level, h[level]);
        }
    }
}

extern "C" noit_status noit_quadtree(noit_ctx* ctx, const float* image, int32_t width, int32_t height,
                                     const noit_qt_params* params, uint32_t* tile_mask,
                                     uint8_t* cell_level, uint32_t* level_hist, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree: ctx is NULL");
    if (!image || !params) return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree: image/params is NULL");
    if (!tile_mask && !cell_level && !level_hist)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree: every output is NULL");
    if (width <= 0 || height <= 0 || (uint64_t)width * (uint64_t)height + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree: bad width/height");
    if (params->metric != NOIT_QT_VARIANCE && params->metric != NOIT_QT_CORNER)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_quadtree: unknown metric %d", params->metric);
    if (!noit_aligned(image, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_quadtree: image needs 16-byte alignment");
    cudaStream_t st = (cudaStream_t)stream;
    if (level_hist) NOIT_CUDA(ctx, cudaMemsetAsync(level_hist, 0, 4 * sizeof(uint32_t), st));
    const int Tx = (width + 63) / 64, Ty = (height + 63) / 64;
    quadtree_kernel<<<Tx * Ty, 256, 0, st>>>(image, width, height, params->metric,
                                             params->var_threshold_q, params->corner_threshold,
                                             tile_mask, cell_level, level_hist);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}
