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

// depth of a base tile's subtree: 0 = not split .. 3 = a grandchild split
__device__ __forceinline__ int mask_depth(uint32_t mask)
{
    if (!(mask & 1u)) return 0;
    if (!(mask & 0x1Eu)) return 1;
    return (mask & 0x1FFFE0u) ? 3 : 2;
}


// NEXT-2 (O11, A26): the previous frame's masks make the split test a hysteresis: a node that
// was not split splits iff metric > split threshold, a node that was split merges iff
// metric < merge threshold.  prev_mask == nullptr: every node "was not split" (plain O6).
struct QtTemporal {
    const uint32_t* prev_mask;
    uint32_t var_merge;
    float corner_merge;
    int max_step;                  // levels a base tile may change per frame (0 = unlimited)
};

__device__ __forceinline__ bool variance_splits(const Moments& m, uint32_t split_thr, uint32_t merge_thr,
                                                bool was_split)
{
    if (m.n == 0) return false;                       // wholly outside the image (A17)
    const uint64_t n = m.n;
    uint64_t lhs = 0;
#pragma unroll
    for (int c = 0; c < 3; ++c) lhs += n * (uint64_t)m.s2[c] - (uint64_t)m.s1[c] * (uint64_t)m.s1[c];
    return was_split ? !(lhs < (uint64_t)merge_thr * n * n) : lhs > (uint64_t)split_thr * n * n;
}

// Corner metric D (A14): mean pairwise Euclidean RGB distance of the 4 corner pixels
// of the node's in-image rectangle; fp32, pairs (01,02,03,12,13,23), nothing contracted.
__device__ bool corner_splits(const float* __restrict__ image, int W, int H, int x0, int y0, int side,
                              float split_thr, float merge_thr, bool was_split)
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
    const float D = __fmul_rn(sum, 1.0f / 6.0f);
    return was_split ? !(D < merge_thr) : D > split_thr;
}

// One warp: leaf level of the tile's 64 cells (2 per lane) from its mask, and the tile's
// contribution to the histogram of leaves that hold >= 1 in-image pixel (a leaf at level l is
// the node whose first cell has level l).  Shared by noit_quadtree and noit_quadtree_balance.
template <int kCellShift>                               // cell side = 1 << kCellShift pixels (8 or 2)
__device__ __forceinline__ void emit_levels_and_hist(uint32_t mask, int X, int Y, int W, int H, int lane,
                                                     uint8_t* __restrict__ cell_level,
                                                     uint32_t* __restrict__ hist)
{
    auto level_of_cell = [&](int cx, int cy) -> int {
        const int c = (cx >> 2) + 2 * (cy >> 2), g = ((cx >> 1) & 1) + 2 * ((cy >> 1) & 1);
        if (!(mask & 1u)) return 0;
        if (!((mask >> (1 + c)) & 1u)) return 1;
        return ((mask >> (5 + 4 * c + g)) & 1u) ? 3 : 2;
    };
    constexpr int kCell = 1 << kCellShift;
    const int cells_w = (W + kCell - 1) >> kCellShift, cells_h = (H + kCell - 1) >> kCellShift;
    uint32_t h3 = 0;
#pragma unroll
    for (int k = 0; k < 2; ++k) {                        // 64 cells, 2 per lane
        const int idx = lane + 32 * k, cx = idx & 7, cy = idx >> 3;
        const int level = level_of_cell(cx, cy);
        const int gx = (X >> kCellShift) + cx, gy = (Y >> kCellShift) + cy;
        const bool in_image = gx < cells_w && gy < cells_h;
        if (cell_level && in_image) cell_level[(size_t)gy * cells_w + gx] = (uint8_t)level;
        h3 += __popc(__ballot_sync(0xffffffffu, in_image && level == 3));
    }
    if (!hist) return;
    bool leaf = false;
    int lv = 0;
    if (lane < 21) {                                     // lane t = node t (mask bit numbering)
        int cx = 0, cy = 0;
        if (lane >= 5) {
            const int c = (lane - 5) >> 2, g = (lane - 5) & 3;
            cx = 4 * (c & 1) + 2 * (g & 1); cy = 4 * (c >> 1) + 2 * (g >> 1); lv = 2;
        } else if (lane >= 1) {
            cx = 4 * ((lane - 1) & 1); cy = 4 * ((lane - 1) >> 1); lv = 1;
        }
        leaf = X + kCell * cx < W && Y + kCell * cy < H && level_of_cell(cx, cy) == lv;
    }
    const uint32_t Lf = __ballot_sync(0xffffffffu, leaf);
    if (lane == 0) {
        const uint32_t h0 = Lf & 1u, h1 = __popc(Lf & 0x1Eu), h2 = __popc(Lf & 0x1FFFE0u);
        if (h0) atomicAdd(hist + 0, h0);
        if (h1) atomicAdd(hist + 1, h1);
        if (h2) atomicAdd(hist + 2, h2);
        if (h3) atomicAdd(hist + 3, h3);
    }
}

// 4 CTAs per SM (<= 64 registers): the 510 tiles of a 1080p frame are ONE wave on 148 SMs (with 3
// CTAs per SM a second wave of 66 CTAs doubled the kernel's time)
__global__ void __launch_bounds__(256, 4)
quadtree_kernel(const float* __restrict__ image, int W, int H, int metric, uint32_t var_thr,
                float corner_thr, QtTemporal tq, uint32_t* __restrict__ tile_mask,
                uint8_t* __restrict__ cell_level, uint32_t* __restrict__ hist_out,
                uint32_t* __restrict__ hist_acc, uint32_t* __restrict__ ticket)
{
    __shared__ Moments cell[64];          // 8x8 cells, index cy*8 + cx
    __shared__ Moments node2[16];         // level-2 nodes (16x16 pixels), index 4c + g
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
            // n <= 64 and S1_c <= 64 * 255 fit 16-bit fields: 5 warp reductions per cell, not 7
            const uint32_t pa = __reduce_add_sync(0xffffffffu, s1[0] | (s1[1] << 16));
            const uint32_t pb = __reduce_add_sync(0xffffffffu, s1[2] | (n << 16));
#pragma unroll
            for (int c = 0; c < 3; ++c) s2[c] = __reduce_add_sync(0xffffffffu, s2[c]);
            if (lane == 0) {
                Moments m;
                m.n = pb >> 16;
                m.s1[0] = pa & 0xffffu; m.s1[1] = pa >> 16; m.s1[2] = pb & 0xffffu;
#pragma unroll
                for (int c = 0; c < 3; ++c) m.s2[c] = s2[c];
                cell[warp * 8 + i] = m;
            }
        }
    }
    __syncthreads();
    if (warp != 0) return;
    // ---- warp 0: node statistics bottom-up, split tests, mask, cell levels, histogram.
    // Lane t < 21 owns node t: 0 root, 1..4 level 1 (c = t-1), 5..20 level 2 (c = (t-5)>>2,
    // g = (t-5)&3) -- the same numbering as the mask bits.
    bool flag = false;
    const uint32_t prev = tq.prev_mask ? tq.prev_mask[tile] : 0u;
    const bool was_split = lane < 21 && ((prev >> lane) & 1u);   // lane t = node t = mask bit t
    if (metric == NOIT_QT_VARIANCE) {
        Moments m = {0, {0, 0, 0}, {0, 0, 0}};
        if (lane >= 5 && lane < 21) {                    // level 2: 2x2 cells
            const int c = (lane - 5) >> 2, g = (lane - 5) & 3;
            const int cx0 = 4 * (c & 1) + 2 * (g & 1), cy0 = 4 * (c >> 1) + 2 * (g >> 1);
#pragma unroll
            for (int v = 0; v < 2; ++v)
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    const Moments& q = cell[(cy0 + v) * 8 + cx0 + u];
                    m.n += q.n;
#pragma unroll
                    for (int k = 0; k < 3; ++k) { m.s1[k] += q.s1[k]; m.s2[k] += q.s2[k]; }
                }
            node2[lane - 5] = m;
        }
        __syncwarp();
        if (lane >= 1 && lane < 5) {                     // level 1: its 4 level-2 children
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                const Moments& q = node2[4 * (lane - 1) + g];
                m.n += q.n;
#pragma unroll
                for (int k = 0; k < 3; ++k) { m.s1[k] += q.s1[k]; m.s2[k] += q.s2[k]; }
            }
        }
        if (lane == 0) {                                 // root: all 16 level-2 nodes
            for (int g = 0; g < 16; ++g) {
                const Moments& q = node2[g];
                m.n += q.n;
#pragma unroll
                for (int k = 0; k < 3; ++k) { m.s1[k] += q.s1[k]; m.s2[k] += q.s2[k]; }
            }
        }
        flag = lane < 21 && variance_splits(m, var_thr, tq.var_merge, was_split);
    } else if (lane < 21) {
        int x0 = X, y0 = Y, side = 64;
        if (lane >= 5) {
            const int c = (lane - 5) >> 2, g = (lane - 5) & 3;
            x0 = X + 32 * (c & 1) + 16 * (g & 1); y0 = Y + 32 * (c >> 1) + 16 * (g >> 1); side = 16;
        } else if (lane >= 1) {
            const int c = lane - 1;
            x0 = X + 32 * (c & 1); y0 = Y + 32 * (c >> 1); side = 32;
        }
        flag = corner_splits(image, W, H, x0, y0, side, corner_thr, tq.corner_merge, was_split);
    }
    // top-down: a node's flag counts only if its parent split
    const uint32_t F = __ballot_sync(0xffffffffu, flag);
    uint32_t mask = 0;
    if (F & 1u) {
        mask = 1u;
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if ((F >> (1 + c)) & 1u) mask |= (1u << (1 + c)) | (F & (0xFu << (5 + 4 * c)));
    }
    if (tq.prev_mask && tq.max_step > 0) {               // at most max_step levels per frame
        const int pd = mask_depth(prev), d = mask_depth(mask);
        if (d > pd + tq.max_step) {                      // truncate below depth pd + max_step
            const int lim = pd + tq.max_step;
            mask &= lim == 0 ? 0u : (lim == 1 ? 0x1u : (lim == 2 ? 0x1Fu : 0x1FFFFFu));
        } else if (d < pd - tq.max_step) {               // refine uniformly to depth pd - max_step
            const int lim = pd - tq.max_step;
            mask |= (lim >= 1 ? 1u : 0u) | (lim >= 2 ? 0x1Eu : 0u) | (lim >= 3 ? 0x1FFFE0u : 0u);
        }
    }
    if (tile_mask && lane == 0) tile_mask[tile] = mask;
    emit_levels_and_hist<3>(mask, X, Y, W, H, lane, cell_level, hist_out ? hist_acc : nullptr);
    // the histogram is accumulated in context counters and published by the last tile (atomic
    // ticket), which also re-arms them: the caller's level_hist needs no memset before the launch
    if (!hist_out) return;
    __syncwarp();
    if (lane == 0) {
        __threadfence();
        if (atomicAdd(ticket, 1u) == gridDim.x - 1) {
            __threadfence();
            for (int l = 0; l < 4; ++l) {
                hist_out[l] = __ldcg(hist_acc + l);
                hist_acc[l] = 0u;
            }
            *ticket = 0u;
        }
    }
}

static noit_status quadtree_launch(noit_ctx* ctx, const char* who, const float* image, int32_t width,
                                   int32_t height, int32_t metric, uint32_t var_thr, float corner_thr,
                                   QtTemporal tq, uint32_t* tile_mask, uint8_t* cell_level,
                                   uint32_t* level_hist, void* stream)
{
    if (!tile_mask && !cell_level && !level_hist)
        return noit_fail(ctx, NOIT_ERR_NULL, "%s: every output is NULL", who);
    if (width <= 0 || height <= 0 || (uint64_t)width * (uint64_t)height + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "%s: bad width/height", who);
    if (metric != NOIT_QT_VARIANCE && metric != NOIT_QT_CORNER)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: unknown metric %d", who, metric);
    if (!noit_aligned(image, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "%s: image needs 16-byte alignment", who);
    cudaStream_t st = (cudaStream_t)stream;
    const int Tx = (width + 63) / 64, Ty = (height + 63) / 64;
    quadtree_kernel<<<Tx * Ty, 256, 0, st>>>(image, width, height, metric, var_thr, corner_thr, tq,
                                             tile_mask, cell_level, level_hist, ctx->d_counters + 8,
                                             ctx->d_counters + 12);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

extern "C" noit_status noit_quadtree_temporal(noit_ctx* ctx, const float* image, int32_t width,
                                              int32_t height, const noit_qt_temporal_params* params,
                                              const uint32_t* prev_tile_mask, uint32_t* tile_mask,
                                              uint8_t* cell_level, uint32_t* level_hist, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree_temporal: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_quadtree_temporal"));
    if (!image || !params)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree_temporal: image/params is NULL");
    if (params->max_level_step < 0 || params->max_level_step > 3)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree_temporal: max_level_step must be in [0, 3]");
    // either order of the two thresholds is a well-defined rule (merge <= split: a band in which a
    // node keeps its state, A26; merge > split: P:61's sentence read literally, a band in which a
    // node alternates) -- both are callable
    if (prev_tile_mask && prev_tile_mask == tile_mask)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_quadtree_temporal: prev_tile_mask aliases tile_mask");
    QtTemporal tq = {prev_tile_mask, params->var_merge_q, params->corner_merge, params->max_level_step};
    return quadtree_launch(ctx, "noit_quadtree_temporal", image, width, height, params->metric,
                           params->var_split_q, params->corner_split, tq, tile_mask, cell_level,
                           level_hist, stream);
}

extern "C" noit_status noit_quadtree(noit_ctx* ctx, const float* image, int32_t width, int32_t height,
                                     const noit_qt_params* params, uint32_t* tile_mask,
                                     uint8_t* cell_level, uint32_t* level_hist, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_quadtree"));
    if (!image || !params) return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree: image/params is NULL");
    QtTemporal tq = {nullptr, 0u, 0.f, 0};
    return quadtree_launch(ctx, "noit_quadtree", image, width, height, params->metric,
                           params->var_threshold_q, params->corner_threshold, tq, tile_mask, cell_level,
                           level_hist, stream);
}

// ------------------------------------------------------------------------------------------
// NEXT-1: quadtree consistency + demand index (O10, reading A25)
// ------------------------------------------------------------------------------------------
// One warp per base tile.  k Jacobi steps of L <- max(L, max over edge neighbours of L - 1)
// equal the max-plus convolution of the initial depths with the Manhattan diamond of radius k
// (induction on k), so each tile is finished in one pass over its diamond -- no ping-pong
// buffers, no grid synchronisation.  A tile that rises to depth L is refined uniformly to L.
// The masks are balanced "in place" for the caller, but no tile may see a neighbour's balanced
// mask: every warp reads the ORIGINAL masks (depth of a subtree = three bit tests), writes its
// balanced mask to a scratch array, and the last block to finish (atomic ticket) copies the
// scratch over tile_mask -- one launch, no depth pre-pass, no grid synchronisation.  The leaf
// histogram is accumulated in context counters (re-armed by the last block), so the caller's
// level_hist needs no memset either.  The last block also turns the histogram into
// w = sum l N_l / sum N_l and s_p = clamp(2^(w - delta_p), 0.25, 1) (Eq. 2).
__global__ void __launch_bounds__(128)
balance_kernel(int W, int H, int Tx, int Ty, int k, float delta2, float delta3,
               uint32_t* __restrict__ tile_mask, uint32_t* __restrict__ mask_tmp,
               uint8_t* __restrict__ tile_level, uint8_t* __restrict__ cell_level,
               uint32_t* __restrict__ hist_out, float* __restrict__ scales, uint32_t* __restrict__ ticket,
               uint32_t* __restrict__ hist_acc)
{
    const int lane = threadIdx.x & 31;
    const int n = Tx * Ty;
    const int tile = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    __shared__ uint32_t block_hist[4];                   // one set of global atomics per block
    if (threadIdx.x < 4) block_hist[threadIdx.x] = 0u;
    __syncthreads();
    if (tile < n) {
        const int tx = tile % Tx, ty = tile / Tx;
        // the diamond has 2k(k+1)+1 tiles; lanes stride over its bounding square, one independent
        // load per lane and step (k = 2: 13 of 25 cells, a single step)
        int best = 0;
        const int side = 2 * k + 1;
        for (int i = lane; i < side * side; i += 32) {
            const int dy = i / side - k, dx = i - (dy + k) * side - k;
            const int dist = abs(dx) + abs(dy), x = tx + dx, y = ty + dy;
            if (dist > k || x < 0 || x >= Tx || y < 0 || y >= Ty) continue;
            best = max(best, mask_depth(__ldcg(tile_mask + y * Tx + x)) - dist);
        }
        best = __reduce_max_sync(0xffffffffu, best);
        uint32_t mask = __ldcg(tile_mask + tile);
        if (best >= 1) mask |= 1u;                       // every node above depth `best` splits
        if (best >= 2) mask |= 0x1Eu;
        if (best >= 3) mask |= 0x1FFFE0u;
        __syncwarp();
        if (lane == 0) {
            mask_tmp[tile] = mask;
            if (tile_level) tile_level[tile] = (uint8_t)best;
        }
        emit_levels_and_hist<3>(mask, tx << 6, ty << 6, W, H, lane, cell_level, block_hist);
    }
    // last block: publish the balanced masks, the histogram, the demand index and Eq. 2
    __shared__ bool last;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int l = 0; l < 4; ++l)
            if (block_hist[l]) atomicAdd(hist_acc + l, block_hist[l]);
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    for (int i = threadIdx.x; i < n; i += blockDim.x) tile_mask[i] = __ldcg(mask_tmp + i);
    if (threadIdx.x == 0) {
        uint32_t nl[4];
        for (int l = 0; l < 4; ++l) {
            nl[l] = __ldcg(hist_acc + l);
            hist_acc[l] = 0u;                            // re-arm for the next call
            if (hist_out) hist_out[l] = nl[l];
        }
        if (scales) {
            const float den = (float)(nl[0] + nl[1] + nl[2] + nl[3]);
            const float w = den > 0.f ? __fdiv_rn((float)(nl[1] + 2u * nl[2] + 3u * nl[3]), den) : 0.f;
            scales[0] = w;
            scales[1] = fminf(fmaxf(exp2f(w - delta2), 0.25f), 1.0f);
            scales[2] = fminf(fmaxf(exp2f(w - delta3), 0.25f), 1.0f);
        }
        *ticket = 0u;
    }
}

extern "C" noit_status noit_quadtree_balance(noit_ctx* ctx, int32_t width, int32_t height,
                                             int32_t iterations, float delta2, float delta3,
                                             uint32_t* tile_mask, uint8_t* tile_level,
                                             uint8_t* cell_level, uint32_t* level_hist, float* scales,
                                             void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree_balance: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_quadtree_balance"));
    if (!tile_mask) return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree_balance: tile_mask is NULL");
    if (scales && !level_hist)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree_balance: scales needs level_hist");
    if (width <= 0 || height <= 0 || (uint64_t)width * (uint64_t)height + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree_balance: bad width/height");
    if (iterations < 0 || iterations > 16)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree_balance: iterations must be in [0, 16]");
    cudaStream_t st = (cudaStream_t)stream;
    const int Tx = (width + 63) / 64, Ty = (height + 63) / 64, n = Tx * Ty;
    if (ctx->tile_depth_cap < (size_t)n) {
        if (ctx->d_tile_depth) {
            NOIT_CUDA(ctx, cudaStreamSynchronize(st));
            NOIT_CUDA(ctx, cudaFree(ctx->d_tile_depth));
            ctx->d_tile_depth = nullptr;
            ctx->tile_depth_cap = 0;
        }
        NOIT_CUDA(ctx, cudaMalloc(&ctx->d_tile_depth, (size_t)n * sizeof(uint32_t)));
        ctx->tile_depth_cap = (size_t)n;
    }
    balance_kernel<<<(n + 3) / 4, 128, 0, st>>>(width, height, Tx, Ty, iterations, delta2, delta3, tile_mask,
                                                ctx->d_tile_depth, tile_level, cell_level, level_hist, scales,
                                                ctx->d_counters + 2, ctx->d_counters + 4);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

// ------------------------------------------------------------------------------------------
// NEXT-3: the paper's own tile geometry: 16x16 base tiles, four levels down to 2x2
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ Moments moments_xor_add(const Moments& m, int lane_mask)
{
    Moments r;
    r.n = m.n + __shfl_xor_sync(0xffffffffu, m.n, lane_mask);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        r.s1[k] = m.s1[k] + __shfl_xor_sync(0xffffffffu, m.s1[k], lane_mask);
        r.s2[k] = m.s2[k] + __shfl_xor_sync(0xffffffffu, m.s2[k], lane_mask);
    }
    return r;
}

// One WARP per 16x16 tile (a tile is 4 KB: a CTA per tile would be all latency).  The tile's 64
// cells are 2x2 pixels; lane l holds cells (cx, cy) = (l & 7, l >> 3) and (cx, cy + 4), so the
// sums of a level-2 node (2x2 cells) are a butterfly over lane bits 0 and 3, of a level-1 node
// additionally over bits 1 and 4, of the root over bit 2 plus the lane's two halves.  Every lane
// then knows the split flag of each node it belongs to; lane t < 21 picks node t's flag from the
// ballot of a representative lane, and the mask is assembled exactly as in quadtree_kernel.
__global__ void __launch_bounds__(128)
quadtree16_kernel(const float* __restrict__ image, int W, int H, int metric, uint32_t var_thr,
                  float corner_thr, uint32_t* __restrict__ tile_mask, uint8_t* __restrict__ cell_level,
                  uint32_t* __restrict__ hist)
{
    const int Tx = (W + 15) >> 4, Ty = (H + 15) >> 4;
    const int tile = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (tile >= Tx * Ty) return;
    const int tx = tile % Tx, ty = tile / Tx, X = tx << 4, Y = ty << 4;
    bool flag = false;
    if (metric == NOIT_QT_VARIANCE) {
        Moments half[2];
#pragma unroll
        for (int hb = 0; hb < 2; ++hb) {
            Moments m = {0, {0, 0, 0}, {0, 0, 0}};
            const int cx = lane & 7, cy = (lane >> 3) + 4 * hb;
#pragma unroll
            for (int v = 0; v < 2; ++v) {
                const int y = Y + 2 * cy + v, x = X + 2 * cx;
                if (y >= H) continue;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    if (x + u >= W) continue;
                    const float4 px = __ldcs(reinterpret_cast<const float4*>(image) + (size_t)y * W + x + u);
                    const uint32_t q[3] = {quant8(px.x), quant8(px.y), quant8(px.z)};
                    m.n += 1;
#pragma unroll
                    for (int k = 0; k < 3; ++k) { m.s1[k] += q[k]; m.s2[k] += q[k] * q[k]; }
                }
            }
            half[hb] = m;
        }
        Moments n2[2], n1[2];
#pragma unroll
        for (int hb = 0; hb < 2; ++hb) {
            n2[hb] = moments_xor_add(moments_xor_add(half[hb], 1), 8);    // 2x2 cells
            n1[hb] = moments_xor_add(moments_xor_add(n2[hb], 2), 16);     // 4x4 cells
        }
        Moments root = n1[0];
        root.n += n1[1].n;
#pragma unroll
        for (int k = 0; k < 3; ++k) { root.s1[k] += n1[1].s1[k]; root.s2[k] += n1[1].s2[k]; }
        root = moments_xor_add(root, 4);
        const uint32_t F0 = __ballot_sync(0xffffffffu, variance_splits(root, var_thr, 0u, false));
        const uint32_t F1[2] = {__ballot_sync(0xffffffffu, variance_splits(n1[0], var_thr, 0u, false)),
                                __ballot_sync(0xffffffffu, variance_splits(n1[1], var_thr, 0u, false))};
        const uint32_t F2[2] = {__ballot_sync(0xffffffffu, variance_splits(n2[0], var_thr, 0u, false)),
                                __ballot_sync(0xffffffffu, variance_splits(n2[1], var_thr, 0u, false))};
        if (lane == 0) {
            flag = F0 & 1u;
        } else if (lane < 5) {                           // child c: cells (4(c&1).., 4(c>>1)..)
            const int c = lane - 1;
            flag = (F1[c >> 1] >> (4 * (c & 1))) & 1u;
        } else if (lane < 21) {                          // grandchild g of child c
            const int c = (lane - 5) >> 2, g = (lane - 5) & 3;
            flag = (F2[c >> 1] >> (16 * (g >> 1) + 4 * (c & 1) + 2 * (g & 1))) & 1u;
        }
    } else if (lane < 21) {
        int x0 = X, y0 = Y, side = 16;
        if (lane >= 5) {
            const int c = (lane - 5) >> 2, g = (lane - 5) & 3;
            x0 = X + 8 * (c & 1) + 4 * (g & 1); y0 = Y + 8 * (c >> 1) + 4 * (g >> 1); side = 4;
        } else if (lane >= 1) {
            const int c = lane - 1;
            x0 = X + 8 * (c & 1); y0 = Y + 8 * (c >> 1); side = 8;
        }
        flag = corner_splits(image, W, H, x0, y0, side, corner_thr, 0.f, false);
    }
    const uint32_t F = __ballot_sync(0xffffffffu, flag);    // top-down gating
    uint32_t mask = 0;
    if (F & 1u) {
        mask = 1u;
#pragma unroll
        for (int c = 0; c < 4; ++c)
            if ((F >> (1 + c)) & 1u) mask |= (1u << (1 + c)) | (F & (0xFu << (5 + 4 * c)));
    }
    if (tile_mask && lane == 0) tile_mask[tile] = mask;
    emit_levels_and_hist<1>(mask, X, Y, W, H, lane, cell_level, hist);
}

extern "C" noit_status noit_quadtree16(noit_ctx* ctx, const float* image, int32_t width, int32_t height,
                                       const noit_qt_params* params, uint32_t* tile_mask,
                                       uint8_t* cell_level, uint32_t* level_hist, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree16: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_quadtree16"));
    if (!image || !params) return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree16: image/params is NULL");
    if (!tile_mask && !cell_level && !level_hist)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree16: every output is NULL");
    if (width <= 0 || height <= 0 || (uint64_t)width * (uint64_t)height + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree16: bad width/height");
    if (params->metric != NOIT_QT_VARIANCE && params->metric != NOIT_QT_CORNER)
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_quadtree16: unknown metric %d", params->metric);
    if (!noit_aligned(image, 16))
        return noit_fail(ctx, NOIT_ERR_FORMAT, "noit_quadtree16: image needs 16-byte alignment");
    cudaStream_t st = (cudaStream_t)stream;
    if (level_hist) NOIT_CUDA(ctx, cudaMemsetAsync(level_hist, 0, 4 * sizeof(uint32_t), st));
    const int tiles = ((width + 15) / 16) * ((height + 15) / 16);
    quadtree16_kernel<<<(tiles + 3) / 4, 128, 0, st>>>(image, width, height, params->metric,
                                                       params->var_threshold_q, params->corner_threshold,
                                                       tile_mask, cell_level, level_hist);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

// ------------------------------------------------------------------------------------------
// noit_quadtree_balance_static: the same balance pass for callers that cannot allocate
// ------------------------------------------------------------------------------------------
// noit_quadtree_balance keeps the balanced masks in context scratch that it cudaMallocs on first
// use / growth.  Code under CUDA-graph capture, tight serving loops and harnesses that forbid
// allocation get this variant: the SAME kernel (balance_kernel), with its scratch -- the balanced
// masks before they are published, the finish ticket and the histogram accumulators -- in a
// file-scope device array of fixed size.  Every GPU that loads libnoit.so holds these 64.25 KB until
// the process exits.  All calls on a device share the array (whatever context or stream they come
// from): calls that overlap on the GPU race.  The call makes no cudaMalloc / cudaFree and calls no
// allocating library routine; the counters that must start at zero are cleared by a memset node on
// `stream` in front of the kernel (the kernel also re-arms them, but a failed or aborted launch
// must not poison the next call).
// NOIT_BALANCE_STATIC_MAX_TILES (include/noit.h): 16384 base tiles, e.g. 8192 x 8192 pixels
constexpr uint32_t kStaticCounterWords = 64;           // [0] ticket, [4..7] histogram accumulators
static __device__ __align__(256) uint32_t g_balance_scratch[kStaticCounterWords + NOIT_BALANCE_STATIC_MAX_TILES];

// In host code `g_balance_scratch` is a host-side stand-in, not a device address: the address the
// kernel may use comes from cudaGetSymbolAddress, once per device, with that device current.
static uint32_t* balance_scratch_address(noit_ctx* ctx)
{
    static uint32_t* per_device[64] = {nullptr};
    const int dev = ctx->device;
    if (dev < 0 || dev >= 64) {
        noit_fail(ctx, NOIT_ERR_UNSUPPORTED, "noit_quadtree_balance_static: device index %d beyond 63", dev);
        return nullptr;
    }
    if (!per_device[dev]) {
        uint32_t* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_balance_scratch);   // current device == ctx->device (checked)
        if (e != cudaSuccess || !p) {
            noit_cuda_check(ctx, e != cudaSuccess ? e : cudaErrorInvalidSymbol,
                            "cudaGetSymbolAddress(g_balance_scratch)");
            return nullptr;
        }
        per_device[dev] = p;
    }
    return per_device[dev];
}

extern "C" noit_status noit_quadtree_balance_static(noit_ctx* ctx, int32_t width, int32_t height,
                                                    int32_t iterations, float delta2, float delta3,
                                                    uint32_t* tile_mask, uint8_t* tile_level,
                                                    uint8_t* cell_level, uint32_t* level_hist,
                                                    float* scales, void* stream)
{
    if (!ctx) return noit_fail(nullptr, NOIT_ERR_NULL, "noit_quadtree_balance_static: ctx is NULL");
    NOIT_TRY(noit_check_device(ctx, "noit_quadtree_balance_static"));
    if (!tile_mask) return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree_balance_static: tile_mask is NULL");
    if (scales && !level_hist)
        return noit_fail(ctx, NOIT_ERR_NULL, "noit_quadtree_balance_static: scales needs level_hist");
    if (width <= 0 || height <= 0 || (uint64_t)width * (uint64_t)height + 1 > 0xFFFFFFFFull)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree_balance_static: bad width/height");
    if (iterations < 0 || iterations > 16)
        return noit_fail(ctx, NOIT_ERR_SIZE, "noit_quadtree_balance_static: iterations must be in [0, 16]");
    const int64_t Tx = ((int64_t)width + 63) / 64, Ty = ((int64_t)height + 63) / 64, n = Tx * Ty;
    if (n > NOIT_BALANCE_STATIC_MAX_TILES)
        return noit_fail(ctx, NOIT_ERR_SIZE,
                         "noit_quadtree_balance_static: %lld base tiles (%d x %d pixels) exceed the static scratch of %d "
                         "tiles; use noit_quadtree_balance",
                         (long long)n, width, height, NOIT_BALANCE_STATIC_MAX_TILES);
    uint32_t* scratch = balance_scratch_address(ctx);
    if (!scratch) return NOIT_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: ticket and accumulators must start at zero (the
    // mask area needs no clearing -- every tile's word is written before the last block reads it)
    NOIT_CUDA(ctx, cudaMemsetAsync(scratch, 0, kStaticCounterWords * sizeof(uint32_t), st));
    balance_kernel<<<(int)((n + 3) / 4), 128, 0, st>>>(width, height, (int)Tx, (int)Ty, iterations, delta2, delta3,
                                                       tile_mask, scratch + kStaticCounterWords, tile_level, cell_level,
                                                       level_hist, scales, scratch + 0, scratch + 4);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}
