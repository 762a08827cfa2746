// noit_internal.cuh -- shared by the translation units of libnoit.so (CUDA path only).
// Nothing under oracle/ includes this file and this file includes nothing from there.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "noit.h"

// MLP parameter block passed BY VALUE as a kernel argument: kernel parameters live in constant
// bank 0, so every weight is a uniform constant-bank operand of an FFMA (no load instructions,
// no per-context __constant__ symbol).  Layout = noit_set_weights order.
struct MlpWeights {
    float w1[32][5];
    float b1[32];
    float w2[16][32];
    float b2[16];
    float w3[3][16];
    float b3[3];
};
static_assert(sizeof(MlpWeights) == NOIT_MLP_PARAMS * 4, "771 parameters (P:97)");

// The same parameters, input-major and padded, for the FFMA2 form of the MLP (two adjacent output
// neurons per instruction): w1t[i][o], w2t[i][o], w3t[i][o] with o padded to 4 in layer 3.
struct MlpWeightsT {
    float w1t[5][32];
    float b1[32];
    float w2t[32][16];
    float b2[16];
    float w3t[16][4];
    float b3[4];
};
static_assert(sizeof(MlpWeightsT) <= 4096, "fits the classic kernel-parameter space");

// NEXT-4 (comparison variant): the DFAOIT network, input-major and padded for FFMA2
// (w1t[i][o], w2t[i][o], w3t[i][o] with o padded to 4 in layer 3); 948 floats as a kernel argument
struct MlpWeights10T {
    float w1t[10][32];
    float b1[32];
    float w2t[32][16];
    float b2[16];
    float w3t[16][4];
    float b3[4];
};
static_assert(sizeof(MlpWeights10T) + 512 <= 4096 * 8, "kernel argument space");

#define NOIT_HOST_BANDS 8
// work counters: [0, 64) small counters of the quadtree / balance / resolve kernels, then the
// resolve's ticket counters, one per 128-byte line
#define NOIT_DEBUG_COUNTER 24          // d_counters[24]: violations counted by a NOIT_DEBUG_BOUNDS build
#define NOIT_TICKET_COUNTERS_LOG2 2
#define NOIT_COUNTER_WORDS (64 + 32 * (1 << NOIT_TICKET_COUNTERS_LOG2))
struct noit_ctx {
    int device = 0;
    bool has_weights = false;
    int precision = 0;
    MlpWeights w;                    // effective weights, host copy (kernel argument source)
    MlpWeightsT wt;                  // the same weights, input-major (FFMA2 form)
    uint8_t* d_tile_lod = nullptr;   // S7 per-tile mode: lod summary byte per 32-pixel tile
    size_t tile_lod_cap = 0;
    void* d_mlp = nullptr;           // device copy of the packed tensor-core operands (bf16 path)
    uint64_t launches = 0;
    char err[512] = {0};
    // device scratch (lazily allocated, kept between calls)
    uint32_t* d_counters = nullptr;  // small zero-initialised work counters
    float* d_coarse_g[2] = {nullptr, nullptr};   // S7: G[10] per half / quarter pixel
    size_t coarse_g_cap[2] = {0, 0};
    uint32_t* d_tile_depth = nullptr;            // NEXT-1: balanced masks before they are published (u32 per tile)
    size_t tile_depth_cap = 0;
    // staging for noit_resolve_host
    void* d_stage = nullptr;
    size_t stage_cap = 0;
    // noit_resolve_host pipelines the frame in bands: H2D copies, kernels (caller's stream) and
    // D2H copies run on three streams chained by events (created on first use)
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    cudaEvent_t host_ev[2 * NOIT_HOST_BANDS + 2] = {};
    int num_sms = 148;
};

noit_status noit_fail(noit_ctx* ctx, noit_status st, const char* fmt, ...);
noit_status noit_cuda_check(noit_ctx* ctx, cudaError_t e, const char* what);
noit_status noit_check_fragbuf(noit_ctx* ctx, const noit_fragbuf* fb, const char* name);
// a context lives on the device that was current at noit_create; every launching entry point checks it
noit_status noit_check_device(noit_ctx* ctx, const char* who);

#define NOIT_TRY(expr)                      \
    do {                                    \
        noit_status _st = (expr);           \
        if (_st != NOIT_OK) return _st;     \
    } while (0)
#define NOIT_CUDA(ctx, expr) NOIT_TRY(noit_cuda_check((ctx), (expr), #expr))

static inline bool noit_aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

// ------------------------------------------------------------------------------------------
// device helpers
// ------------------------------------------------------------------------------------------
#ifdef __CUDACC__

// fp16 -> fp32 widening is exact (O2).
__device__ __forceinline__ float4 load_rgba(const __half* rgba, uint32_t j)
{
    uint2 raw = __ldg(reinterpret_cast<const uint2*>(rgba) + j);
    __half2 rg = *reinterpret_cast<__half2*>(&raw.x);
    __half2 ba = *reinterpret_cast<__half2*>(&raw.y);
    float2 a = __half22float2(rg), b = __half22float2(ba);
    return make_float4(a.x, a.y, b.x, b.y);
}
__device__ __forceinline__ float4 load_rgba(const float* rgba, uint32_t j)
{
    return __ldg(reinterpret_cast<const float4*>(rgba) + j);
}

// Running k=2 selection (O1) + tail accumulators (O2) of one pixel, O(1) state.
// Fragments are pushed in index order, so a new fragment has a LARGER index than everything
// held: under the key (depth, index) it wins a slot only on a strictly smaller depth.  The
// candidate that ends up in neither slot (the new one, or the old layer 2) is folded into the
// tail -- never "all minus top-2", which cancels (S:7 hard parts).  Empty slots carry
// depth = +inf, alpha = 0: evicting one adds 0 and multiplies by 1.
template <bool kTrackIdx>
struct PixelState {
    float d1, d2;
    float4 c1, c2;
    uint32_t i1, i2;
    float acc_r, acc_g, acc_b, a_tail, t_tail;

    __device__ __forceinline__ void init()
    {
        d1 = d2 = __int_as_float(0x7f800000);
        c1 = c2 = make_float4(0.f, 0.f, 0.f, 0.f);
        i1 = i2 = NOIT_ABSENT;
        acc_r = acc_g = acc_b = a_tail = 0.f;
        t_tail = 1.f;
    }
    __device__ __forceinline__ void push(float d, float4 c, uint32_t j)
    {
        const bool lt1 = d < d1, lt2 = d < d2;
        float4 ev;                        // evicted candidate -> tail
        ev.x = lt2 ? c2.x : c.x; ev.y = lt2 ? c2.y : c.y;
        ev.z = lt2 ? c2.z : c.z; ev.w = lt2 ? c2.w : c.w;
        // new layer 2 = old layer 1 (if the newcomer is nearest), else newcomer, else unchanged
        c2.x = lt1 ? c1.x : (lt2 ? c.x : c2.x); c2.y = lt1 ? c1.y : (lt2 ? c.y : c2.y);
        c2.z = lt1 ? c1.z : (lt2 ? c.z : c2.z); c2.w = lt1 ? c1.w : (lt2 ? c.w : c2.w);
        d2 = lt1 ? d1 : (lt2 ? d : d2);
        c1.x = lt1 ? c.x : c1.x; c1.y = lt1 ? c.y : c1.y;
        c1.z = lt1 ? c.z : c1.z; c1.w = lt1 ? c.w : c1.w;
        d1 = lt1 ? d : d1;
        if (kTrackIdx) {
            i2 = lt1 ? i1 : (lt2 ? j : i2);
            i1 = lt1 ? j : i1;
        }
        acc_r = fmaf(ev.w, ev.x, acc_r);
        acc_g = fmaf(ev.w, ev.y, acc_g);
        acc_b = fmaf(ev.w, ev.z, acc_b);
        a_tail += ev.w;
        t_tail *= (1.f - ev.w);
    }
};

// O4: 5 -> 32 -> 16 -> 3, ReLU everywhere (A3).  One pixel per thread, everything in
// registers, weights as constant-bank operands.  Dot products start from the bias and run in
// input-index order (same order as the oracle; fp32 instead of double).
__device__ __forceinline__ void mlp_forward(const MlpWeights& W, const float x[5], float f[3])
{
    float h1[32], h2[16];
#pragma unroll
    for (int o = 0; o < 32; ++o) {
        float a = W.b1[o];
#pragma unroll
        for (int i = 0; i < 5; ++i) a = fmaf(W.w1[o][i], x[i], a);
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
        f[o] = fmaxf(a, 0.f);
    }
}

// fma.rn.f32x2 (sm_100): two independent IEEE fp32 FMAs in one instruction (SASS FFMA2).
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    unsigned long long ra = *reinterpret_cast<unsigned long long*>(&a);
    unsigned long long rb = *reinterpret_cast<unsigned long long*>(&b);
    unsigned long long rc = *reinterpret_cast<unsigned long long*>(&c);
    unsigned long long rd;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(rd) : "l"(ra), "l"(rb), "l"(rc));
    return *reinterpret_cast<float2*>(&rd);
}

// O4 with FFMA2: output neurons (o, o+1) share one instruction; each dot product still starts
// from its bias and runs in input-index order, so the result is bit-identical to mlp_forward.
__device__ __forceinline__ void mlp_forward_packed(const MlpWeightsT& W, const float x[5], float f[3])
{
    float2 h1[16], h2[8], h3[2];
#pragma unroll
    for (int o = 0; o < 16; ++o) h1[o] = make_float2(W.b1[2 * o], W.b1[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const float2 xi = make_float2(x[i], x[i]);
#pragma unroll
        for (int o = 0; o < 16; ++o)
            h1[o] = fma2(make_float2(W.w1t[i][2 * o], W.w1t[i][2 * o + 1]), xi, h1[o]);
    }
#pragma unroll
    for (int o = 0; o < 8; ++o) h2[o] = make_float2(W.b2[2 * o], W.b2[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const float v = fmaxf((i & 1) ? h1[i >> 1].y : h1[i >> 1].x, 0.f);
        const float2 hi = make_float2(v, v);
#pragma unroll
        for (int o = 0; o < 8; ++o)
            h2[o] = fma2(make_float2(W.w2t[i][2 * o], W.w2t[i][2 * o + 1]), hi, h2[o]);
    }
#pragma unroll
    for (int o = 0; o < 2; ++o) h3[o] = make_float2(W.b3[2 * o], W.b3[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const float v = fmaxf((i & 1) ? h2[i >> 1].y : h2[i >> 1].x, 0.f);
        const float2 hi = make_float2(v, v);
#pragma unroll
        for (int o = 0; o < 2; ++o)
            h3[o] = fma2(make_float2(W.w3t[i][2 * o], W.w3t[i][2 * o + 1]), hi, h3[o]);
    }
    f[0] = fmaxf(h3[0].x, 0.f);
    f[1] = fmaxf(h3[0].y, 0.f);
    f[2] = fmaxf(h3[1].x, 0.f);
}

// O12's network with FFMA2 (same structure as mlp_forward_packed): 10 -> 32 -> 16 -> 3, ReLU hidden,
// SIGMOID output ("differs only in the output activation"); dot products start from the bias
// and run in input-index order.
__device__ __forceinline__ void mlp10_forward_packed(const MlpWeights10T& W, const float x[10], float f[3])
{
    float2 h1[16], h2[8], h3[2];
#pragma unroll
    for (int o = 0; o < 16; ++o) h1[o] = make_float2(W.b1[2 * o], W.b1[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        const float2 xi = make_float2(x[i], x[i]);
#pragma unroll
        for (int o = 0; o < 16; ++o)
            h1[o] = fma2(make_float2(W.w1t[i][2 * o], W.w1t[i][2 * o + 1]), xi, h1[o]);
    }
#pragma unroll
    for (int o = 0; o < 8; ++o) h2[o] = make_float2(W.b2[2 * o], W.b2[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const float v = fmaxf((i & 1) ? h1[i >> 1].y : h1[i >> 1].x, 0.f);
        const float2 hi = make_float2(v, v);
#pragma unroll
        for (int o = 0; o < 8; ++o)
            h2[o] = fma2(make_float2(W.w2t[i][2 * o], W.w2t[i][2 * o + 1]), hi, h2[o]);
    }
#pragma unroll
    for (int o = 0; o < 2; ++o) h3[o] = make_float2(W.b3[2 * o], W.b3[2 * o + 1]);
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        const float v = fmaxf((i & 1) ? h2[i >> 1].y : h2[i >> 1].x, 0.f);
        const float2 hi = make_float2(v, v);
#pragma unroll
        for (int o = 0; o < 2; ++o)
            h3[o] = fma2(make_float2(W.w3t[i][2 * o], W.w3t[i][2 * o + 1]), hi, h3[o]);
    }
    f[0] = 1.0f / (1.0f + expf(-h3[0].x));
    f[1] = 1.0f / (1.0f + expf(-h3[0].y));
    f[2] = 1.0f / (1.0f + expf(-h3[1].x));
}

// ---- O4 on the tensor cores (weights exactly representable in TF32, i.e. NOIT_MLP_BF16) --------
// mma.sync.m16n8k8 TF32 with fp32 accumulation; every activation a is split into
// a_hi = a & 0xffffe000 (a valid TF32) and a_lo = a - a_hi (exact), and a*w = a_hi*w + a_lo*w is
// issued as two MMAs.  With w exact in TF32 the only loss is the truncation of a_lo to TF32
// inside the second MMA (< 2^-21 |a|): fp32-class accuracy, NOT bf16/tf32 activations (A6).
// One warp = 32 pixels = 2 m-tiles; row r of the MMA is lane r's pixel.  The C fragment of
// layer l's n-tile s is, register for register, the A fragment of layer l+1's k-step s once
// the hidden units are re-labelled (A col t <-> C col 2t, A col t+4 <-> C col 2t+1); that
// re-labelling lives in the packed weights (noit_set_weights), so layers chain with no shuffle.
// The bias of layer 1 rides in the zero padding of its K = 8: feature column 5 is the constant 1
// (hi = 1, lo = 0) and row 5 of the B operand is b1, so those chains start from C = 0; the biases
// of layers 2 and 3 are stored as whole C fragments {b[2t], b[2t+1], b[2t], b[2t+1]}, which a
// chain's first MMA reads in place (no register moves to assemble the quad).
// Packed weights: 10 float4 per lane, chunk v of lane l at wp[v*32 + l] (g = l>>2, t = l&3):
//   0-1 W1 B-frags (4 n-tiles x {k=t, k=t+4}; k=5 is b1), 2-5 W2 B-frags ((n-tile j, k-step s) x 2),
//   6-7 b2 C-frags (n-tile j), 8 W3 B-frags (2 k-steps x 2), 9 b3 C-frag.
#define NOIT_MMA_CHUNKS 10
__device__ __forceinline__ void mma_tf32(float (&d)[4], const float (&a)[4], float b0, float b1,
                                         const float (&c)[4])
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%10,%11,%12,%13};"
        : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
        : "r"(__float_as_uint(a[0])), "r"(__float_as_uint(a[1])), "r"(__float_as_uint(a[2])),
          "r"(__float_as_uint(a[3])), "r"(__float_as_uint(b0)), "r"(__float_as_uint(b1)),
          "f"(c[0]), "f"(c[1]), "f"(c[2]), "f"(c[3]));
}
__device__ __forceinline__ void split_tf32(float v, float& hi, float& lo)
{
    hi = __uint_as_float(__float_as_uint(v) & 0xffffe000u);
    lo = v - hi;
}
// relu + re-order of a C fragment into the next layer's A fragment, split into hi / lo
__device__ __forceinline__ void c_to_a(const float (&c)[4], float (&hi)[4], float (&lo)[4])
{
    split_tf32(fmaxf(c[0], 0.f), hi[0], lo[0]);
    split_tf32(fmaxf(c[2], 0.f), hi[1], lo[1]);
    split_tf32(fmaxf(c[1], 0.f), hi[2], lo[2]);
    split_tf32(fmaxf(c[3], 0.f), hi[3], lo[3]);
}
// All 32 lanes must call this.  x = this lane's features; scratch = 32 x 12 floats of shared
// memory private to the warp; f = tail colour of this lane's pixel; wv = this lane's packed
// weights, wv[v] = wp[v*32 + lane].
// Weight sources: registers (the 10 float4 of this lane, loaded once per tile) or the CTA's copy
// of the packed block in shared memory (read at the point of use: 40 registers fewer).
struct MmaWeightsReg {
    const float4 (&wv)[NOIT_MMA_CHUNKS];
    __device__ __forceinline__ float2 pair(int i) const      // packed values (i, i+1), i even
    {
        const float4& v = wv[i >> 2];
        return (i & 2) ? make_float2(v.z, v.w) : make_float2(v.x, v.y);
    }
    __device__ __forceinline__ float4 quad(int v) const { return wv[v]; }
};
struct MmaWeightsSmem {
    const float4* wl;                                        // &wsm[lane]; chunk v at wl[v * 32]
    __device__ __forceinline__ float2 pair(int i) const
    {
        return *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(wl + (i >> 2) * 32) + (i & 2));
    }
    __device__ __forceinline__ float4 quad(int v) const { return wl[v * 32]; }
};
template <typename WSrc>
__device__ __forceinline__ void mlp_forward_mma(const WSrc wsrc, float* scratch,
                                                int lane, const float x[5], float f[3])
{
    const int g = lane >> 2, t = lane & 3;
    // features -> A fragments of layer 1 through the scratch (row = lane, stride 12: no conflicts)
    __syncwarp();
    *reinterpret_cast<float4*>(scratch + 12 * lane) = make_float4(x[0], x[1], x[2], x[3]);
    scratch[12 * lane + 4] = x[4];
    __syncwarp();
    float fout[2][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const float* r0 = scratch + 12 * (16 * mt + g), *r1 = r0 + 12 * 8;
        float ahi[4], alo[4];
        split_tf32(r0[t], ahi[0], alo[0]);
        split_tf32(r1[t], ahi[1], alo[1]);
        split_tf32(t == 0 ? r0[4] : 0.f, ahi[2], alo[2]);
        split_tf32(t == 0 ? r1[4] : 0.f, ahi[3], alo[3]);
        if (t == 1) ahi[2] = ahi[3] = 1.0f;                   // column 5: the constant feature
        // layer 1: 4 n-tiles, K = 8 (5 features + the constant + zero padding)
        const float zero[4] = {0.f, 0.f, 0.f, 0.f};
        float h1hi[4][4], h1lo[4][4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float c[4];
            const float2 b = wsrc.pair(2 * j);
            mma_tf32(c, ahi, b.x, b.y, zero);
            mma_tf32(c, alo, b.x, b.y, c);
            c_to_a(c, h1hi[j], h1lo[j]);
        }
        // layer 2: 2 n-tiles, 4 k-steps (k-step s = layer-1 n-tile s)
        float h2hi[2][4], h2lo[2][4];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const float4 bq = wsrc.quad(6 + j);
            const float bias[4] = {bq.x, bq.y, bq.z, bq.w};
            float c[4];
#pragma unroll
            for (int s = 0; s < 4; ++s) {
                const float2 b = wsrc.pair(8 + 2 * (4 * j + s));
                if (s == 0) mma_tf32(c, h1hi[s], b.x, b.y, bias);
                else mma_tf32(c, h1hi[s], b.x, b.y, c);
                mma_tf32(c, h1lo[s], b.x, b.y, c);
            }
            c_to_a(c, h2hi[j], h2lo[j]);
        }
        // layer 3: 1 n-tile (3 outputs, padded to 8), 2 k-steps
        const float4 b3q = wsrc.quad(9);
        const float bias3[4] = {b3q.x, b3q.y, b3q.z, b3q.w};
        float c[4];
#pragma unroll
        for (int s = 0; s < 2; ++s) {
            const float2 b = wsrc.pair(32 + 2 * s);
            if (s == 0) mma_tf32(c, h2hi[s], b.x, b.y, bias3);
            else mma_tf32(c, h2hi[s], b.x, b.y, c);
            mma_tf32(c, h2lo[s], b.x, b.y, c);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) fout[mt][k] = fmaxf(c[k], 0.f);
    }
    // C fragments (row g / g+8, cols 2t, 2t+1) -> one row per lane
    __syncwarp();
    if (t < 2) {
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
            float* r0 = scratch + 12 * (16 * mt + g) + 2 * t, *r1 = r0 + 12 * 8;
            *reinterpret_cast<float2*>(r0) = make_float2(fout[mt][0], fout[mt][1]);
            *reinterpret_cast<float2*>(r1) = make_float2(fout[mt][2], fout[mt][3]);
        }
    }
    __syncwarp();
    const float4 o = *reinterpret_cast<const float4*>(scratch + 12 * lane);
    f[0] = o.x; f[1] = o.y; f[2] = o.z;
}

// O3 features from raw accumulators; returns has_tail (A2).
__device__ __forceinline__ bool make_features(float n, float t_tail, float ar, float ag, float ab,
                                              float a_tail, float x[5])
{
    const bool has_tail = a_tail > 0.f;
    x[0] = n;
    x[1] = t_tail;
    x[2] = has_tail ? ar / a_tail : 0.f;
    x[3] = has_tail ? ag / a_tail : 0.f;
    x[4] = has_tail ? ab / a_tail : 0.f;
    return has_tail;
}

#endif  // __CUDACC__
