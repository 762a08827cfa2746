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

struct noit_ctx {
    int device = 0;
    bool has_weights = false;
    int precision = 0;
    MlpWeights w;                    // effective weights, host copy (kernel argument source)
    MlpWeightsT wt;                  // the same weights, input-major (FFMA2 form)
    void* d_mlp = nullptr;           // device copy of the packed tensor-core operands (bf16 path)
    uint64_t launches = 0;
    char err[512] = {0};
    // device scratch (lazily allocated, kept between calls)
    uint32_t* d_counters = nullptr;  // small zero-initialised work counters
    float* d_coarse_g[2] = {nullptr, nullptr};   // S7: G[10] per half / quarter pixel
    size_t coarse_g_cap[2] = {0, 0};
    // staging for noit_resolve_host
    void* d_stage = nullptr;
    size_t stage_cap = 0;
    int num_sms = 148;
};

noit_status noit_fail(noit_ctx* ctx, noit_status st, const char* fmt, ...);
noit_status noit_cuda_check(noit_ctx* ctx, cudaError_t e, const char* what);
noit_status noit_check_fragbuf(noit_ctx* ctx, const noit_fragbuf* fb, const char* name);

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
