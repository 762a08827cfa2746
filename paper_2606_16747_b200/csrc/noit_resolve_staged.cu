// noit_resolve_staged.cu -- the plain fused resolve (S1-S5, Eq. 4) of a whole frame:
// persistent warps, fragment ranges staged into shared memory by 1-D TMA bulk copies
// (cp.async.bulk + mbarrier), two passes over the staged lists, MLP on the tensor cores
// (mma.sync TF32 with a two-pass activation split) or with packed FFMA2 (fp32 weights).
// One kernel, three modes: whole frame (S1-S5), adaptive frame (S7), pixel list (S9).
//
// Why this shape (ncu evidence in profiles/r01_*): a thread-per-pixel kernel that reads its
// list straight from global memory is bound by L1 data-stage wavefronts (every lane of a load
// touches a different 128-byte line: 12.5 wavefronts per request, 74 % of the LSU data pipe at
// 48 % of the HBM roofline) and by its instruction count (36 per fragment, ~1000 per MLP).
// Here
//   * a WARP owns a tile of 32 consecutive pixels; their CSR lists are one contiguous fragment
//     range, which lane 0 copies into the warp's private shared-memory stage with bulk copies
//     that complete on the warp's mbarrier: no LSU wavefronts, no registers, coalesced HBM reads;
//   * selection and reduction are two passes over the staged list: pass 1 tracks
//     (d1,i1,d2,i2) on the depths only; the owner lane fetches the two layer colours and
//     overwrites their alpha with 0 in the stage; pass 2 then accumulates EVERY staged fragment
//     of the pixel (a zero alpha adds 0 and multiplies by 1), so the tail is never "all minus
//     top-2" (O2) and pass 2 has no per-fragment test;
//   * LIGHT tiles (all 32 lists fit the stage: 76 % of cfg3's tiles, 9 fragments per pixel on
//     average) run one lane per pixel: no shuffles, no merges -- there the per-tile overhead,
//     not the per-fragment work, is what counts;
//   * HEAVY tiles (72 fragments per pixel on average in cfg3) run L = 4 lanes per pixel in 4
//     rounds of 8 pixels (lane q of a group reads fragments b+q, b+q+4, ...: balanced trip
//     counts, few bank conflicts).  The stage is used twice: first for depths only (3x the
//     fragments fit), pass 1 of all rounds, ONE transposed butterfly that leaves lane q of a
//     group with round q's merged top-2 (log2(L) exchange steps, L-1 merges, instead of L full
//     butterflies); then for colours only, in chunks of rounds, pass 2, and one transposed
//     butterfly of the five sums;
//   * every lane then owns one pixel: features, MLP (noit_internal.cuh: mlp_forward_mma /
//     mlp_forward_packed), composite, 128-bit stores.  The next tile's first fill is issued
//     before the MLP, which hides its latency.
// Tiles are handed out by an atomic counter (fragment counts vary 0..128 per pixel) whose result
// is broadcast one tile later, and which the last warp to finish resets (no memset per launch).
#include "noit_resolve_common.cuh"

namespace {

#ifndef NOIT_X_STAGE
#define NOIT_X_STAGE 12000
#endif
#ifndef NOIT_X_WARPS
#define NOIT_X_WARPS 4
#endif
#ifndef NOIT_X_CTAS
#define NOIT_X_CTAS 4
#endif
#ifndef NOIT_X_WSMEM
#define NOIT_X_WSMEM 0
#endif
#ifndef NOIT_X_LIST_L
#define NOIT_X_LIST_L 2              // lanes per listed pixel in S9 (32 / L pixels per warp tile)
#endif
#ifndef NOIT_X_PAD
#define NOIT_X_PAD 0                 // extra dynamic shared memory per CTA: lowers the occupancy, same code
#endif
constexpr uint32_t kStageBytesFrame = NOIT_X_STAGE;   // per warp stage (1000 fragments with fp16 colour)
constexpr uint32_t kScratchFloats = 32 * 12;   // per warp: feature / output transpose of the MMA MLP
constexpr int kWarpsPerCta = NOIT_X_WARPS;
constexpr bool kWeightsInSmem = NOIT_X_WSMEM != 0;
constexpr uint32_t kWeightBytes = kWeightsInSmem ? NOIT_MMA_CHUNKS * 32 * 16 : 0;

// Bounds-checked build (-DNOIT_DEBUG_BOUNDS, libnoit_debug.so; compute-sanitizer is closed on the
// GPU pool): every range of the warp's stage a scan, a layer fetch or a bulk copy is about to touch
// is checked against the stage, every global fragment range against [0, F); a violation is counted
// in a context counter (noit_debug_bounds_violations) and the access is still made, so a parity
// run of this build that counts zero has made no out-of-stage shared or out-of-range global access.
#ifdef NOIT_DEBUG_BOUNDS
#define NOIT_CHK_STAGE(ptr, bytes)                                                                  \
    do {                                                                                            \
        const unsigned char* _q = reinterpret_cast<const unsigned char*>(ptr);                     \
        if ((bytes) != 0 && (_q < stage || _q + (bytes) > stage + kStageBytes))                    \
            atomicAdd(A.tile_counter + NOIT_DEBUG_COUNTER, 1u);                                     \
    } while (0)
#define NOIT_CHK_FRAGS(first, count)                                                                \
    do {                                                                                            \
        if ((uint64_t)(first) + (uint64_t)(count) > (uint64_t)A.F) atomicAdd(A.tile_counter + NOIT_DEBUG_COUNTER, 1u); \
    } while (0)
#else
#define NOIT_CHK_STAGE(ptr, bytes) do {} while (0)
#define NOIT_CHK_FRAGS(first, count) do {} while (0)
#endif
constexpr uint32_t kCounterShift = NOIT_TICKET_COUNTERS_LOG2;

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}
// 1-D TMA: global -> this CTA's shared memory, completion counted in bytes on `bar`.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}

// ---- colour formats ------------------------------------------------------------------------
template <typename ColorT> struct Color;
template <> struct Color<__half> {
    typedef uint2 Packed;                                   // 4 halves
    static constexpr uint32_t kBytes = 8;
    static __device__ __forceinline__ Packed zero() { return make_uint2(0u, 0u); }
    static __device__ __forceinline__ float4 unpack(Packed v)
    {
        const float2 a = __half22float2(*reinterpret_cast<__half2*>(&v.x));
        const float2 b = __half22float2(*reinterpret_cast<__half2*>(&v.y));
        return make_float4(a.x, a.y, b.x, b.y);
    }
    static __device__ __forceinline__ void zero_alpha(Packed* slot)
    {
        reinterpret_cast<unsigned short*>(slot)[3] = 0;
    }
    static __device__ __forceinline__ Packed zero_alpha_reg(Packed v)
    {
        v.y &= 0x0000FFFFu;
        return v;
    }
    static __device__ __forceinline__ void zero_all(Packed* slot) { *slot = make_uint2(0u, 0u); }
    // O2's tail sums for one fragment.  sm_100a has mixed-precision fp32 += fp16 * fp16
    // (`fma.rn.f32.f16`, SASS FHFMA, with half-select operands) and fp32 += fp16 (FHADD): the
    // product of two halves is exact in fp32 and the sum is rounded once, i.e. bit for bit what
    // fmaf(float(a), float(c), acc) gives -- without the three conversions (6 instead of 9
    // instructions per fragment; only alpha is converted, for the transmittance product).
    static __device__ __forceinline__ float fhfma(unsigned short a, unsigned short b, float c)
    {
        asm("fma.rn.f32.f16 %0, %1, %2, %0;" : "+f"(c) : "h"(a), "h"(b));
        return c;
    }
    static __device__ __forceinline__ float fhadd(unsigned short a, float c)
    {
        asm("add.rn.f32.f16 %0, %1, %0;" : "+f"(c) : "h"(a));
        return c;
    }
    static __device__ __forceinline__ void accumulate(Packed v, float& r, float& g, float& b, float& a, float& t)
    {
        const unsigned short x = (unsigned short)(v.x & 0xffffu), y = (unsigned short)(v.x >> 16);
        const unsigned short z = (unsigned short)(v.y & 0xffffu), w = (unsigned short)(v.y >> 16);
        r = fhfma(w, x, r);
        g = fhfma(w, y, g);
        b = fhfma(w, z, b);
        a = fhadd(w, a);
        const float wf = __half2float(__ushort_as_half(w));
        t = fmaf(-wf, t, t);                               // t *= (1 - alpha), one rounding
    }
    // O12 (DFAOIT features): also the plain colour sums of the tail (three more FHADD)
    static __device__ __forceinline__ void accumulate_colour(Packed v, float& cr, float& cg, float& cb)
    {
        cr = fhadd((unsigned short)(v.x & 0xffffu), cr);
        cg = fhadd((unsigned short)(v.x >> 16), cg);
        cb = fhadd((unsigned short)(v.y & 0xffffu), cb);
    }
};
template <> struct Color<float> {
    typedef float4 Packed;
    static constexpr uint32_t kBytes = 16;
    static __device__ __forceinline__ Packed zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }
    static __device__ __forceinline__ float4 unpack(Packed v) { return v; }
    static __device__ __forceinline__ void zero_alpha(Packed* slot) { slot->w = 0.f; }
    static __device__ __forceinline__ Packed zero_alpha_reg(Packed v) { v.w = 0.f; return v; }
    static __device__ __forceinline__ void zero_all(Packed* slot) { *slot = make_float4(0.f, 0.f, 0.f, 0.f); }
    static __device__ __forceinline__ void accumulate_colour(Packed c, float& cr, float& cg, float& cb)
    {
        cr += c.x; cg += c.y; cb += c.z;
    }
    static __device__ __forceinline__ void accumulate(Packed c, float& r, float& g, float& b, float& a, float& t)
    {
        r = fmaf(c.w, c.x, r);
        g = fmaf(c.w, c.y, g);
        b = fmaf(c.w, c.z, b);
        a += c.w;
        t = fmaf(-c.w, t, t);                              // t *= (1 - alpha), one rounding
    }
};

// key (depth, index) lexicographic (O1)
__device__ __forceinline__ bool key_less(float da, uint32_t ia, float db, uint32_t ib)
{
    return da < db || (da == db && ia < ib);
}

}  // namespace


// ------------------------------------------------------------------------------------------
// building blocks
// ------------------------------------------------------------------------------------------
// What a lane owns at the end of a tile.
template <typename ColorT>
struct Owned {
    typename Color<ColorT>::Packed c1, c2;
    float d1;
    uint32_t n;
    float acc_r, acc_g, acc_b, a_tail, t_tail;
    float sum_r, sum_g, sum_b;            // O12 only: plain colour sums of the tail
};

struct Top2 { float d1, d2; uint32_t i1, i2; };
struct Sums { float r, g, b, a, t, cr, cg, cb; };

// newcomer at a larger index wins a slot only on a strictly smaller depth (O1 tie rule)
__device__ __forceinline__ void top2_push(Top2& s, float d, uint32_t pos)
{
    const bool lt1 = d < s.d1, lt2 = d < s.d2;
    s.i2 = lt1 ? s.i1 : (lt2 ? pos : s.i2);
    s.d2 = lt1 ? s.d1 : (lt2 ? d : s.d2);
    s.i1 = lt1 ? pos : s.i1;
    s.d1 = lt1 ? d : s.d1;
}
// merge another sorted pair into s under the key (depth, index)
__device__ __forceinline__ void top2_merge(Top2& s, float od1, uint32_t oi1, float od2, uint32_t oi2)
{
    const bool mine = key_less(s.d1, s.i1, od1, oi1);
    const float xd = mine ? s.d2 : od2, yd = mine ? od1 : s.d1;     // runner-up of the winner side,
    const uint32_t xi = mine ? s.i2 : oi2, yi = mine ? oi1 : s.i1;  // best of the loser side
    const bool xy = key_less(xd, xi, yd, yi);
    s.d1 = mine ? s.d1 : od1;
    s.i1 = mine ? s.i1 : oi1;
    s.d2 = xy ? xd : yd;
    s.i2 = xy ? xi : yi;
}

// pass 1 over positions first, first+S, ... < end of the staged depths
template <int S>
__device__ __forceinline__ Top2 scan_depths(const float* D, uint32_t first, uint32_t end)
{
    Top2 s;
    s.d1 = s.d2 = __int_as_float(0x7f800000);
    s.i1 = s.i2 = NOIT_ABSENT;
    uint32_t pos = first;
#pragma unroll 1
    for (; pos + S < end; pos += 2 * S) {
        const float da = D[pos], db = D[pos + S];
        top2_push(s, da, pos);
        top2_push(s, db, pos + S);
    }
    if (pos < end) top2_push(s, D[pos], pos);
    return s;
}
// pass 2 over the same positions of the staged colours (layers carry alpha 0)
template <typename ColorT, int S, bool kFeat10 = false>
__device__ __forceinline__ Sums scan_colours(const typename Color<ColorT>::Packed* C, uint32_t first,
                                             uint32_t end)
{
    typedef typename Color<ColorT>::Packed Packed;
    Sums s;
    s.r = s.g = s.b = s.a = 0.f;
    s.cr = s.cg = s.cb = 0.f;
    s.t = 1.f;
    auto acc = [&](Packed raw) {
        Color<ColorT>::accumulate(raw, s.r, s.g, s.b, s.a, s.t);
        if (kFeat10) Color<ColorT>::accumulate_colour(raw, s.cr, s.cg, s.cb);
    };
    uint32_t pos = first;
#pragma unroll 1
    for (; pos + S < end; pos += 2 * S) {
        const Packed ra = C[pos], rb = C[pos + S];
        acc(ra);
        acc(rb);
    }
    if (pos < end) acc(C[pos]);
    return s;
}

// Transposed butterfly over L items held by each of the L lanes of a group: at step m the
// live slots are [0, 2m); a lane with bit m of q clear keeps slot r and sends slot r+m (r < m),
// its partner q^m does the opposite; the combined item goes to slot r.  After the last step
// slot 0 of lane q holds item q combined over the whole group.
template <int L>
__device__ __forceinline__ void transposed_merge(Top2 (&s)[L], int q)
{
#pragma unroll
    for (int m = L / 2; m >= 1; m >>= 1) {
        const bool up = (q & m) != 0;
#pragma unroll
        for (int r = 0; r < L; ++r) {
            if (r >= m) continue;
            Top2 keep = up ? s[r + m] : s[r];
            const Top2 send = up ? s[r] : s[r + m];
            top2_merge(keep, __shfl_xor_sync(0xffffffffu, send.d1, m), __shfl_xor_sync(0xffffffffu, send.i1, m),
                       __shfl_xor_sync(0xffffffffu, send.d2, m), __shfl_xor_sync(0xffffffffu, send.i2, m));
            s[r] = keep;
        }
    }
}
template <int L, bool kFeat10 = false>
__device__ __forceinline__ void transposed_sum(Sums (&s)[L], int q)
{
#pragma unroll
    for (int m = L / 2; m >= 1; m >>= 1) {
        const bool up = (q & m) != 0;
#pragma unroll
        for (int r = 0; r < L; ++r) {
            if (r >= m) continue;
            const Sums keep = up ? s[r + m] : s[r];
            const Sums send = up ? s[r] : s[r + m];
            s[r].r = keep.r + __shfl_xor_sync(0xffffffffu, send.r, m);
            s[r].g = keep.g + __shfl_xor_sync(0xffffffffu, send.g, m);
            s[r].b = keep.b + __shfl_xor_sync(0xffffffffu, send.b, m);
            s[r].a = keep.a + __shfl_xor_sync(0xffffffffu, send.a, m);
            s[r].t = keep.t * __shfl_xor_sync(0xffffffffu, send.t, m);
            if (kFeat10) {
                s[r].cr = keep.cr + __shfl_xor_sync(0xffffffffu, send.cr, m);
                s[r].cg = keep.cg + __shfl_xor_sync(0xffffffffu, send.cg, m);
                s[r].cb = keep.cb + __shfl_xor_sync(0xffffffffu, send.cb, m);
            }
        }
    }
}

// ---- cold path: a tile with a round too long for the stage (lists far beyond BASELINE.json's
// 128-fragment cap) reads global memory directly; the two layers are skipped by index in pass 2.
template <typename ColorT, int L, int kRounds, bool kFeat10 = false>
__device__ __noinline__ Owned<ColorT> tile_from_global(int lane, uint32_t o0, uint32_t o1,
                                                       const float* __restrict__ depth,
                                                       const typename Color<ColorT>::Packed* __restrict__ rgba)
{
    constexpr int PPR = 32 / L;
    const int g = lane / L, q = lane % L;
    Owned<ColorT> own;
    own.c1 = own.c2 = Color<ColorT>::zero();
    own.d1 = 1.0f; own.n = 0;
    own.acc_r = own.acc_g = own.acc_b = own.a_tail = 0.f; own.t_tail = 1.f;
    own.sum_r = own.sum_g = own.sum_b = 0.f;
    for (int r = 0; r < kRounds; ++r) {
        const int px = r * PPR + g;
        const uint32_t b = __shfl_sync(0xffffffffu, o0, px), e = __shfl_sync(0xffffffffu, o1, px);
        Top2 s;
        s.d1 = s.d2 = __int_as_float(0x7f800000);
        s.i1 = s.i2 = NOIT_ABSENT;
        // latency-bound (scattered lists): eight loads in flight per lane; the depth lines of the
        // whole list are requested into L2 up front (later batches of eight then hit L2), and the
        // colours are pulled into L2 while the depths are scanned
        for (uint32_t j = b + 32u * q; j < e; j += 32u * L)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(depth + j));
#pragma unroll 8
        for (uint32_t j = b + q; j < e; j += L) {
            asm volatile("prefetch.global.L2 [%0];" ::"l"(rgba + j));
            top2_push(s, __ldg(depth + j), j);
        }
#pragma unroll
        for (int m = 1; m < L; m <<= 1)
            top2_merge(s, __shfl_xor_sync(0xffffffffu, s.d1, m), __shfl_xor_sync(0xffffffffu, s.i1, m),
                       __shfl_xor_sync(0xffffffffu, s.d2, m), __shfl_xor_sync(0xffffffffu, s.i2, m));
        float ar = 0.f, ag = 0.f, ab = 0.f, at = 0.f, tt = 1.f, cr = 0.f, cg = 0.f, cb = 0.f;
#pragma unroll 8
        for (uint32_t j = b + q; j < e; j += L) {
            typename Color<ColorT>::Packed raw = __ldg(rgba + j);
            if (j == s.i1 || j == s.i2) raw = kFeat10 ? Color<ColorT>::zero() : Color<ColorT>::zero_alpha_reg(raw);
            Color<ColorT>::accumulate(raw, ar, ag, ab, at, tt);
            if (kFeat10) Color<ColorT>::accumulate_colour(raw, cr, cg, cb);
        }
#pragma unroll
        for (int m = 1; m < L; m <<= 1) {
            ar += __shfl_xor_sync(0xffffffffu, ar, m); ag += __shfl_xor_sync(0xffffffffu, ag, m);
            ab += __shfl_xor_sync(0xffffffffu, ab, m); at += __shfl_xor_sync(0xffffffffu, at, m);
            tt *= __shfl_xor_sync(0xffffffffu, tt, m);
            if (kFeat10) {
                cr += __shfl_xor_sync(0xffffffffu, cr, m); cg += __shfl_xor_sync(0xffffffffu, cg, m);
                cb += __shfl_xor_sync(0xffffffffu, cb, m);
            }
        }
        if (q == r) {
            own.c1 = s.i1 != NOIT_ABSENT ? __ldg(rgba + s.i1) : Color<ColorT>::zero();
            own.c2 = s.i2 != NOIT_ABSENT ? __ldg(rgba + s.i2) : Color<ColorT>::zero();
            own.d1 = s.d1;
            own.n = e - b;
            own.acc_r = ar; own.acc_g = ag; own.acc_b = ab; own.a_tail = at; own.t_tail = tt;
            own.sum_r = cr; own.sum_g = cg; own.sum_b = cb;
        }
    }
    return own;
}

// ------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------
// WT = MlpWeightsT: the paper's resolve (O1-O5); WT = MlpWeights10T: the DFAOIT resolve it is
// compared with (O12: ten features, sigmoid network predicting C_t, Eq. 3) -- same scan, three
// more sums per tail fragment, the two layers zeroed whole in the stage.
template <typename ColorT, int L, bool kMma, int kMode, typename WT = MlpWeightsT>
__global__ void __launch_bounds__(kWarpsPerCta * 32, kMode == NOIT_RESOLVE_LIST ? 7 : NOIT_X_CTAS)
resolve_staged_kernel(const __grid_constant__ ResolveArgs A, const __grid_constant__ WT W)
{
    constexpr bool kFeat10 = sizeof(WT) == sizeof(MlpWeights10T);
    static_assert(!kFeat10 || (!kMma && kMode == NOIT_RESOLVE_ALL), "O12 runs on whole frames with the FFMA2 network");
    typedef typename Color<ColorT>::Packed Packed;
    constexpr uint32_t CB = Color<ColorT>::kBytes;
    // per warp; S9 reads global memory directly and allocates no stage (more CTAs per SM)
    // fragments of a light tile (depths and colours staged together)
    constexpr uint32_t kCap = (kStageBytesFrame / (4u + CB)) & ~3u;
    constexpr uint32_t kStageBytes = kMode == NOIT_RESOLVE_LIST ? 0u : kStageBytesFrame;
    // fragments when the stage holds depths only / colours only; multiples of 4 because a copy
    // is rounded up to 4 fragments
    constexpr uint32_t kCapD = (kStageBytes / 4u) & ~3u;
    constexpr uint32_t kCapC = (kStageBytes / CB) & ~3u;
    constexpr int PPR = 32 / L;
    constexpr bool kGlobal = kMode == NOIT_RESOLVE_GLOBAL;              // frame-global lods (O7g)
    constexpr bool kCoarse = kMode == NOIT_RESOLVE_ADAPTIVE || kGlobal;   // some pixels may read G
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned char* stage = smem_raw + warp * kStageBytes;
    float* const sD = reinterpret_cast<float*>(stage);                   // depths (both views)
    Packed* const sC2 = reinterpret_cast<Packed*>(stage + kCap * 4u);    // colours behind kCap depths
    Packed* const sC = reinterpret_cast<Packed*>(stage);                 // colours only
    // layout: stages | scratch (16-byte aligned rows) | mbarriers
    float* const scratch = reinterpret_cast<float*>(smem_raw + kWarpsPerCta * kStageBytes) + warp * kScratchFloats;
    const uint32_t bar = smem_u32(reinterpret_cast<uint64_t*>(smem_raw + kWarpsPerCta * kStageBytes +
                                                              kWarpsPerCta * kScratchFloats * sizeof(float)) + warp);
    static_assert(kStageBytes % 16 == 0 && (kCap * 4u) % 16 == 0, "bulk copies need 16-byte aligned destinations");
    static_assert(kMode != NOIT_RESOLVE_LIST || kStageBytes == 0, "S9 never touches the stage");
    if (lane == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    // the CTA's copy of the packed MMA weights (read at the point of use instead of held in 40 registers)
    const float4* const wsm = reinterpret_cast<const float4*>(
        smem_raw + kWarpsPerCta * kStageBytes + kWarpsPerCta * kScratchFloats * sizeof(float) + kWarpsPerCta * 8u);
    if (kMma && kWeightsInSmem) {
        for (uint32_t i = threadIdx.x; i < NOIT_MMA_CHUNKS * 32u; i += kWarpsPerCta * 32u)
            const_cast<float4*>(wsm)[i] = __ldg(A.mlp_packed + i);
        __syncthreads();
    }
    uint32_t parity = 0;

    const uint32_t* __restrict__ offsets = A.offsets;
    const Packed* __restrict__ g_rgba = static_cast<const Packed*>(A.rgba);

    // lane 0's atomic result is broadcast one tile later: its latency hides behind a tile
    // (inline PTX: the compiler turns `if (lane == 0) atomicAdd` into a warp-aggregated atomic
    // followed by an immediate SHFL of its result, which waits for the atomic on the spot)
    // The first three tiles of a warp are static (warp id + k * warps): no atomic round trips at
    // start-up; the counter hands out the tiles after those.
    const uint32_t n_warps = gridDim.x * kWarpsPerCta, warp_id = blockIdx.x * kWarpsPerCta + warp;
    // (ptxas warp-aggregates an atomic whose address and addend are uniform -- vote, leader
    // election, and a SHFL of the result right behind the ATOMG, which stalls the warp for the
    // whole round trip -- even for inline PTX under `if (lane == 0)`.  The addend below is
    // laneid + 1 under the predicate laneid == 0: not uniform to ptxas, so the atomic stays a
    // plain predicated ATOMG and nothing waits for it until the broadcast a tile later.)
    // Tickets are dealt from 2^kCounterShift counters on separate 128-byte lines: warp w draws
    // from counter c = w mod 2^kCounterShift, whose k-th value stands for ticket
    // (k << kCounterShift) | c, so every counter covers an evenly interleaved share of the frame.
    // (With ONE counter a 4K frame of short lists -- 259 200 same-address atomics -- was measured
    // in two states, 344 us and 640 us per frame, same bytes and instructions, the second with
    // the long-scoreboard stall 16x higher: the atomics serialise in their L2 slice.  Four
    // counters never showed the slow state; profiles/r02_resolve.md.)
    const uint32_t my_c = warp_id & ((1u << kCounterShift) - 1u);
    uint32_t* const my_counter = A.tile_counter + 64u + 32u * my_c;
    auto fetch_raw = [&]() -> uint32_t {
        uint32_t t = 0;
        asm volatile("{\n"
                     ".reg .pred p;\n"
                     ".reg .u32 l, inc;\n"
                     "mov.u32 l, %%laneid;\n"
                     "setp.eq.u32 p, l, 0;\n"
                     "add.u32 inc, l, 1;\n"
                     "@p atom.global.add.u32 %0, [%1], inc;\n"
                     "}\n"
                     : "+r"(t)
                     : "l"(my_counter)
                     : "memory");
        return t;                                        // raw: turned into a ticket a tile later
    };
    // S9 (kMode LIST): "tile" t = entries [t*32/L, (t+1)*32/L) of the pixel list; the lists of a
    // tile are not contiguous, so such tiles always take the global path.
    const uint32_t list_total = kMode == NOIT_RESOLVE_LIST ? min(__ldg(A.pixel_count), A.P) : 0u;
    const uint32_t num_tiles = kMode == NOIT_RESOLVE_LIST ? (list_total + PPR - 1u) / PPR : A.num_tiles;
    // pixel index this lane loads the offsets of (kMode ALL / ADAPTIVE: tiles are taken from the
    // end of the frame backwards -- shorter tail in cfg3: 1.5 % vs 4.6 % of the makespan in a
    // list-scheduling model of the measured tile costs)
    auto lane_pixel = [&](uint32_t tile) -> uint32_t {
        if constexpr (kMode == NOIT_RESOLVE_LIST) {
            const uint32_t i = tile * PPR + (lane % PPR);        // lanes 0..PPR-1 hold the entries
            return i < list_total ? __ldg(A.pixel_list + i) : 0xFFFFFFFFu;
        }
        return (num_tiles - 1u - tile) * 32u + lane;
    };
    auto load_offsets = [&](uint32_t pix, uint32_t& a, uint32_t& b) {
        if (kMode == NOIT_RESOLVE_LIST) {
            a = pix < A.P ? __ldg(offsets + pix) : 0u;
            b = pix < A.P ? __ldg(offsets + pix + 1u) : a;
        } else {
            a = __ldg(offsets + min(pix, A.P));
            b = __ldg(offsets + min(pix + 1u, A.P));
        }
    };
    // S7 (kMode ADAPTIVE): lod of a pixel.  Every tile runs the staged path; pixels with lod > 0
    // then take layer 2 / the tail from the coarse G in the epilogue, and a tile whose pixels ALL
    // do stages only its depths.
    // frame-global lods of pass 2 / pass 3 from the Eq. 2 scales (O7g, A27), decided here
    int g_lod2 = 0, g_lod3 = 0;
    if (kGlobal) {
        const float s2 = __ldg(A.pass_scales + 1), s3 = __ldg(A.pass_scales + 2);
        g_lod2 = s2 > 0.70710678f ? 0 : (s2 > 0.35355339f ? 1 : 2);
        g_lod3 = s3 > 0.70710678f ? 0 : (s3 > 0.35355339f ? 1 : 2);
    }
    auto lane_lod = [&](uint32_t pix, int& level) -> int {
        level = 3;
        if (!kCoarse || pix >= A.P) return 0;
        if (kGlobal) return max(g_lod2, g_lod3);
        const uint32_t y = pix / (uint32_t)A.W, x = pix - y * (uint32_t)A.W;
        level = A.cell_level[(size_t)(y >> 3) * ((A.W + 7) >> 3) + (x >> 3)] & 3;
        return A.level_to_lod[level];
    };
    // What the tile loop needs to know about a tile's lods: bit 0 = some pixel has lod > 0
    // ("mixed": the epilogue looks at G), bit 1 = every pixel takes layer 2 AND the tail from a
    // coarse buffer (only the depths are staged).  Per-tile mode: one byte per tile written by the
    // pre-pass (tile_lod_summary in noit_resolve.cu) -- a level lookup per lane plus two votes per
    // tile cost the mode 100 instructions per tile; frame-global mode: the same for every tile.
    const uint32_t g_flags = (max(g_lod2, g_lod3) > 0 ? 1u : 0u) | ((g_lod2 > 0 && g_lod3 > 0) ? 3u : 0u);
    auto tile_flags = [&](uint32_t tile) -> uint32_t {
        if (!kCoarse) return 0u;
        if (kGlobal) return g_flags;
        return __ldg(A.tile_lod + (num_tiles - 1u - tile));
    };
    // Issue the copy of fragments [fs, fe) (fs a multiple of 4 = 16 bytes) into the stage; the
    // caller has made sure nobody still reads the old contents.  The bulk copies never read
    // past the arrays: the last < 4 fragments of the frame are copied by lanes.
    bool pend = false;                                   // warp-uniform: a bulk copy is in flight
    // (which of the two arrays is copied is a literal at every call site: testing the shared-memory
    // pointers against NULL instead costs a generic-address conversion per test)
    auto issue_fill = [&](const bool has_d, const bool has_c, float* dst_d, Packed* dst_c, uint32_t fs,
                          uint32_t fe) {
        __syncwarp();
        uint32_t n4 = (fe - fs + 3u) & ~3u;
        if (fs + n4 > A.F) {                             // the frame's last tile only
            n4 = (A.F - fs) & ~3u;
            const uint32_t rem = fe - fs > n4 ? fe - fs - n4 : 0u;
            if ((uint32_t)lane < rem) {
                NOIT_CHK_FRAGS(fs + n4 + lane, 1u);
                if (has_d) { NOIT_CHK_STAGE(dst_d + n4 + lane, 4u); dst_d[n4 + lane] = __ldg(A.depth + fs + n4 + lane); }
                if (has_c) { NOIT_CHK_STAGE(dst_c + n4 + lane, CB); dst_c[n4 + lane] = __ldg(g_rgba + fs + n4 + lane); }
            }
        }
        if (lane == 0 && n4) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(bar, n4 * ((has_d ? 4u : 0u) + (has_c ? CB : 0u)));
            NOIT_CHK_FRAGS(fs, n4);
            if (has_d) { NOIT_CHK_STAGE(dst_d, n4 * 4u); bulk_g2s(smem_u32(dst_d), A.depth + fs, n4 * 4u, bar); }
            if (has_c) { NOIT_CHK_STAGE(dst_c, n4 * CB); bulk_g2s(smem_u32(dst_c), g_rgba + fs, n4 * CB, bar); }
        }
        pend = n4 != 0;
    };
    auto wait_fill = [&]() {
        if (pend) {
            mbar_wait(bar, parity);
            parity ^= 1u;
            pend = false;
        }
        __syncwarp();
    };
    // First fill of a tile with offsets (a, b): light tile = depths and colours of all 32 lists,
    // heavy tile = depths of its first chunk of rounds.  Issued as soon as the previous tile
    // no longer needs the stage, i.e. BEFORE that tile's MLP, which hides the copy's latency.
    auto chunk_end = [&](const uint32_t (&B)[L + 1], int r, uint32_t cap, uint32_t& bk) -> int {
        int k = r + 1;                                   // greedy: rounds [r, k) fit `cap` fragments
        bk = B[r + 1];
#pragma unroll
        for (int c = 1; c < L; ++c)
            if (c > r && k == c && B[c + 1] - (B[r] & ~3u) <= cap) { k = c + 1; bk = B[c + 1]; }
        return k;
    };
    auto round_bounds = [&](uint32_t a, uint32_t te, uint32_t (&B)[L + 1]) -> bool {
#pragma unroll
        for (int r = 0; r < L; ++r) B[r] = __shfl_sync(0xffffffffu, a, r * PPR);
        B[L] = te;
        bool fits = true;                                // every round fits the colour stage
#pragma unroll
        for (int r = 0; r < L; ++r) fits = fits && (B[r + 1] - (B[r] & ~3u) <= kCapC);
        return fits;
    };
    auto first_fill = [&](uint32_t a, uint32_t b, bool depth_only_tile) {
        if (kMode == NOIT_RESOLVE_LIST) return;
        const uint32_t tb = __shfl_sync(0xffffffffu, a, 0), te = __shfl_sync(0xffffffffu, b, 31);
        const uint32_t fs = tb & ~3u;
        if (te <= tb) return;
        if (depth_only_tile && te - fs <= kCapD) {
            issue_fill(true, false, sD, nullptr, fs, te);
        } else if (te - fs <= kCap) {
            issue_fill(true, true, sD, sC2, fs, te);
        } else {
            uint32_t B[L + 1], bk;
            if (!round_bounds(a, te, B)) return;
            chunk_end(B, 0, kCapD, bk);
            if (bk > B[0]) issue_fill(true, false, sD, nullptr, fs, bk);
        }
    };

    // one tile per atomic (4 consecutive tiles per atomic measured slower, 204 vs 168 us: heavy
    // tiles cluster and the load imbalance costs more than the atomics)
    uint32_t t_cur = warp_id;
    uint32_t raw_nxt = warp_id + n_warps, raw_nn = warp_id + 2u * n_warps;   // then two atomics in flight
    uint32_t n_static = 2;                               // queued values that are tickets already
    uint32_t o0 = 0, o1 = 0, pix = 0;
    bool mixed = false;                                  // S7 / O7g: some pixel of the tile has lod > 0
    bool depth_only = false;                             // ... every pixel takes layer 2 AND tail coarse
    if (t_cur < num_tiles) {
        pix = lane_pixel(t_cur);
        load_offsets(pix, o0, o1);
        const uint32_t fl = tile_flags(t_cur);
        mixed = (fl & 1u) != 0;
        depth_only = (fl & 2u) != 0;
        first_fill(o0, o1, depth_only);
    }
    while (t_cur < num_tiles) {
        uint32_t t_nxt = __shfl_sync(0xffffffffu, raw_nxt, 0);
        // (the counter value becomes a ticket only here, behind the broadcast: nothing may depend
        // on the atomic's result in the tile that issued it)
        if (n_static) --n_static;
        else t_nxt = ((t_nxt << kCounterShift) | my_c) + 3u * n_warps;
        raw_nxt = raw_nn;
        raw_nn = fetch_raw();
        uint32_t no0 = 0, no1 = 0, npix = 0;
        uint32_t nflags = 0;
        if (t_nxt < num_tiles) {                         // lands while this tile runs
            npix = lane_pixel(t_nxt);
            load_offsets(npix, no0, no1);
            nflags = tile_flags(t_nxt);
        }

        Owned<ColorT> own;
        own.c1 = own.c2 = Color<ColorT>::zero();
        own.d1 = 1.0f; own.n = 0;
        own.acc_r = own.acc_g = own.acc_b = own.a_tail = 0.f; own.t_tail = 1.f;
        own.sum_r = own.sum_g = own.sum_b = 0.f;
        uint32_t px_own = lane;                          // pixel of the tile this lane ends up owning

        // inputs of the epilogue
        float xf[5];
        float4 e_c1 = make_float4(0.f, 0.f, 0.f, 0.f), e_l2 = e_c1;
        float e_d1 = 1.0f, e_tt = 1.0f;
        bool has_tail = false;

        const uint32_t tb = __shfl_sync(0xffffffffu, o0, 0), te = __shfl_sync(0xffffffffu, o1, 31);
        const uint32_t fs = tb & ~3u;
        if (kMode == NOIT_RESOLVE_LIST) {
            // ---- S9: 32/L scattered pixels, L lanes per pixel straight from global memory (one
            // round: the lists are scattered, so the work is latency-bound and small tiles keep
            // every warp of the machine busy); lanes with lane % L == 0 own a pixel
            px_own = (uint32_t)(lane / L);
            own = tile_from_global<ColorT, L, 1>(lane, o0, o1, A.depth, g_rgba);
        } else if (kCoarse && depth_only && te - fs <= kCapD) {
            // ---- S7 / O7g tile whose 32 pixels all take layer 2 and the tail from a coarse buffer:
            // only layer 1 is needed from the full-resolution lists, so only the DEPTHS are
            // staged (4 of the 12 bytes per fragment) and the winner's colour is fetched directly
            if (te > tb) {
                wait_fill();
                NOIT_CHK_STAGE(sD + (o0 - fs), (o1 - o0) * 4u);
                const Top2 s = scan_depths<1>(sD, o0 - fs, o1 - fs);
                if (s.i1 != NOIT_ABSENT) { NOIT_CHK_FRAGS(fs + s.i1, 1u); own.c1 = __ldg(g_rgba + fs + s.i1); }
                own.d1 = s.d1;
                own.n = o1 - o0;
            }
        } else if (te - fs <= kCap) {
            // ---- light tile: one lane per pixel, depths and colours staged together
            if (te > tb) {
                wait_fill();                             // issued before the previous tile's MLP
                const uint32_t first = o0 - fs, end = o1 - fs;
                NOIT_CHK_STAGE(sD + first, (end - first) * 4u);
                NOIT_CHK_STAGE(sC2 + first, (end - first) * CB);
                const Top2 s = scan_depths<1>(sD, first, end);
                if (s.i1 != NOIT_ABSENT) {
                    NOIT_CHK_STAGE(sC2 + s.i1, CB);
                    own.c1 = sC2[s.i1];
                    if (kFeat10) Color<ColorT>::zero_all(&sC2[s.i1]);
                    else Color<ColorT>::zero_alpha(&sC2[s.i1]);
                }
                if (s.i2 != NOIT_ABSENT) {
                    NOIT_CHK_STAGE(sC2 + s.i2, CB);
                    own.c2 = sC2[s.i2];
                    if (kFeat10) Color<ColorT>::zero_all(&sC2[s.i2]);
                    else Color<ColorT>::zero_alpha(&sC2[s.i2]);
                }
                const Sums z = scan_colours<ColorT, 1, kFeat10>(sC2, first, end);    // own list only: no sync
                own.d1 = s.d1;
                own.n = o1 - o0;
                own.acc_r = z.r; own.acc_g = z.g; own.acc_b = z.b; own.a_tail = z.a; own.t_tail = z.t;
                own.sum_r = z.cr; own.sum_g = z.cg; own.sum_b = z.cb;
            }
        } else {
            // ---- heavy tile: L lanes per pixel, L rounds of PPR pixels
            const int g = lane / L, q = lane % L;
            px_own = (uint32_t)(q * PPR + g);
            uint32_t B[L + 1];                           // fragment bounds of the rounds
            const bool fits = round_bounds(o0, te, B);
            if (!fits) {
                own = tile_from_global<ColorT, L, L, kFeat10>(lane, o0, o1, A.depth, g_rgba);
            } else {
                Top2 t2[L];
                uint32_t first[L], end[L];
                int staged_to = 0;
                const float* Dv = sD;                    // staged depths, indexed by fragment index
#pragma unroll
                for (int r = 0; r < L; ++r) {
                    if (r == staged_to) {                // stage the next chunk of rounds (depths)
                        uint32_t bk;
                        const int k = chunk_end(B, r, kCapD, bk);
                        const uint32_t base = B[r] & ~3u;
                        if (r > 0 && bk > B[r]) issue_fill(true, false, sD, nullptr, base, bk);   // r == 0: first_fill
                        wait_fill();
                        Dv = sD - base;
                        staged_to = k;
                    }
                    const int px = r * PPR + g;
                    first[r] = __shfl_sync(0xffffffffu, o0, px) + q;
                    end[r] = __shfl_sync(0xffffffffu, o1, px);
                    if (end[r] > first[r]) NOIT_CHK_STAGE(Dv + first[r], (end[r] - first[r]) * 4u);
                    t2[r] = scan_depths<L>(Dv, first[r], end[r]);
                }
                transposed_merge<L>(t2, q);              // t2[0]: this lane's pixel, global indices
                Sums sm[L];
                staged_to = 0;
                Packed* Cv = sC;
#pragma unroll
                for (int r = 0; r < L; ++r) {
                    if (r == staged_to) {                // stage the next chunk of rounds (colours)
                        uint32_t bk;
                        const int k = chunk_end(B, r, kCapC, bk);
                        const uint32_t base = B[r] & ~3u;
                        if (bk > B[r]) issue_fill(false, true, nullptr, sC, base, bk);
                        wait_fill();
                        Cv = sC - base;
                        if (q >= r && q < k) {           // owners of the chunk's rounds
                            if (t2[0].i1 != NOIT_ABSENT) {
                                NOIT_CHK_STAGE(Cv + t2[0].i1, CB);
                                own.c1 = Cv[t2[0].i1];
                                if (kFeat10) Color<ColorT>::zero_all(&Cv[t2[0].i1]);
                                else Color<ColorT>::zero_alpha(&Cv[t2[0].i1]);
                            }
                            if (t2[0].i2 != NOIT_ABSENT) {
                                NOIT_CHK_STAGE(Cv + t2[0].i2, CB);
                                own.c2 = Cv[t2[0].i2];
                                if (kFeat10) Color<ColorT>::zero_all(&Cv[t2[0].i2]);
                                else Color<ColorT>::zero_alpha(&Cv[t2[0].i2]);
                            }
                        }
                        __syncwarp();
                        staged_to = k;
                    }
                    if (end[r] > first[r]) NOIT_CHK_STAGE(Cv + first[r], (end[r] - first[r]) * CB);
                    sm[r] = scan_colours<ColorT, L, kFeat10>(Cv, first[r], end[r]);
                }
                transposed_sum<L, kFeat10>(sm, q);
                own.d1 = t2[0].d1;
                own.n = __shfl_sync(0xffffffffu, o1 - o0, (int)px_own);
                own.acc_r = sm[0].r; own.acc_g = sm[0].g; own.acc_b = sm[0].b;
                own.a_tail = sm[0].a; own.t_tail = sm[0].t;
                own.sum_r = sm[0].cr; own.sum_g = sm[0].cg; own.sum_b = sm[0].cb;
            }
        }
        // the stage is free: start the next tile's first fill, then do this tile's MLP
        // the MLP's packed weights (L1-resident) are requested before the fill is issued, so they
        // are in registers when the MLP starts
        float4 wv[NOIT_MMA_CHUNKS];
        if (kMma && !kWeightsInSmem) {
#pragma unroll
            for (int v = 0; v < NOIT_MMA_CHUNKS; ++v) wv[v] = __ldg(A.mlp_packed + v * 32 + lane);
        }
        const bool nmixed = (nflags & 1u) != 0, ndepth_only = (nflags & 2u) != 0;
        if (t_nxt < num_tiles) first_fill(no0, no1, ndepth_only);
        // ---- every lane now owns one pixel: features (O3), MLP (O4), composite (O5)
        uint32_t p = __shfl_sync(0xffffffffu, pix, (int)px_own);
        if (kMode == NOIT_RESOLVE_LIST && (lane % L) != 0) p = 0xFFFFFFFFu;   // not an owner
        {
            float f[3];
            {
                // O3 with one IEEE reciprocal instead of three divisions
                has_tail = own.a_tail > 0.f;
                const float inv = has_tail ? 1.0f / own.a_tail : 0.f;
                xf[0] = (float)own.n; xf[1] = own.t_tail;
                xf[2] = own.acc_r * inv; xf[3] = own.acc_g * inv; xf[4] = own.acc_b * inv;
                const float4 c2 = Color<ColorT>::unpack(own.c2);
                e_c1 = Color<ColorT>::unpack(own.c1);
                e_l2 = make_float4(c2.w * c2.x, c2.w * c2.y, c2.w * c2.z, c2.w);
                e_d1 = own.n ? own.d1 : 1.0f;
                e_tt = own.t_tail;
            }
            if (kCoarse && mixed && p < A.P) {
                // S7 / O7g: layer 2 and / or the raw tail accumulators of this pixel come from a
                // coarse buffer's G, bilinearly sampled at the pixel centre; layer 1 stays
                // the full-resolution one
                int plevel;
                const int plod = lane_lod(p, plevel);                // of the OWNED pixel
                const int y = (int)(p / (uint32_t)A.W), x = (int)(p - (uint32_t)y * (uint32_t)A.W);
                float G2[10], G3[10];
                if (kGlobal) {                                       // frame-global lods, image clamp
                    if (g_lod2 > 0)
                        sample_coarse_g(A.coarse_g[g_lod2 - 1], A.coarse_w[g_lod2 - 1], A.coarse_h[g_lod2 - 1],
                                        g_lod2, 30, x, y, G2);
                    if (g_lod3 > 0 && g_lod3 != g_lod2)
                        sample_coarse_g(A.coarse_g[g_lod3 - 1], A.coarse_w[g_lod3 - 1], A.coarse_h[g_lod3 - 1],
                                        g_lod3, 30, x, y, G3);
                    if (g_lod2 > 0) e_l2 = make_float4(G2[0], G2[1], G2[2], G2[3]);
                    if (g_lod3 > 0) {
                        const float* T = g_lod3 == g_lod2 ? G2 : G3;
                        has_tail = make_features(T[9], T[8], T[4], T[5], T[6], T[7], xf);
                        e_tt = T[8];
                    }
                } else if (plod > 0) {                               // per-tile lod, leaf clamp
                    sample_coarse_g(A.coarse_g[plod - 1], A.coarse_w[plod - 1], A.coarse_h[plod - 1],
                                    plod, 6 - plevel, x, y, G2);
                    e_l2 = make_float4(G2[0], G2[1], G2[2], G2[3]);
                    has_tail = make_features(G2[9], G2[8], G2[4], G2[5], G2[6], G2[7], xf);
                    e_tt = G2[8];
                }
            }
            if constexpr (kFeat10) {
                // O12 (A29): x = [two-layer "over" blend (3), C_avg (3), alpha_avg, C_acc (3)],
                // averages over the m = max(n - 2, 0) tail fragments; the sigmoid network predicts the
                // whole transparency colour; Eq. 3: C_p = C_t + C_b prod (1 - alpha_i)
                const uint32_t m = own.n > 2u ? own.n - 2u : 0u;
                const float inv_m = m ? 1.0f / (float)m : 0.f;
                const float t1 = 1.f - e_c1.w;
                float x10[10];
                x10[0] = fmaf(t1, e_l2.x, e_c1.w * e_c1.x);
                x10[1] = fmaf(t1, e_l2.y, e_c1.w * e_c1.y);
                x10[2] = fmaf(t1, e_l2.z, e_c1.w * e_c1.z);
                x10[3] = own.sum_r * inv_m; x10[4] = own.sum_g * inv_m; x10[5] = own.sum_b * inv_m;
                x10[6] = own.a_tail * inv_m;
                x10[7] = own.acc_r; x10[8] = own.acc_g; x10[9] = own.acc_b;
                mlp10_forward_packed(W, x10, f);
                if (p < A.P) {
                    if (A.features10) {
#pragma unroll
                        for (int k = 0; k < 10; k += 2)
                            *reinterpret_cast<float2*>(A.features10 + 10 * (size_t)p + k) = make_float2(x10[k], x10[k + 1]);
                    }
                    const float keep = own.n ? 1.f : 0.f;            // an empty pixel has no transparency colour
                    const float ct_r = keep * f[0], ct_g = keep * f[1], ct_b = keep * f[2];
                    const float t_tot = t1 * (1.f - e_l2.w) * e_tt;
                    if (A.out_trans)
                        __stcs(reinterpret_cast<float4*>(A.out_trans) + p, make_float4(ct_r, ct_g, ct_b, t_tot));
                    if (A.out_final)
                        __stcs(reinterpret_cast<float4*>(A.out_final) + p,
                               make_float4(fmaf(t_tot, A.bg[0], ct_r), fmaf(t_tot, A.bg[1], ct_g),
                                           fmaf(t_tot, A.bg[2], ct_b), 1.f - t_tot));
                    if (A.out_depth1) __stcs(A.out_depth1 + p, e_d1);
                }
            } else {
                if (kMma) {                                          // all 32 lanes
                    if (kWeightsInSmem) mlp_forward_mma(MmaWeightsSmem{wsm + lane}, scratch, lane, xf, f);
                    else mlp_forward_mma(MmaWeightsReg{wv}, scratch, lane, xf, f);
                }
                else mlp_forward_packed(W, xf, f);
                if (p < A.P) composite_store(A, p, e_c1, e_l2, e_d1, has_tail, f, e_tt);
            }
        }
        pix = npix; mixed = nmixed; depth_only = ndepth_only;
        t_cur = t_nxt; o0 = no0; o1 = no1;
    }
    // the last warp to finish re-arms the counters for the next launch
    // (the fence orders this warp's outstanding, result-unused ticket atomics before its finish
    // ticket, so no late add can land after the reset)
    uint32_t last = 0;
    if (lane == 0) {
        __threadfence();
        last = atomicAdd(A.tile_counter + 1, 1u) == gridDim.x * kWarpsPerCta - 1u ? 1u : 0u;
    }
    if (__shfl_sync(0xffffffffu, last, 0)) {
        for (uint32_t c = lane; c < (1u << kCounterShift); c += 32u) A.tile_counter[64u + 32u * c] = 0u;
        if (lane == 0) A.tile_counter[1] = 0u;
    }
}

template <typename ColorT, int L, bool kMma, int kMode, typename WT = MlpWeightsT>
static noit_status launch_staged(noit_ctx* ctx, const ResolveArgs& A, cudaStream_t st, const WT* w10 = nullptr)
{
    const size_t stage = kMode == NOIT_RESOLVE_LIST ? 0 : (size_t)kStageBytesFrame;
    const size_t smem = kWarpsPerCta * stage + kWarpsPerCta * sizeof(uint64_t) +
                        kWarpsPerCta * kScratchFloats * sizeof(float) + (kMma ? kWeightBytes : 0) +
                        (kMode == NOIT_RESOLVE_LIST ? 0 : NOIT_X_PAD);
    // the shared-memory attribute and the occupancy are per device (and per instantiation)
    static int per_sm_dev[64] = {0};
    const int dev = ctx->device >= 0 && ctx->device < 64 ? ctx->device : 0;
    if (per_sm_dev[dev] == 0) {
        NOIT_CUDA(ctx, cudaFuncSetAttribute(resolve_staged_kernel<ColorT, L, kMma, kMode, WT>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int q = 0;
        NOIT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                           &q, resolve_staged_kernel<ColorT, L, kMma, kMode, WT>, kWarpsPerCta * 32, smem));
        per_sm_dev[dev] = q < 1 ? -1 : q;
    }
    const int per_sm = per_sm_dev[dev];
    if (per_sm < 1) return noit_fail(ctx, NOIT_ERR_CUDA, "resolve_staged_kernel does not fit an SM");
    // S9 reads its tile count on the device: the persistent grid is sized for the machine
    const uint32_t want = kMode == NOIT_RESOLVE_LIST ? 0xFFFFFFFFu
                                                     : (A.num_tiles + kWarpsPerCta - 1) / kWarpsPerCta;
    const uint32_t grid = min((uint32_t)(ctx->num_sms * per_sm), max(want, 1u));
    if constexpr (sizeof(WT) == sizeof(MlpWeights10T))
        resolve_staged_kernel<ColorT, L, kMma, kMode, WT><<<grid, kWarpsPerCta * 32, smem, st>>>(A, *w10);
    else
        resolve_staged_kernel<ColorT, L, kMma, kMode, WT><<<grid, kWarpsPerCta * 32, smem, st>>>(A, ctx->wt);
    ctx->launches += 1;
    const cudaError_t e = cudaGetLastError();
    // a failed launch may leave the self-re-arming counters armed: zero them for the next call
    if (e != cudaSuccess) cudaMemsetAsync(ctx->d_counters, 0, NOIT_COUNTER_WORDS * sizeof(uint32_t), st);
    NOIT_CUDA(ctx, e);
    return NOIT_OK;
}

template <typename ColorT, int kMode>
static noit_status launch_mode(noit_ctx* ctx, const ResolveArgs& A, cudaStream_t st)
{
    // bf16-rounded weights are exact in TF32: the MLP runs on the tensor cores (two-pass split
    // of the activations, fp32-class accuracy); fp32 weights keep the FFMA2 form.
    const bool mma = ctx->precision == NOIT_MLP_BF16 && ctx->d_mlp != nullptr;
    // lanes per pixel: 4 for frames; 2 for the pixel list (16 listed pixels per warp tile).  Measured on
    // cfg3 with lists of 0.5 / 1.7 / 5 / 20 % of the pixels (profiles/r02_launches.md): 8 lanes
    // 18.4 / 31.8 / 56.1 / 163.9 us, 4 lanes 21.0 / 29.7 / 43.2 / 105.4, 2 lanes 23.9 / 25.7 / 41.2 / 91.6,
    // 1 lane 31.3 / 33.0 / 45.4 / 112.3: with scattered lists the chain offsets -> depths -> colours ->
    // network is latency, and fewer, fuller tiles mean fewer of those chains per warp.
    constexpr int L = kMode == NOIT_RESOLVE_LIST ? NOIT_X_LIST_L : 4;
    // S9 is bound by the latency chain of its few scattered tiles, not by issue slots: the FFMA2
    // MLP needs 40 registers fewer than the tensor-core one, which with no stage allocated
    // gives 7 CTAs per SM instead of 4 and so fewer tiles in sequence per warp
    if (kMode == NOIT_RESOLVE_LIST) return launch_staged<ColorT, L, false, kMode>(ctx, A, st);
    return mma ? launch_staged<ColorT, L, true, kMode>(ctx, A, st)
               : launch_staged<ColorT, L, false, kMode>(ctx, A, st);
}

noit_status noit_launch_resolve_staged(noit_ctx* ctx, const ResolveArgs& A0, int color_fmt, int mode,
                                       cudaStream_t st)
{
    ResolveArgs A = A0;
    A.num_tiles = (A.P + 31u) / 32u;
    A.tile_counter = ctx->d_counters;
    A.mlp_packed = static_cast<const float4*>(ctx->d_mlp);
    const bool f16 = color_fmt == NOIT_RGBA_F16;
    switch (mode) {
    case NOIT_RESOLVE_LIST:
        return f16 ? launch_mode<__half, NOIT_RESOLVE_LIST>(ctx, A, st)
                   : launch_mode<float, NOIT_RESOLVE_LIST>(ctx, A, st);
    case NOIT_RESOLVE_ADAPTIVE:
        return f16 ? launch_mode<__half, NOIT_RESOLVE_ADAPTIVE>(ctx, A, st)
                   : launch_mode<float, NOIT_RESOLVE_ADAPTIVE>(ctx, A, st);
    case NOIT_RESOLVE_GLOBAL:
        return f16 ? launch_mode<__half, NOIT_RESOLVE_GLOBAL>(ctx, A, st)
                   : launch_mode<float, NOIT_RESOLVE_GLOBAL>(ctx, A, st);
    default:
        return f16 ? launch_mode<__half, NOIT_RESOLVE_ALL>(ctx, A, st)
                   : launch_mode<float, NOIT_RESOLVE_ALL>(ctx, A, st);
    }
}

// NEXT-4 (O12): the DFAOIT resolve of a whole frame -- same kernel, ten-feature epilogue
noit_status noit_launch_resolve_dfaoit(noit_ctx* ctx, const ResolveArgs& A0, int color_fmt,
                                       const MlpWeights10T& w10, cudaStream_t st)
{
    ResolveArgs A = A0;
    A.num_tiles = (A.P + 31u) / 32u;
    A.tile_counter = ctx->d_counters;
    A.mlp_packed = nullptr;
    return color_fmt == NOIT_RGBA_F16
               ? launch_staged<__half, 4, false, NOIT_RESOLVE_ALL, MlpWeights10T>(ctx, A, st, &w10)
               : launch_staged<float, 4, false, NOIT_RESOLVE_ALL, MlpWeights10T>(ctx, A, st, &w10);
}
