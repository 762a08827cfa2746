// noit_resolve_staged.cu -- the plain fused resolve (S1-S5, Eq. 4) of a whole frame:
// persistent warps, fragment ranges staged into shared memory by 1-D TMA bulk copies
// (cp.async.bulk + mbarrier), L lanes per pixel, MLP with packed FFMA2.
//
// Why this shape (ncu evidence in profiles/r01_*): a thread-per-pixel kernel that reads its
// list straight from global memory is bound by L1 data-stage wavefronts (every lane of a load
// touches a different 128-byte line: 12.5 wavefronts per request, 74 % of the LSU data pipe at
// 48 % of the HBM roofline) and by its instruction count (36 per fragment, ~1000 per MLP).
// Here
//   * a WARP owns a tile of 32 consecutive pixels; their CSR lists are one contiguous fragment
//     range, which lane 0 copies into the warp's private shared-memory stage with two bulk
//     copies (depth, colour) that complete on the warp's mbarrier: no LSU wavefronts, no
//     registers, fully coalesced HBM reads;
//   * the tile is processed in L rounds of 32/L pixels with L lanes per pixel: lane q of a
//     group reads fragments b+q, b+q+L, ... so a warp-wide shared-memory load reads 32/L runs of
//     L consecutive words (few bank conflicts whatever the list lengths are, no alignment
//     peeling), and the loop trip count is max over 32/L pixels of ceil(n/L);
//   * selection and reduction are two passes over the staged list: pass 1 tracks
//     (d1,i1,d2,i2) on the depths only; the group merges its partial top-2 under the key
//     (depth, index) (O1); the owner lane fetches the two layer colours and overwrites their
//     alpha with 0 in the stage; pass 2 then accumulates EVERY staged fragment of the pixel
//     (a zero alpha adds 0 and multiplies by 1), so the tail is never "all minus top-2" (O2);
//   * after L rounds every lane owns one pixel: features, MLP (FFMA2: two output neurons per
//     instruction, same summation order as the scalar form), composite, 128-bit stores.
// Tiles are handed out by an atomic counter (fragment counts vary 0..128 per pixel), which the
// last warp to finish resets, so a launch needs no memset.
#include "noit_resolve_common.cuh"

namespace {

constexpr uint32_t kCap = 1032;          // fragments per warp stage: 8 px * 128 + alignment slack
constexpr int kWarpsPerCta = 4;

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
};
template <> struct Color<float> {
    typedef float4 Packed;
    static constexpr uint32_t kBytes = 16;
    static __device__ __forceinline__ Packed zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }
    static __device__ __forceinline__ float4 unpack(Packed v) { return v; }
    static __device__ __forceinline__ void zero_alpha(Packed* slot) { slot->w = 0.f; }
    static __device__ __forceinline__ Packed zero_alpha_reg(Packed v) { v.w = 0.f; return v; }
};

// key (depth, index) lexicographic (O1)
__device__ __forceinline__ bool key_less(float da, uint32_t ia, float db, uint32_t ib)
{
    return da < db || (da == db && ia < ib);
}

}  // namespace

// ------------------------------------------------------------------------------------------
// the kernel
// ------------------------------------------------------------------------------------------
// One warp's private stage.
template <typename ColorT>
struct WarpStage {
    float depth[kCap];
    typename Color<ColorT>::Packed rgba[kCap];
};

// Per-lane results of the rounds: after round r the lanes with (lane % L) == r own pixel
// r*(32/L) + lane/L of the tile.
template <typename ColorT>
struct Owned {
    typename Color<ColorT>::Packed c1, c2;
    float d1;
    uint32_t n;
    float acc_r, acc_g, acc_b, a_tail, t_tail;
};

// One round: pixels r*PPR .. r*PPR+PPR-1 of the tile, L lanes each.  D / C point at fragment
// `base` (shared-memory stage when kStaged, global arrays with base = 0 otherwise).  Fragments
// are addressed by their position relative to `base`; positions order like fragment indices.
template <typename ColorT, int L, bool kStaged>
__device__ __forceinline__ void resolve_round_body(int r, int lane, uint32_t o0, uint32_t o1,
                                                   const float* D, typename Color<ColorT>::Packed* C,
                                                   uint32_t base, Owned<ColorT>& own)
{
    typedef typename Color<ColorT>::Packed Packed;
    constexpr int PPR = 32 / L;
    const int g = lane / L, q = lane % L;
    const int px = r * PPR + g;
    const uint32_t b = __shfl_sync(0xffffffffu, o0, px), e = __shfl_sync(0xffffffffu, o1, px);
    const uint32_t first = b - base + q, end = e - base;

    // ---- pass 1: partial top-2 over this lane's fragments, in increasing index order, so a
    // newcomer wins a slot only on a strictly smaller depth (ties keep the earlier index, O1)
    float d1 = __int_as_float(0x7f800000), d2 = d1;
    uint32_t i1 = NOIT_ABSENT, i2 = NOIT_ABSENT;
    auto step1 = [&](float d, uint32_t pos) {
        const bool lt1 = d < d1, lt2 = d < d2;
        i2 = lt1 ? i1 : (lt2 ? pos : i2);
        d2 = lt1 ? d1 : (lt2 ? d : d2);
        i1 = lt1 ? pos : i1;
        d1 = lt1 ? d : d1;
    };
    {
        uint32_t pos = first;
#pragma unroll 1
        for (; pos + L < end; pos += 2 * L) {
            const float da = D[pos], db = D[pos + L];
            step1(da, pos);
            step1(db, pos + L);
        }
        if (pos < end) step1(D[pos], pos);
    }
    // ---- merge the L partial results (butterfly: every lane of the group ends with the result)
#pragma unroll
    for (int s = 1; s < L; s <<= 1) {
        const float od1 = __shfl_xor_sync(0xffffffffu, d1, s), od2 = __shfl_xor_sync(0xffffffffu, d2, s);
        const uint32_t oi1 = __shfl_xor_sync(0xffffffffu, i1, s), oi2 = __shfl_xor_sync(0xffffffffu, i2, s);
        const bool mine = key_less(d1, i1, od1, oi1);
        // x = runner-up of the winning side, y = best of the losing side
        const float xd = mine ? d2 : od2, yd = mine ? od1 : d1;
        const uint32_t xi = mine ? i2 : oi2, yi = mine ? oi1 : i1;
        d1 = mine ? d1 : od1;
        i1 = mine ? i1 : oi1;
        const bool xy = key_less(xd, xi, yd, yi);
        d2 = xy ? xd : yd;
        i2 = xy ? xi : yi;
    }
    // ---- the owner lane fetches the two layers; their alpha is then neutralised for pass 2
    const bool owner = q == r;
    Packed c1 = Color<ColorT>::zero(), c2 = Color<ColorT>::zero();
    if (owner) {
        if (i1 != NOIT_ABSENT) {
            c1 = C[i1];
            if (kStaged) Color<ColorT>::zero_alpha(&C[i1]);
        }
        if (i2 != NOIT_ABSENT) {
            c2 = C[i2];
            if (kStaged) Color<ColorT>::zero_alpha(&C[i2]);
        }
    }
    if (kStaged) __syncwarp();
    // ---- pass 2: tail accumulators over every fragment of the pixel (layers carry alpha 0)
    float ar = 0.f, ag = 0.f, ab = 0.f, at = 0.f, tt = 1.f;
    auto step2 = [&](Packed raw, uint32_t pos) {
        if (!kStaged && (pos == i1 || pos == i2)) raw = Color<ColorT>::zero_alpha_reg(raw);
        const float4 c = Color<ColorT>::unpack(raw);
        ar = fmaf(c.w, c.x, ar);
        ag = fmaf(c.w, c.y, ag);
        ab = fmaf(c.w, c.z, ab);
        at += c.w;
        tt = fmaf(-c.w, tt, tt);                       // tt *= (1 - alpha), one rounding
    };
    {
        uint32_t pos = first;
#pragma unroll 1
        for (; pos + L < end; pos += 2 * L) {
            const Packed ra = C[pos], rb = C[pos + L];
            step2(ra, pos);
            step2(rb, pos + L);
        }
        if (pos < end) step2(C[pos], pos);
    }
#pragma unroll
    for (int s = 1; s < L; s <<= 1) {
        ar += __shfl_xor_sync(0xffffffffu, ar, s);
        ag += __shfl_xor_sync(0xffffffffu, ag, s);
        ab += __shfl_xor_sync(0xffffffffu, ab, s);
        at += __shfl_xor_sync(0xffffffffu, at, s);
        tt *= __shfl_xor_sync(0xffffffffu, tt, s);
    }
    if (owner) {
        own.c1 = c1; own.c2 = c2;
        own.d1 = d1;
        own.n = e - b;
        own.acc_r = ar; own.acc_g = ag; own.acc_b = ab; own.a_tail = at; own.t_tail = tt;
    }
}

template <typename ColorT, int L>
__device__ __forceinline__ void resolve_round_staged(int r, int lane, uint32_t o0, uint32_t o1,
                                                     WarpStage<ColorT>* stage, uint32_t base,
                                                     Owned<ColorT>& own)
{
    resolve_round_body<ColorT, L, true>(r, lane, o0, o1, stage->depth, stage->rgba, base, own);
}
// cold path: a round whose fragments do not fit the stage reads global memory directly
template <typename ColorT, int L>
__device__ __noinline__ Owned<ColorT> resolve_round_global(int r, int lane, uint32_t o0, uint32_t o1,
                                                           const float* depth,
                                                           typename Color<ColorT>::Packed* rgba,
                                                           Owned<ColorT> own)
{
    resolve_round_body<ColorT, L, false>(r, lane, o0, o1, depth, rgba, 0u, own);
    return own;
}

// A whole tile whose fragments are staged at once (the common case): pass 1 of all L rounds,
// ONE transposed butterfly that leaves lane q of each group with the merged top-2 of the
// group's round-q pixel (log2(L) exchange steps that halve the items a lane holds, instead of
// L full butterflies), layer fetch + alpha neutralisation, one __syncwarp, pass 2 of all L
// rounds, one transposed butterfly of the five sums.  Lane (g, q) ends up owning pixel
// q*(32/L) + g.
template <typename ColorT, int L>
__device__ __forceinline__ void resolve_tile_staged(int lane, uint32_t o0, uint32_t o1,
                                                    WarpStage<ColorT>* stage, uint32_t base,
                                                    Owned<ColorT>& own)
{
    typedef typename Color<ColorT>::Packed Packed;
    constexpr int PPR = 32 / L;
    const int g = lane / L, q = lane % L;
    const float* D = stage->depth;
    Packed* C = stage->rgba;
    float d1[L], d2[L];
    uint32_t i1[L], i2[L], first[L], end[L];
#pragma unroll
    for (int r = 0; r < L; ++r) {
        const int px = r * PPR + g;
        const uint32_t b = __shfl_sync(0xffffffffu, o0, px), e = __shfl_sync(0xffffffffu, o1, px);
        first[r] = b - base + q;
        end[r] = e - base;
        float a1 = __int_as_float(0x7f800000), a2 = a1;
        uint32_t j1 = NOIT_ABSENT, j2 = NOIT_ABSENT;
        auto step1 = [&](float d, uint32_t pos) {
            const bool lt1 = d < a1, lt2 = d < a2;
            j2 = lt1 ? j1 : (lt2 ? pos : j2);
            a2 = lt1 ? a1 : (lt2 ? d : a2);
            j1 = lt1 ? pos : j1;
            a1 = lt1 ? d : a1;
        };
        uint32_t pos = first[r];
#pragma unroll 1
        for (; pos + L < end[r]; pos += 2 * L) {
            const float da = D[pos], db = D[pos + L];
            step1(da, pos);
            step1(db, pos + L);
        }
        if (pos < end[r]) step1(D[pos], pos);
        d1[r] = a1; d2[r] = a2; i1[r] = j1; i2[r] = j2;
    }
    // transposed butterfly: at step m the live slots are [0, 2m); a lane with bit m of q clear
    // keeps slot r and sends slot r + m (r < m), its partner q ^ m does the opposite; both
    // slots hold the same two items on both lanes, the merged item goes to slot r.  After the
    // last step slot 0 holds item (round) q.
#pragma unroll
    for (int m = L / 2; m >= 1; m >>= 1) {
        const bool up = (q & m) != 0;
#pragma unroll
        for (int r = 0; r < L; ++r) {
            if (r >= m) continue;       // live slots are [0, 2m): pair slot r with slot r + m
            const int rk0 = r, rk1 = r + m;
            // keep = up ? item[rk1] : item[rk0];  send = up ? item[rk0] : item[rk1]
            const float kd1 = up ? d1[rk1] : d1[rk0], kd2 = up ? d2[rk1] : d2[rk0];
            const uint32_t ki1 = up ? i1[rk1] : i1[rk0], ki2 = up ? i2[rk1] : i2[rk0];
            const float sd1 = up ? d1[rk0] : d1[rk1], sd2 = up ? d2[rk0] : d2[rk1];
            const uint32_t si1 = up ? i1[rk0] : i1[rk1], si2 = up ? i2[rk0] : i2[rk1];
            const float od1 = __shfl_xor_sync(0xffffffffu, sd1, m), od2 = __shfl_xor_sync(0xffffffffu, sd2, m);
            const uint32_t oi1 = __shfl_xor_sync(0xffffffffu, si1, m), oi2 = __shfl_xor_sync(0xffffffffu, si2, m);
            const bool mine = key_less(kd1, ki1, od1, oi1);
            const float xd = mine ? kd2 : od2, yd = mine ? od1 : kd1;
            const uint32_t xi = mine ? ki2 : oi2, yi = mine ? oi1 : ki1;
            const bool xy = key_less(xd, xi, yd, yi);
            // the merged item is stored in slot rk0 (slot index with bit m cleared)
            d1[rk0] = mine ? kd1 : od1;
            i1[rk0] = mine ? ki1 : oi1;
            d2[rk0] = xy ? xd : yd;
            i2[rk0] = xy ? xi : yi;
        }
    }
    // slot 0 now holds the merged top-2 of pixel q*PPR + g
    Packed c1 = Color<ColorT>::zero(), c2 = Color<ColorT>::zero();
    if (i1[0] != NOIT_ABSENT) {
        c1 = C[i1[0]];
        Color<ColorT>::zero_alpha(&C[i1[0]]);
    }
    if (i2[0] != NOIT_ABSENT) {
        c2 = C[i2[0]];
        Color<ColorT>::zero_alpha(&C[i2[0]]);
    }
    __syncwarp();
    float ar[L], ag[L], ab[L], at[L], tt[L];
#pragma unroll
    for (int r = 0; r < L; ++r) {
        float xr = 0.f, xg = 0.f, xb = 0.f, xa = 0.f, xt = 1.f;
        auto step2 = [&](Packed raw) {
            const float4 c = Color<ColorT>::unpack(raw);
            xr = fmaf(c.w, c.x, xr);
            xg = fmaf(c.w, c.y, xg);
            xb = fmaf(c.w, c.z, xb);
            xa += c.w;
            xt = fmaf(-c.w, xt, xt);                   // xt *= (1 - alpha), one rounding
        };
        uint32_t pos = first[r];
#pragma unroll 1
        for (; pos + L < end[r]; pos += 2 * L) {
            const Packed ra = C[pos], rb = C[pos + L];
            step2(ra);
            step2(rb);
        }
        if (pos < end[r]) step2(C[pos]);
        ar[r] = xr; ag[r] = xg; ab[r] = xb; at[r] = xa; tt[r] = xt;
    }
#pragma unroll
    for (int m = L / 2; m >= 1; m >>= 1) {
        const bool up = (q & m) != 0;
#pragma unroll
        for (int r = 0; r < L; ++r) {
            if (r >= m) continue;
            const int rk0 = r, rk1 = r + m;
            const float sr = up ? ar[rk0] : ar[rk1], sg = up ? ag[rk0] : ag[rk1];
            const float sb = up ? ab[rk0] : ab[rk1], sa = up ? at[rk0] : at[rk1];
            const float st = up ? tt[rk0] : tt[rk1];
            ar[rk0] = (up ? ar[rk1] : ar[rk0]) + __shfl_xor_sync(0xffffffffu, sr, m);
            ag[rk0] = (up ? ag[rk1] : ag[rk0]) + __shfl_xor_sync(0xffffffffu, sg, m);
            ab[rk0] = (up ? ab[rk1] : ab[rk0]) + __shfl_xor_sync(0xffffffffu, sb, m);
            at[rk0] = (up ? at[rk1] : at[rk0]) + __shfl_xor_sync(0xffffffffu, sa, m);
            tt[rk0] = (up ? tt[rk1] : tt[rk0]) * __shfl_xor_sync(0xffffffffu, st, m);
        }
    }
    own.c1 = c1; own.c2 = c2;
    own.d1 = d1[0];
    own.n = __shfl_sync(0xffffffffu, o1 - o0, q * PPR + g);
    own.acc_r = ar[0]; own.acc_g = ag[0]; own.acc_b = ab[0]; own.a_tail = at[0]; own.t_tail = tt[0];
}

template <typename ColorT, int L>
__global__ void __launch_bounds__(kWarpsPerCta * 32)
resolve_staged_kernel(const __grid_constant__ ResolveArgs A, const __grid_constant__ MlpWeightsT W)
{
    typedef typename Color<ColorT>::Packed Packed;
    constexpr uint32_t CB = Color<ColorT>::kBytes;
    constexpr int PPR = 32 / L;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpStage<ColorT>* stage = reinterpret_cast<WarpStage<ColorT>*>(smem_raw) + warp;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw + kWarpsPerCta * sizeof(WarpStage<ColorT>));
    const uint32_t bar = smem_u32(bars + warp);
    const uint32_t s_depth = smem_u32(stage->depth), s_rgba = smem_u32(stage->rgba);
    if (lane == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    uint32_t parity = 0;

    const uint32_t* __restrict__ offsets = A.offsets;
    const Packed* __restrict__ g_rgba = static_cast<const Packed*>(A.rgba);

    auto fetch_tile = [&]() -> uint32_t {
        uint32_t t = 0;
        if (lane == 0) t = atomicAdd(A.tile_counter, 1u);
        return __shfl_sync(0xffffffffu, t, 0);
    };
    // stage fragments [fs, fe) (fs a multiple of 4) into the warp's stage and wait for them
    auto stage_range = [&](uint32_t fs, uint32_t fe) {
        __syncwarp();                                   // everyone is done with the old contents
        uint32_t n4 = (fe - fs + 3u) & ~3u;
        if (fs + n4 > A.F) n4 = (A.F - fs) & ~3u;       // never read past the arrays
        if (lane == 0 && n4) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(bar, n4 * (4u + CB));
            bulk_g2s(s_depth, A.depth + fs, n4 * 4u, bar);
            bulk_g2s(s_rgba, g_rgba + fs, n4 * CB, bar);
        }
        const uint32_t rem = fe - fs > n4 ? fe - fs - n4 : 0u;   // < 4, last fragments of the frame
        if ((uint32_t)lane < rem) {
            stage->depth[n4 + lane] = __ldg(A.depth + fs + n4 + lane);
            stage->rgba[n4 + lane] = __ldg(g_rgba + fs + n4 + lane);
        }
        if (n4) {
            mbar_wait(bar, parity);
            parity ^= 1u;
        }
        __syncwarp();
    };
    auto load_offsets = [&](uint32_t tile, uint32_t& o0, uint32_t& o1) {
        const uint32_t p = tile * 32u + lane;
        o0 = __ldg(offsets + min(p, A.P));
        o1 = __ldg(offsets + min(p + 1u, A.P));
    };

    uint32_t tile = fetch_tile(), o0 = 0, o1 = 0;
    if (tile < A.num_tiles) load_offsets(tile, o0, o1);
    while (tile < A.num_tiles) {
        // next tile's index and offsets travel while this tile is processed
        const uint32_t next = fetch_tile();
        uint32_t no0 = 0, no1 = 0;
        if (next < A.num_tiles) load_offsets(next, no0, no1);

        Owned<ColorT> own;
        own.c1 = own.c2 = Color<ColorT>::zero();
        own.d1 = 1.0f; own.n = 0;
        own.acc_r = own.acc_g = own.acc_b = own.a_tail = 0.f; own.t_tail = 1.f;

        const uint32_t tb = __shfl_sync(0xffffffffu, o0, 0), te = __shfl_sync(0xffffffffu, o1, 31);
        const uint32_t fs = tb & ~3u;
        const bool heavy = te - fs > kCap;               // warp-uniform
        if (!heavy) {
            if (te > tb) {
                stage_range(fs, te);
                resolve_tile_staged<ColorT, L>(lane, o0, o1, stage, fs, own);
            }
        } else {
#pragma unroll 1
            for (int r = 0; r < L; ++r) {                // stage round by round
                const uint32_t rb = __shfl_sync(0xffffffffu, o0, r * PPR);
                const uint32_t re = __shfl_sync(0xffffffffu, o1, r * PPR + PPR - 1);
                const uint32_t base = rb & ~3u;
                if (re - base > kCap) {                  // lists longer than the stage
                    own = resolve_round_global<ColorT, L>(r, lane, o0, o1, A.depth,
                                                          const_cast<Packed*>(g_rgba), own);
                    continue;
                }
                if (re > rb) stage_range(base, re);
                resolve_round_staged<ColorT, L>(r, lane, o0, o1, stage, base, own);
            }
        }
        // ---- every lane now owns one pixel: features (O3), MLP (O4), composite (O5)
        const uint32_t p = tile * 32u + (uint32_t)((lane % L) * PPR + lane / L);
        if (p < A.P) {
            float xf[5], f[3];
            // O3 with one IEEE reciprocal instead of three divisions
            const bool has_tail = own.a_tail > 0.f;
            const float inv = has_tail ? 1.0f / own.a_tail : 0.f;
            xf[0] = (float)own.n; xf[1] = own.t_tail;
            xf[2] = own.acc_r * inv; xf[3] = own.acc_g * inv; xf[4] = own.acc_b * inv;
            mlp_forward_packed(W, xf, f);
            const float4 c1 = Color<ColorT>::unpack(own.c1), c2 = Color<ColorT>::unpack(own.c2);
            composite_store(A, p, c1, make_float4(c2.w * c2.x, c2.w * c2.y, c2.w * c2.z, c2.w),
                            own.n ? own.d1 : 1.0f, has_tail, f, own.t_tail);
        }
        tile = next; o0 = no0; o1 = no1;
    }
    // the last warp to finish re-arms the counters for the next launch
    if (lane == 0) {
        const uint32_t total = gridDim.x * kWarpsPerCta;
        if (atomicAdd(A.tile_counter + 1, 1u) == total - 1u) {
            A.tile_counter[0] = 0u;
            A.tile_counter[1] = 0u;
            __threadfence();
        }
    }
}

template <typename ColorT, int L>
static noit_status launch_staged(noit_ctx* ctx, const ResolveArgs& A, cudaStream_t st)
{
    const size_t smem = kWarpsPerCta * sizeof(WarpStage<ColorT>) + kWarpsPerCta * sizeof(uint64_t);
    static bool configured = false;                     // per instantiation
    if (!configured) {
        NOIT_CUDA(ctx, cudaFuncSetAttribute(resolve_staged_kernel<ColorT, L>,
                                            cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        configured = true;
    }
    int per_sm = 0;
    NOIT_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(
                       &per_sm, resolve_staged_kernel<ColorT, L>, kWarpsPerCta * 32, smem));
    if (per_sm < 1) return noit_fail(ctx, NOIT_ERR_CUDA, "resolve_staged_kernel does not fit an SM");
    const uint32_t want = (A.num_tiles + kWarpsPerCta - 1) / kWarpsPerCta;
    const uint32_t grid = min((uint32_t)(ctx->num_sms * per_sm), max(want, 1u));
    resolve_staged_kernel<ColorT, L><<<grid, kWarpsPerCta * 32, smem, st>>>(A, ctx->wt);
    ctx->launches += 1;
    NOIT_CUDA(ctx, cudaGetLastError());
    return NOIT_OK;
}

noit_status noit_launch_resolve_staged(noit_ctx* ctx, const ResolveArgs& A0, int color_fmt,
                                       cudaStream_t st)
{
    ResolveArgs A = A0;
    A.num_tiles = (A.P + 31u) / 32u;
    A.tile_counter = ctx->d_counters;
    if (color_fmt == NOIT_RGBA_F16) return launch_staged<__half, 4>(ctx, A, st);
    return launch_staged<float, 4>(ctx, A, st);
}
