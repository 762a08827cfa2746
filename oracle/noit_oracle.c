/* noit_oracle.c -- plain, slow, obviously-correct CPU oracle for the neural-OIT resolve.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * `--impl reference` legs may build, load or call this file.  It shares no code, header, table
 * or helper with the CUDA path (paper_2606_16747_b200/csrc/, include/noit.h) and never calls it.
 *
 * Written from /root/reference/PAPER.md ("P:n" = line n of that file) under the readings of
 * SURVEY.md section 8(c) (O1..O9, A1..A24), restated in DESIGN.md.  The method is an
 * approximation (a learned tail colour), so this is the algorithm step by step in the paper's
 * order and notation, not an "exact composite".  Every sum / product whose GPU counterpart is
 * an fp32 reduction is carried in double here; every DECISION that must be bit-exact (layer
 * selection, quadtree split, reprojection accept) is taken in the precision the readings fix
 * (fp32 compare + integer index; exact integers; fp32 in a fixed operation order).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC noit_oracle.c -lm
 * (-ffp-contract=off: nothing fuses unless written as fmaf).  OpenMP only parallelises the
 * outer pixel / tile loops; every pixel is computed by the same scalar code.
 *
 * Pins (tests/test_oracle_pins.py; every FUNCTION here is pinned against something other than
 * itself): brute-force sort, empty-tail identity, exact-tail identity, closed forms, numpy float64
 * MLP, quadtree closed forms + big-int brute force + the quantiser's clamp on out-of-range colours,
 * adaptive / frame-global identities, reprojection identity / integer shift / threshold flips /
 * M = s*I (the homogeneous divide) / a dyadic depth row / two cameras against a float64
 * un-projection, balance closed forms, temporal hysteresis in both threshold orders, the DFAOIT
 * features against a numpy lexsort restatement and Eq. 3's structure.
 * PARITY UNPINNED (readings, not functions): agreement of features O3 (reading A1), of the corner
 * metric's constant, of any threshold, of the trained weights and of the DFAOIT feature order
 * (reading A29) with the authors' shaders / supplemental material -- none of those is available
 * (P:55).
 */
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ABSENT 0xFFFFFFFFu

/* ---------------------------------------------------------------------------------------- */
/* fragment access                                                                           */
/* ---------------------------------------------------------------------------------------- */
typedef struct {
    int32_t width, height;
    const uint32_t *offsets; /* [P+1] */
    const float *depth;      /* [F]   */
    const void *rgba;        /* [F][4] _Float16 (fmt 0) or float (fmt 1), straight colour, .w=alpha */
    int32_t color_fmt;
} frag_view;

/* fp16 inputs are widened exactly (O2). */
static void frag_rgba(const frag_view *fb, uint32_t j, double out[4])
{
    if (fb->color_fmt == 0) {
        const _Float16 *h = (const _Float16 *)fb->rgba + 4 * (size_t)j;
        for (int k = 0; k < 4; ++k) out[k] = (double)(float)h[k];
    } else {
        const float *f = (const float *)fb->rgba + 4 * (size_t)j;
        for (int k = 0; k < 4; ++k) out[k] = (double)f[k];
    }
}

/* ---------------------------------------------------------------------------------------- */
/* O1 selection + O2 tail accumulators of ONE pixel                                          */
/* ---------------------------------------------------------------------------------------- */
typedef struct {
    uint32_t n;          /* N = n_p */
    uint32_t i1, i2;     /* GLOBAL fragment indices, ABSENT if missing       */
    double c1[4], c2[4]; /* straight RGBA of layers 1, 2 (zeros if absent)   */
    float d1;            /* depth of layer 1, 1.0f if the pixel is empty     */
    double c_acc[3];     /* C_acc = sum_{tail} alpha_i C_i */
    double a_tail;       /* sum_{tail} alpha_i                (reading A1)   */
    double t_tail;       /* prod_{tail} (1 - alpha_i)         (reading A1)   */
} pixel_layers;

/* key order: fp32 '<' on depth, then integer '<' on the fragment index (O1; tie rule from
 * BASELINE.json north_star "ties broken by fragment index").  Smaller depth = nearer (A9). */
static int key_less(float da, uint32_t ia, float db, uint32_t ib)
{
    if (da < db) return 1;
    if (db < da) return 0;
    return ia < ib;
}

static void pixel_select_reduce(const frag_view *fb, size_t p, pixel_layers *L)
{
    uint32_t b = fb->offsets[p], e = fb->offsets[p + 1];
    memset(L, 0, sizeof *L);
    L->n = e - b;
    L->i1 = L->i2 = ABSENT;
    L->d1 = 1.0f;
    L->t_tail = 1.0;
    /* O1: i1 = smallest key; i2 = smallest key among the rest.  Two plain scans. (P:55, P:95:
     * "the first two passes compute the first and the second closest fragments")            */
    for (uint32_t j = b; j < e; ++j)
        if (L->i1 == ABSENT || key_less(fb->depth[j], j, fb->depth[L->i1], L->i1)) L->i1 = j;
    for (uint32_t j = b; j < e; ++j) {
        if (j == L->i1) continue;
        if (L->i2 == ABSENT || key_less(fb->depth[j], j, fb->depth[L->i2], L->i2)) L->i2 = j;
    }
    if (L->i1 != ABSENT) { frag_rgba(fb, L->i1, L->c1); L->d1 = fb->depth[L->i1]; }
    if (L->i2 != ABSENT) frag_rgba(fb, L->i2, L->c2);
    /* O2: third pass -- every fragment that is not one of the two peeled layers, in index
     * order (P:117 C_acc = sum_{i=3}^{N} alpha_i C_i; P:111 prod (1 - a_i)).                 */
    for (uint32_t j = b; j < e; ++j) {
        if (j == L->i1 || j == L->i2) continue;
        double c[4];
        frag_rgba(fb, j, c);
        for (int k = 0; k < 3; ++k) L->c_acc[k] += c[3] * c[k];
        L->a_tail += c[3];
        L->t_tail *= (1.0 - c[3]);
    }
}

/* ---------------------------------------------------------------------------------------- */
/* O3 features                                                                               */
/* ---------------------------------------------------------------------------------------- */
/* x = [N, t_tail, C_acc / a_tail]  (readings A1, A2, A5); rounded to fp32 once.   */
static int features_from(double n, double t_tail, const double c_acc[3], double a_tail, float x[5])
{
    int has_tail = a_tail > 0.0;
    x[0] = (float)n;
    x[1] = (float)t_tail;
    for (int k = 0; k < 3; ++k) x[2 + k] = has_tail ? (float)(c_acc[k] / a_tail) : 0.0f;
    return has_tail;
}

/* ---------------------------------------------------------------------------------------- */
/* O4 MLP 5 -> 32 -> 16 -> 3, ReLU on both hidden layers (A3) and on the output        */
/* ---------------------------------------------------------------------------------------- */
/* w: 771 EFFECTIVE weights W1[32][5], b1[32], W2[16][32], b2[16], W3[3][16], b3[3] (row =
 * output neuron).  Each dot product is accumulated in double, in input-index order, starting
 * from the bias.  Activations are never rounded (A6).                                        */
static void mlp_forward(const float *w, const float x[5], double f[3])
{
    const float *W1 = w, *b1 = W1 + 32 * 5, *W2 = b1 + 32, *b2 = W2 + 16 * 32;
    const float *W3 = b2 + 16, *b3 = W3 + 3 * 16;
    double h1[32], h2[16];
    for (int o = 0; o < 32; ++o) {
        double a = (double)b1[o];
        for (int i = 0; i < 5; ++i) a += (double)W1[o * 5 + i] * (double)x[i];
        h1[o] = a > 0.0 ? a : 0.0;
    }
    for (int o = 0; o < 16; ++o) {
        double a = (double)b2[o];
        for (int i = 0; i < 32; ++i) a += (double)W2[o * 32 + i] * h1[i];
        h2[o] = a > 0.0 ? a : 0.0;
    }
    for (int o = 0; o < 3; ++o) {
        double a = (double)b3[o];
        for (int i = 0; i < 16; ++i) a += (double)W3[o * 16 + i] * h2[i];
        f[o] = a > 0.0 ? a : 0.0;
    }
}

/* bf16 weight mode (A6): each weight rounded to bf16, round-to-nearest-even, then widened.   */
void oracle_round_weights_bf16(float *w, int32_t count)
{
    for (int32_t i = 0; i < count; ++i) {
        uint32_t u;
        memcpy(&u, &w[i], 4);
        if ((u & 0x7F800000u) != 0x7F800000u) {           /* finite */
            uint32_t lsb = (u >> 16) & 1u;
            u += 0x7FFFu + lsb;
        }
        u &= 0xFFFF0000u;
        memcpy(&w[i], &u, 4);
    }
}

int32_t oracle_infer(const float *weights, const float *features, uint32_t n, float *tail_rgb)
{
    if (!weights || !features || !tail_rgb) return 1;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < (int64_t)n; ++r) {
        double f[3];
        mlp_forward(weights, features + 5 * r, f);
        for (int k = 0; k < 3; ++k) tail_rgb[3 * r + k] = (float)f[k];
    }
    return 0;
}

/* NEXT-4 (comparison variant): the network DFAOIT feeds with 10 input features and  */
/* a SIGMOID output, "the architecture differs only in the output activation":           */
/* 10 -> 32 -> 16 -> 3 = 931 parameters, W1[32][10], b1[32], W2[16][32], b2[16], W3[3][16],     */
/* b3[3].  Only the network is built (inference-cost ratio 10 -> 5 features); what the  */
/* ten features ARE is only summarised in this paper: parity of the inputs unpinned.   */
int32_t oracle_infer10(const float *w, const float *features, uint32_t n, float *rgb)
{
    if (!w || !features || !rgb) return 1;
    const float *W1 = w, *b1 = W1 + 32 * 10, *W2 = b1 + 32, *b2 = W2 + 16 * 32;
    const float *W3 = b2 + 16, *b3 = W3 + 3 * 16;
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < (int64_t)n; ++r) {
        const float *x = features + 10 * r;
        double h1[32], h2[16];
        for (int o = 0; o < 32; ++o) {
            double a = (double)b1[o];
            for (int i = 0; i < 10; ++i) a += (double)W1[o * 10 + i] * (double)x[i];
            h1[o] = a > 0.0 ? a : 0.0;
        }
        for (int o = 0; o < 16; ++o) {
            double a = (double)b2[o];
            for (int i = 0; i < 32; ++i) a += (double)W2[o * 32 + i] * h1[i];
            h2[o] = a > 0.0 ? a : 0.0;
        }
        for (int o = 0; o < 3; ++o) {
            double a = (double)b3[o];
            for (int i = 0; i < 16; ++i) a += (double)W3[o * 16 + i] * h2[i];
            rgb[3 * r + o] = (float)(1.0 / (1.0 + exp(-a)));
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* S1-S3: layers, tail accumulators, features for every pixel                                */
/* ---------------------------------------------------------------------------------------- */
/* Any output may be NULL.  idx1/idx2 are LOCAL indices (j - offsets[p]), ABSENT if missing.  */
int32_t oracle_build_features(int32_t width, int32_t height, const uint32_t *offsets,
                              const float *depth, const void *rgba, int32_t color_fmt,
                              uint32_t *idx1, uint32_t *idx2, uint32_t *count, float *layer1,
                              float *layer2, float *depth1, float *tail_raw, float *features)
{
    frag_view fb = {width, height, offsets, depth, rgba, color_fmt};
    int64_t P = (int64_t)width * height;
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t p = 0; p < P; ++p) {
        pixel_layers L;
        pixel_select_reduce(&fb, (size_t)p, &L);
        if (idx1) idx1[p] = L.i1 == ABSENT ? ABSENT : L.i1 - offsets[p];
        if (idx2) idx2[p] = L.i2 == ABSENT ? ABSENT : L.i2 - offsets[p];
        if (count) count[p] = L.n;
        if (layer1) for (int k = 0; k < 4; ++k) layer1[4 * p + k] = (float)L.c1[k];
        if (layer2) for (int k = 0; k < 4; ++k) layer2[4 * p + k] = (float)L.c2[k];
        if (depth1) depth1[p] = L.d1;
        if (tail_raw) {
            for (int k = 0; k < 3; ++k) tail_raw[5 * p + k] = (float)L.c_acc[k];
            tail_raw[5 * p + 3] = (float)L.a_tail;
            tail_raw[5 * p + 4] = (float)L.t_tail;
        }
        if (features) features_from((double)L.n, L.t_tail, L.c_acc, L.a_tail, features + 5 * p);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O5 composite (Eq. 4) and O7 adaptive variant                                    */
/* ---------------------------------------------------------------------------------------- */
static void store_outputs(int64_t p, const double ct[3], double t_tot, const float bg[3], float d1,
                          float *out_trans, float *out_final, float *out_depth1)
{
    if (out_trans) {
        for (int k = 0; k < 3; ++k) out_trans[4 * p + k] = (float)ct[k];
        out_trans[4 * p + 3] = (float)t_tot;
    }
    if (out_final) {                 /* C_p = C_t + prod(1-a_i) C_b  (Eq. 3, Eq. 4)     */
        for (int k = 0; k < 3; ++k) out_final[4 * p + k] = (float)(ct[k] + t_tot * (double)bg[k]);
        out_final[4 * p + 3] = (float)(1.0 - t_tot);
    }
    if (out_depth1) out_depth1[p] = d1;
}

/* Plain pixel (lod 0): O1-O5.  tail_override (oracle-only test hook): if non-NULL, f(x) is
 * replaced by tail_override[p] so that Eq. 4's structure can be pinned without any weights.  */
static void resolve_pixel_full(const frag_view *fb, int64_t p, const float *weights,
                               const float *tail_override, const float bg[3], float *out_trans,
                               float *out_final, float *out_depth1)
{
    pixel_layers L;
    float x[5];
    double f[3], ct[3];
    pixel_select_reduce(fb, (size_t)p, &L);
    int has_tail = features_from((double)L.n, L.t_tail, L.c_acc, L.a_tail, x);
    if (tail_override) for (int k = 0; k < 3; ++k) f[k] = (double)tail_override[3 * p + k];
    else mlp_forward(weights, x, f);
    double a1 = L.c1[3], a2 = L.c2[3];           /* absent layers have alpha = 0 (A10)        */
    double t2 = (1.0 - a1) * (1.0 - a2);         /* T_2                               */
    for (int k = 0; k < 3; ++k) {
        double c_ex = a1 * L.c1[k] + (1.0 - a1) * a2 * L.c2[k];      /* C_exact,2     */
        ct[k] = c_ex + (has_tail ? t2 * f[k] : 0.0);                 /* A2: no tail, no term  */
    }
    store_outputs(p, ct, t2 * L.t_tail, bg, L.d1, out_trans, out_final, out_depth1);
}

/* G = [a2*C2 (3), a2, C_acc (3), A_tail, T_tail, N] of ONE coarse pixel, self-contained
 * O1-O2 on the coarse buffer (O7, A19: each coarse pixel peels its own top-2).               */
static void coarse_G(const frag_view *cb, int cx, int cy, double G[10])
{
    pixel_layers L;
    pixel_select_reduce(cb, (size_t)cy * cb->width + cx, &L);
    for (int k = 0; k < 3; ++k) G[k] = L.c2[3] * L.c2[k];
    G[3] = L.c2[3];
    for (int k = 0; k < 3; ++k) G[4 + k] = L.c_acc[k];
    G[7] = L.a_tail;
    G[8] = L.t_tail;
    G[9] = (double)L.n;
}

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* lod > 0 pixel (O7; P:76 pass 1 always full-res; P:87 bilinear upsample of passes 2/3, then
 * inference and composite at full resolution).  r = 2^lod; leaf_side = 64 >> level.          */
static void resolve_pixel_coarse(const frag_view *fb, const frag_view *cb, int r, int leaf_side,
                                 int x, int y, const float *weights, const float bg[3],
                                 float *out_trans, float *out_final, float *out_depth1)
{
    int64_t p = (int64_t)y * fb->width + x;
    pixel_layers L;
    pixel_select_reduce(fb, (size_t)p, &L);      /* only layer 1 of it is used                */
    /* sample position in coarse texel units; taps clamped to the leaf and to the image       */
    double u = (x + 0.5) / r - 0.5, v = (y + 0.5) / r - 0.5;
    int i0 = (int)floor(u), j0 = (int)floor(v);
    double wx = u - i0, wy = v - j0;
    int lx0 = (x / leaf_side) * leaf_side, ly0 = (y / leaf_side) * leaf_side;
    int tx_lo = lx0 / r, tx_hi = (lx0 + leaf_side - 1) / r;
    int ty_lo = ly0 / r, ty_hi = (ly0 + leaf_side - 1) / r;
    if (tx_hi > cb->width - 1) tx_hi = cb->width - 1;
    if (ty_hi > cb->height - 1) ty_hi = cb->height - 1;
    int xa = clampi(i0, tx_lo, tx_hi), xb = clampi(i0 + 1, tx_lo, tx_hi);
    int ya = clampi(j0, ty_lo, ty_hi), yb = clampi(j0 + 1, ty_lo, ty_hi);
    double g00[10], g10[10], g01[10], g11[10], G[10];
    coarse_G(cb, xa, ya, g00);
    coarse_G(cb, xb, ya, g10);
    coarse_G(cb, xa, yb, g01);
    coarse_G(cb, xb, yb, g11);
    for (int k = 0; k < 10; ++k) {               /* lerp x first, then y                      */
        double top = g00[k] + wx * (g10[k] - g00[k]);
        double bot = g01[k] + wx * (g11[k] - g01[k]);
        G[k] = top + wy * (bot - top);
    }
    float xf[5];
    double f[3], ct[3];
    int has_tail = features_from(G[9], G[8], &G[4], G[7], xf);
    mlp_forward(weights, xf, f);
    double a1 = L.c1[3];
    double t2 = (1.0 - a1) * (1.0 - G[3]);
    for (int k = 0; k < 3; ++k)
        ct[k] = a1 * L.c1[k] + (1.0 - a1) * G[k] + (has_tail ? t2 * f[k] : 0.0);
    store_outputs(p, ct, t2 * G[8], bg, L.d1, out_trans, out_final, out_depth1);
}

/* bilinear sample of G at the full-res pixel centre, taps clamped to the image only            */
static void sample_G_image(const frag_view *cb, int r, int x, int y, double G[10])
{
    double u = (x + 0.5) / r - 0.5, v = (y + 0.5) / r - 0.5;
    int i0 = (int)floor(u), j0 = (int)floor(v);
    double wx = u - i0, wy = v - j0;
    int xa = clampi(i0, 0, cb->width - 1), xb = clampi(i0 + 1, 0, cb->width - 1);
    int ya = clampi(j0, 0, cb->height - 1), yb = clampi(j0 + 1, 0, cb->height - 1);
    double g00[10], g10[10], g01[10], g11[10];
    coarse_G(cb, xa, ya, g00);
    coarse_G(cb, xb, ya, g10);
    coarse_G(cb, xa, yb, g01);
    coarse_G(cb, xb, yb, g11);
    for (int k = 0; k < 10; ++k) {               /* lerp x first, then y                      */
        double top = g00[k] + wx * (g10[k] - g00[k]);
        double bot = g01[k] + wx * (g11[k] - g01[k]);
        G[k] = top + wy * (bot - top);
    }
}

/* O7g frame-global resolution control as the paper does it:      */
/* pass 1 (layer 1) always at full resolution; pass 2 (layer 2) at lod2 and pass 3 (tail */
/* statistics and N) at lod3 for the WHOLE frame, lod_p = the power-of-two snap of the Eq. 2     */
/* scale s_p (reading A27: lod 0 if s > 2^-0.5, 1 if s > 2^-1.5, else 2); lod 0 takes the        */
/* pixel's own full-resolution list, lod > 0 the bilinear upsample of that pass's outputs from   */
/* the half / quarter buffer, taps clamped to the image; features, MLP and composite at   */
/* full resolution as in O7.                                                                     */
int32_t oracle_resolve_global(int32_t width, int32_t height, const uint32_t *offsets, const float *depth,
                              const void *rgba, int32_t color_fmt,
                              int32_t hw, int32_t hh, const uint32_t *hoff, const float *hdepth,
                              const void *hrgba,
                              int32_t qw, int32_t qh, const uint32_t *qoff, const float *qdepth,
                              const void *qrgba, int32_t lod2, int32_t lod3, const float *weights,
                              const float *background, float *out_trans, float *out_final,
                              float *out_depth1)
{
    frag_view fb = {width, height, offsets, depth, rgba, color_fmt};
    frag_view hb = {hw, hh, hoff, hdepth, hrgba, color_fmt};
    frag_view qb = {qw, qh, qoff, qdepth, qrgba, color_fmt};
    if (lod2 < 0 || lod2 > 2 || lod3 < 0 || lod3 > 2) return 2;
    int64_t P = (int64_t)width * height;
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t p = 0; p < P; ++p) {
        int x = (int)(p % width), y = (int)(p / width);
        pixel_layers L;
        pixel_select_reduce(&fb, (size_t)p, &L);
        double own[10], G2[10], G3[10];
        for (int k = 0; k < 3; ++k) own[k] = L.c2[3] * L.c2[k];
        own[3] = L.c2[3];
        for (int k = 0; k < 3; ++k) own[4 + k] = L.c_acc[k];
        own[7] = L.a_tail; own[8] = L.t_tail; own[9] = (double)L.n;
        if (lod2 == 0) memcpy(G2, own, sizeof own);
        else sample_G_image(lod2 == 1 ? &hb : &qb, 1 << lod2, x, y, G2);
        if (lod3 == 0) memcpy(G3, own, sizeof own);
        else if (lod3 == lod2) memcpy(G3, G2, sizeof G2);
        else sample_G_image(lod3 == 1 ? &hb : &qb, 1 << lod3, x, y, G3);
        float xf[5];
        double f[3], ct[3];
        int has_tail = features_from(G3[9], G3[8], &G3[4], G3[7], xf);
        mlp_forward(weights, xf, f);
        double a1 = L.c1[3];
        double t2 = (1.0 - a1) * (1.0 - G2[3]);
        for (int k = 0; k < 3; ++k)
            ct[k] = a1 * L.c1[k] + (1.0 - a1) * G2[k] + (has_tail ? t2 * f[k] : 0.0);
        store_outputs(p, ct, t2 * G3[8], background, L.d1, out_trans, out_final, out_depth1);
    }
    return 0;
}

/* S1-S5 (+S7 when cell_level != NULL, +S9 when pixel_list != NULL).
 * half/quarter buffers: pass width 0 to mark a buffer as absent.
 * cell_level[cy*ceil(W/8)+cx] in 0..3 ; level_to_lod[4] in {0,1,2}.
 * pixel_list/pixel_count: resolve exactly those pixels, leave the rest untouched (O9).       */
int32_t oracle_resolve(int32_t width, int32_t height, const uint32_t *offsets, const float *depth,
                       const void *rgba, int32_t color_fmt,
                       int32_t hw, int32_t hh, const uint32_t *hoff, const float *hdepth,
                       const void *hrgba,
                       int32_t qw, int32_t qh, const uint32_t *qoff, const float *qdepth,
                       const void *qrgba,
                       const uint8_t *cell_level, const uint8_t *level_to_lod,
                       const float *weights, const float *tail_override, const float *background,
                       const uint32_t *pixel_list, uint32_t pixel_count,
                       float *out_trans, float *out_final, float *out_depth1,
                       const float *background_image /* [P][4] per-pixel C_b (A11, NEXT-4) or NULL */)
{
    frag_view fb = {width, height, offsets, depth, rgba, color_fmt};
    frag_view hb = {hw, hh, hoff, hdepth, hrgba, color_fmt};
    frag_view qb = {qw, qh, qoff, qdepth, qrgba, color_fmt};
    if (!weights && !tail_override) return 4;
    int64_t P = (int64_t)width * height;
    int64_t count = pixel_list ? (int64_t)pixel_count : P;
    int cells_x = (width + 7) / 8;
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t t = 0; t < count; ++t) {
        int64_t p = pixel_list ? (int64_t)pixel_list[t] : t;
        int x = (int)(p % width), y = (int)(p / width);
        int lod = 0, level = 3;
        if (cell_level) {
            level = cell_level[(y / 8) * cells_x + (x / 8)];
            lod = level_to_lod[level];
        }
        const float *bgp = background_image ? background_image + 4 * p : background;
        if (lod == 0)
            resolve_pixel_full(&fb, p, weights, tail_override, bgp, out_trans, out_final,
                               out_depth1);
        else
            resolve_pixel_coarse(&fb, lod == 1 ? &hb : &qb, 1 << lod, 64 >> level, x, y, weights,
                                 bgp, out_trans, out_final, out_depth1);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O12 (NEXT-4, comparison variant): the DFAOIT resolve STAR-NT starts from (Eq. 3) */
/* ---------------------------------------------------------------------------------------- */
/* "The original DFAOIT directly predicts the transparency color C_t using 10 input features"
 * (P:99), composited as C_p = C_t + C_b prod_{i=1..n} (1 - alpha_i) (Eq. 3).  P:104 lists
 * "the exact Porter-Duff blended color of the two front fragments" (3), "the average color C_avg"
 * (3) "and average opacity alpha_avg" (1) "of the remaining n-2 fragments", "the accumulated
 * premultiplied color C_acc" (3) "and the fragment count n" (1): eleven scalars for ten inputs.
 * Reading A29: the ten network inputs are the ten colour / opacity scalars, in the
 * paper's order; n is the count the two averages are taken over (n - 2), not an input:
 *   x[0..2] = alpha1 C1 + (1 - alpha1) alpha2 C2        (layers by O1; "over", premultiplied)
 *   x[3..5] = (1/m) sum_tail C_i,   x[6] = (1/m) sum_tail alpha_i,   m = max(n - 2, 0)
 *   x[7..9] = sum_tail alpha_i C_i                       (the same C_acc as O2)
 * with all tail entries 0 when m = 0.  The network (oracle_infer10's: 10 -> 32 -> 16 -> 3, ReLU
 * hidden, SIGMOID output) predicts the whole transparency colour C_t for every pixel with
 * n >= 1 -- the two exact layers are NOT decoupled, which is the limitation P:106 names; an
 * empty pixel (n = 0) has C_t = 0 (nothing to predict; the paper is silent).  T_tot is the
 * product over ALL fragments in index order.  Parity with the DFAOIT authors' feature order and
 * scaling: unpinned (their paper and code are not in the container).                          */
static void features10_from(const frag_view *fb, const pixel_layers *L, size_t p, float x[10],
                            double *t_all)
{
    uint32_t b = fb->offsets[p], e = fb->offsets[p + 1];
    double sum_c[3] = {0, 0, 0}, sum_a = 0.0, t = 1.0;
    uint32_t m = 0;
    for (uint32_t j = b; j < e; ++j) {
        double c[4];
        frag_rgba(fb, j, c);
        t *= (1.0 - c[3]);                           /* prod over all n fragments (Eq. 3)     */
        if (j == L->i1 || j == L->i2) continue;
        for (int k = 0; k < 3; ++k) sum_c[k] += c[k];
        sum_a += c[3];
        ++m;
    }
    double a1 = L->c1[3], a2 = L->c2[3];
    for (int k = 0; k < 3; ++k) {
        x[k] = (float)(a1 * L->c1[k] + (1.0 - a1) * a2 * L->c2[k]);
        x[3 + k] = m ? (float)(sum_c[k] / (double)m) : 0.0f;
        x[7 + k] = (float)L->c_acc[k];
    }
    x[6] = m ? (float)(sum_a / (double)m) : 0.0f;
    *t_all = t;
}

/* w931 as in oracle_infer10.  Outputs as oracle_resolve; features10 [P][10] optional.         */
int32_t oracle_resolve10(int32_t width, int32_t height, const uint32_t *offsets, const float *depth,
                         const void *rgba, int32_t color_fmt, const float *w931,
                         const float *background, float *out_trans, float *out_final,
                         float *out_depth1, float *features10)
{
    if (!offsets || !w931 || !background) return 1;
    frag_view fb = {width, height, offsets, depth, rgba, color_fmt};
    int64_t P = (int64_t)width * height;
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t p = 0; p < P; ++p) {
        pixel_layers L;
        float x[10], rgb[3];
        double t_all, ct[3] = {0, 0, 0};
        pixel_select_reduce(&fb, (size_t)p, &L);
        features10_from(&fb, &L, (size_t)p, x, &t_all);
        if (features10) memcpy(features10 + 10 * p, x, sizeof x);
        if (L.n > 0) {
            oracle_infer10(w931, x, 1, rgb);
            for (int k = 0; k < 3; ++k) ct[k] = (double)rgb[k];
        }
        store_outputs(p, ct, t_all, background, L.d1, out_trans, out_final, out_depth1);
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O5x exact reference: sort every fragment (O1 order), then Eq. 1 read with            */
/* premultiplied C_p = alpha_p * C_p (A8) plus the background term of Eq. 3.           */
/* Used by the invariants only.                                                              */
/* ---------------------------------------------------------------------------------------- */
typedef struct { float d; uint32_t j; } sort_key;
static int cmp_key(const void *a, const void *b)
{
    const sort_key *ka = a, *kb = b;
    if (key_less(ka->d, ka->j, kb->d, kb->j)) return -1;
    if (key_less(kb->d, kb->j, ka->d, ka->j)) return 1;
    return 0;
}

/* out_final[P][4] = (C, 1 - T);  out_tail[P][3] (optional) = exact composite of the sorted
 * fragments from the 3rd on, sum_{k>=3} a_k C_k prod_{3<=q<k}(1-a_q), i.e. what f(x) stands for */
int32_t oracle_exact(int32_t width, int32_t height, const uint32_t *offsets, const float *depth,
                     const void *rgba, int32_t color_fmt, const float *background,
                     float *out_final, float *out_tail)
{
    frag_view fb = {width, height, offsets, depth, rgba, color_fmt};
    int64_t P = (int64_t)width * height;
#pragma omp parallel for schedule(dynamic, 1024)
    for (int64_t p = 0; p < P; ++p) {
        uint32_t b = offsets[p], e = offsets[p + 1], n = e - b;
        sort_key *keys = malloc(sizeof(sort_key) * (n ? n : 1));
        for (uint32_t j = b; j < e; ++j) { keys[j - b].d = depth[j]; keys[j - b].j = j; }
        qsort(keys, n, sizeof(sort_key), cmp_key);   /* keys are distinct: order is total     */
        double C[3] = {0, 0, 0}, T = 1.0, Ct[3] = {0, 0, 0}, Tt = 1.0;
        for (uint32_t k = 0; k < n; ++k) {
            double c[4];
            frag_rgba(&fb, keys[k].j, c);
            for (int ch = 0; ch < 3; ++ch) C[ch] += T * c[3] * c[ch];
            T *= (1.0 - c[3]);
            if (k >= 2) {
                for (int ch = 0; ch < 3; ++ch) Ct[ch] += Tt * c[3] * c[ch];
                Tt *= (1.0 - c[3]);
            }
        }
        free(keys);
        if (out_final) {
            for (int ch = 0; ch < 3; ++ch)
                out_final[4 * p + ch] = (float)(C[ch] + T * (double)background[ch]);
            out_final[4 * p + 3] = (float)(1.0 - T);
        }
        if (out_tail) for (int ch = 0; ch < 3; ++ch) out_tail[3 * p + ch] = (float)Ct[ch];
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O6 quadtree (section 3.1; sizes 64 -> 8 from BASELINE.json cfg4, reading A13)       */
/* ---------------------------------------------------------------------------------------- */
typedef struct {
    const float *image; /* [P][4] */
    int32_t width, height;
    int32_t metric;     /* 0 = integer colour variance (primary, A14/A16), 1 = corner D_i    */
    uint32_t var_threshold_q;
    float corner_threshold;
} qt_args;

/* 8-bit quantise: q = rint(255 * clamp(c, 0, 1)), single fp32 multiply, round-half-even.      */
static uint32_t quant8(float c)
{
    float cl = c < 0.0f ? 0.0f : (c > 1.0f ? 1.0f : c);
    return (uint32_t)lrintf(255.0f * cl);
}

/* does the node [x0,x0+side) x [y0,y0+side) split?  (strict '>' against the threshold)        */
static int node_splits(const qt_args *a, int x0, int y0, int side)
{
    int x1 = x0 + side, y1 = y0 + side;
    if (x1 > a->width) x1 = a->width;
    if (y1 > a->height) y1 = a->height;
    if (x0 >= x1 || y0 >= y1) return 0;            /* wholly outside the image (A17)         */
    if (a->metric == 0) {
        uint64_t n = 0, s1[3] = {0, 0, 0}, s2[3] = {0, 0, 0};
        for (int y = y0; y < y1; ++y)
            for (int x = x0; x < x1; ++x) {
                const float *px = a->image + 4 * ((size_t)y * a->width + x);
                for (int c = 0; c < 3; ++c) {
                    uint64_t q = quant8(px[c]);
                    s1[c] += q;
                    s2[c] += q * q;
                }
                ++n;
            }
        /* sum_c (n*S2_c - S1_c^2) > thr * n^2   <=>   sum_c var_c > thr   (8-bit units^2)    */
        uint64_t lhs = 0;
        for (int c = 0; c < 3; ++c) lhs += n * s2[c] - s1[c] * s1[c];
        return lhs > (uint64_t)a->var_threshold_q * n * n;
    }
    /* corner metric D_i: mean pairwise Euclidean colour distance of the 4 corner
     * samples of the node's in-image rectangle; fp32, fixed order (A14)                      */
    int xs[4] = {x0, x1 - 1, x0, x1 - 1}, ys[4] = {y0, y0, y1 - 1, y1 - 1};
    static const int pa[6] = {0, 0, 0, 1, 1, 2}, pb[6] = {1, 2, 3, 2, 3, 3};
    float sum = 0.0f;
    for (int k = 0; k < 6; ++k) {
        const float *A = a->image + 4 * ((size_t)ys[pa[k]] * a->width + xs[pa[k]]);
        const float *B = a->image + 4 * ((size_t)ys[pb[k]] * a->width + xs[pb[k]]);
        float dr = A[0] - B[0], dg = A[1] - B[1], db = A[2] - B[2];
        float s = dr * dr;
        s = s + dg * dg;
        s = s + db * db;
        float root = sqrtf(s);
        sum = k == 0 ? root : sum + root;
    }
    float D = sum * (1.0f / 6.0f);
    return D > a->corner_threshold;
}

/* tile_mask[Ty*Tx] (21 bits), cell_level[ceil(H/8)*ceil(W/8)], hist[4] (zeroed here).
 * Mask bits: 0 = root split; 1+c = level-1 child c split (c = cx + 2cy); 5+4c+g = level-2
 * grandchild g of child c split (g = gx + 2gy).  Top-down: a node is evaluated only if its
 * parent split.  Level-3 nodes (8x8) never split.                                      */
/* Generic in the base tile side B (64: BASELINE.json's sizes, 16: the paper's own 16 -> 2,     */
/* P:61): node sides B, B/2, B/4, leaves down to B/8; cells are B/8 square. */
int32_t oracle_quadtree_base(const float *image, int32_t width, int32_t height, int32_t metric,
                             uint32_t var_threshold_q, float corner_threshold, int32_t base,
                             uint32_t *tile_mask, uint8_t *cell_level, uint32_t *hist)
{
    if (base != 64 && base != 16) return 1;
    qt_args a = {image, width, height, metric, var_threshold_q, corner_threshold};
    const int B = base, cs = base / 8;                   /* cell side */
    int Tx = (width + B - 1) / B, Ty = (height + B - 1) / B;
    int cells_x = (width + cs - 1) / cs, cells_y = (height + cs - 1) / cs;
    uint64_t h[4] = {0, 0, 0, 0};
    for (int ty = 0; ty < Ty; ++ty)
        for (int tx = 0; tx < Tx; ++tx) {
            int X = tx * B, Y = ty * B;
            uint32_t mask = 0;
            uint8_t lvl[8][8];                       /* leaf level of each cell of the tile */
            memset(lvl, 0, sizeof lvl);
            if (node_splits(&a, X, Y, B)) {
                mask |= 1u;
                for (int c = 0; c < 4; ++c) {
                    int cx = X + (B / 2) * (c & 1), cy = Y + (B / 2) * (c >> 1);
                    int child_split = node_splits(&a, cx, cy, B / 2);
                    if (child_split) mask |= 1u << (1 + c);
                    for (int g = 0; g < 4; ++g) {
                        int gx = cx + (B / 4) * (g & 1), gy = cy + (B / 4) * (g >> 1);
                        int level = 1;
                        if (child_split) {
                            level = 2;
                            if (node_splits(&a, gx, gy, B / 4)) {
                                mask |= 1u << (5 + 4 * c + g);
                                level = 3;
                            }
                        }
                        for (int v = 0; v < 2; ++v)
                            for (int u = 0; u < 2; ++u)
                                lvl[(gy - Y) / cs + v][(gx - X) / cs + u] = (uint8_t)level;
                    }
                }
            }
            if (tile_mask) tile_mask[ty * Tx + tx] = mask;
            /* histogram: leaves that contain >= 1 in-image pixel, counted once each           */
            for (int level = 0; level < 4; ++level) {
                int side = B >> level, per = 1 << level;
                for (int ny = 0; ny < per; ++ny)
                    for (int nx = 0; nx < per; ++nx) {
                        int x0 = X + nx * side, y0 = Y + ny * side;
                        if (x0 >= width || y0 >= height) continue;
                        if (lvl[(y0 - Y) / cs][(x0 - X) / cs] != level) continue;
                        /* a leaf at `level` is the node whose own level equals the cell's    */
                        h[level] += 1;
                    }
            }
            for (int v = 0; v < 8; ++v)
                for (int u = 0; u < 8; ++u) {
                    int cxg = X / cs + u, cyg = Y / cs + v;
                    if (cxg < cells_x && cyg < cells_y && cell_level)
                        cell_level[cyg * cells_x + cxg] = lvl[v][u];
                }
        }
    if (hist) for (int k = 0; k < 4; ++k) hist[k] = (uint32_t)h[k];
    return 0;
}

int32_t oracle_quadtree(const float *image, int32_t width, int32_t height, int32_t metric,
                        uint32_t var_threshold_q, float corner_threshold, uint32_t *tile_mask,
                        uint8_t *cell_level, uint32_t *hist)
{
    return oracle_quadtree_base(image, width, height, metric, var_threshold_q, corner_threshold, 64,
                                tile_mask, cell_level, hist);
}

/* ---------------------------------------------------------------------------------------- */
/* O10 quadtree consistency + demand index.          */
/* "neighboring tiles may differ by at most one refinement level ... since refinement levels    */
/* are limited to {0,1,2,3}, two relaxation iterations (k=2) are sufficient".  Reading   */
/* A25: the level of a base tile is the depth of its subtree (0 = unsplit .. 3 = a  */
/* grandchild split); one relaxation iteration is the Jacobi step                               */
/*     L_i <- max(L_i, max over the 4 edge neighbours j of L_j - 1)                             */
/* evaluated for all tiles from the PREVIOUS iteration's levels; a tile whose level rises to L  */
/* is refined uniformly to depth L (every node above depth L splits), which keeps the mask      */
/* valid (child bit => parent bit).  Then cell levels and the histogram of occupied leaves are  */
/* recomputed, w = sum l N_l / sum N_l and s_p = clamp(2^(w - delta_p), 0.25, 1) (Eq. 2  */
/* P:80) with delta_2 = 2.2, delta_3 = 3.0 are formed in double.                                */
static int mask_depth(uint32_t mask)
{
    if (!(mask & 1u)) return 0;
    if (!(mask & 0x1Eu)) return 1;
    if (!(mask & 0x1FFFE0u)) return 2;
    return 3;
}

/* leaf level of every 8x8 cell and the histogram of leaves that hold >= 1 in-image pixel,      */
/* recounted from the 21-bit masks alone                                                       */
static void levels_and_hist_from_masks(int32_t width, int32_t height, const uint32_t *tile_mask,
                                       uint8_t *cell_level, uint64_t h[4])
{
    int Tx = (width + 63) / 64, Ty = (height + 63) / 64;
    int cells_x = (width + 7) / 8, cells_y = (height + 7) / 8;
    h[0] = h[1] = h[2] = h[3] = 0;
    for (int ty = 0; ty < Ty; ++ty)
        for (int tx = 0; tx < Tx; ++tx) {
            uint32_t mask = tile_mask[ty * Tx + tx];
            int X = tx * 64, Y = ty * 64;
            for (int v = 0; v < 8; ++v)
                for (int u = 0; u < 8; ++u) {
                    int c = (u >> 2) + 2 * (v >> 2), g = ((u >> 1) & 1) + 2 * ((v >> 1) & 1);
                    int level = 0;
                    if (mask & 1u) {
                        level = 1;
                        if ((mask >> (1 + c)) & 1u) level = ((mask >> (5 + 4 * c + g)) & 1u) ? 3 : 2;
                    }
                    int cxg = X / 8 + u, cyg = Y / 8 + v;
                    if (cxg >= cells_x || cyg >= cells_y) continue;
                    if (cell_level) cell_level[cyg * cells_x + cxg] = (uint8_t)level;
                    /* a leaf is counted at its first (top-left) cell, which is in the image  */
                    /* whenever the leaf holds an in-image pixel                              */
                    int span = 8 >> level;              /* leaf side in cells */
                    if (u % span == 0 && v % span == 0) h[level] += 1;
                }
        }
}

int32_t oracle_quadtree_balance(int32_t width, int32_t height, int32_t iterations, float delta2,
                                float delta3, uint32_t *tile_mask, uint8_t *tile_level,
                                uint8_t *cell_level, uint32_t *hist, float *scales)
{
    int Tx = (width + 63) / 64, Ty = (height + 63) / 64;
    int cells_x = (width + 7) / 8, cells_y = (height + 7) / 8;
    int n = Tx * Ty;
    int *cur = (int *)malloc(sizeof(int) * (size_t)n), *nxt = (int *)malloc(sizeof(int) * (size_t)n);
    if (!cur || !nxt) { free(cur); free(nxt); return 1; }
    for (int i = 0; i < n; ++i) cur[i] = mask_depth(tile_mask[i]);
    for (int it = 0; it < iterations; ++it) {
        for (int ty = 0; ty < Ty; ++ty)
            for (int tx = 0; tx < Tx; ++tx) {
                int best = cur[ty * Tx + tx];
                if (tx > 0 && cur[ty * Tx + tx - 1] - 1 > best) best = cur[ty * Tx + tx - 1] - 1;
                if (tx + 1 < Tx && cur[ty * Tx + tx + 1] - 1 > best) best = cur[ty * Tx + tx + 1] - 1;
                if (ty > 0 && cur[(ty - 1) * Tx + tx] - 1 > best) best = cur[(ty - 1) * Tx + tx] - 1;
                if (ty + 1 < Ty && cur[(ty + 1) * Tx + tx] - 1 > best) best = cur[(ty + 1) * Tx + tx] - 1;
                nxt[ty * Tx + tx] = best;
            }
        int *t = cur; cur = nxt; nxt = t;
    }
    for (int i = 0; i < n; ++i) {
        int L = cur[i];
        uint32_t mask = tile_mask[i];
        if (L >= 1) mask |= 1u;                          /* every node above depth L splits */
        if (L >= 2) mask |= 0x1Eu;
        if (L >= 3) mask |= 0x1FFFE0u;
        tile_mask[i] = mask;
        if (tile_level) tile_level[i] = (uint8_t)L;
    }
    uint64_t h[4];
    levels_and_hist_from_masks(width, height, tile_mask, cell_level, h);
    if (hist) for (int k = 0; k < 4; ++k) hist[k] = (uint32_t)h[k];
    if (scales) {
        double num = 0.0, den = 0.0;
        for (int k = 0; k < 4; ++k) { num += (double)k * (double)h[k]; den += (double)h[k]; }
        double w = den > 0.0 ? num / den : 0.0;
        double s2 = pow(2.0, w - (double)delta2), s3 = pow(2.0, w - (double)delta3);
        s2 = s2 < 0.25 ? 0.25 : (s2 > 1.0 ? 1.0 : s2);
        s3 = s3 < 0.25 ? 0.25 : (s3 > 1.0 ? 1.0 : s3);
        scales[0] = (float)w; scales[1] = (float)s2; scales[2] = (float)s3;
    }
    free(cur); free(nxt);
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O11 temporal tile state ("tiles computed in frame F_t guide ...     */
/* F_t+1", P:61 split / merge thresholds, "tiles may change by only one level per frame"). */
/* Reading A26: a node that was NOT split in the previous frame splits iff          */
/* metric > split threshold; a node that WAS split merges iff metric < merge threshold, with    */
/* merge <= split (a hysteresis band in which a node keeps its state; P:61's sentence "split    */
/* thresholds being smaller than the merge thresholds" read literally would make a node in the  */
/* band flip every frame, against its stated purpose).  Evaluation is top-down as in O6.  Then  */
/* the depth of each base tile is limited to prev_depth +- max_step: a deeper tree is truncated */
/* (bits below the limit cleared), a shallower one is refined uniformly to the limit.           */
/* metric vs threshold: above = 1 -> metric > thr, above = 0 -> metric < thr                    */
static int node_cmp(const qt_args *a, int x0, int y0, int side, uint32_t var_thr, float corner_thr,
                    int above)
{
    int x1 = x0 + side, y1 = y0 + side;
    if (x1 > a->width) x1 = a->width;
    if (y1 > a->height) y1 = a->height;
    if (a->metric == 0) {
        uint64_t n = 0, s1[3] = {0, 0, 0}, s2[3] = {0, 0, 0};
        for (int y = y0; y < y1; ++y)
            for (int x = x0; x < x1; ++x) {
                const float *px = a->image + 4 * ((size_t)y * a->width + x);
                for (int c = 0; c < 3; ++c) {
                    uint64_t q = quant8(px[c]);
                    s1[c] += q;
                    s2[c] += q * q;
                }
                ++n;
            }
        uint64_t lhs = 0, rhs = (uint64_t)var_thr * n * n;
        for (int c = 0; c < 3; ++c) lhs += n * s2[c] - s1[c] * s1[c];
        return above ? lhs > rhs : lhs < rhs;
    }
    int xs[4] = {x0, x1 - 1, x0, x1 - 1}, ys[4] = {y0, y0, y1 - 1, y1 - 1};
    static const int pa[6] = {0, 0, 0, 1, 1, 2}, pb[6] = {1, 2, 3, 2, 3, 3};
    float sum = 0.0f;
    for (int k = 0; k < 6; ++k) {
        const float *A = a->image + 4 * ((size_t)ys[pa[k]] * a->width + xs[pa[k]]);
        const float *B = a->image + 4 * ((size_t)ys[pb[k]] * a->width + xs[pb[k]]);
        float dr = A[0] - B[0], dg = A[1] - B[1], db = A[2] - B[2];
        float sq = dr * dr;
        sq = sq + dg * dg;
        sq = sq + db * db;
        float root = sqrtf(sq);
        sum = k == 0 ? root : sum + root;
    }
    float D = sum * (1.0f / 6.0f);
    return above ? D > corner_thr : D < corner_thr;
}

typedef struct {
    uint32_t var_split, var_merge;
    float corner_split, corner_merge;
} hyst_args;

/* split state of a node this frame given its state in the previous frame                       */
static int node_state(const qt_args *a, const hyst_args *h, int x0, int y0, int side, int was_split)
{
    if (x0 >= a->width || y0 >= a->height) return 0;     /* wholly outside the image (A17) */
    if (was_split) return !node_cmp(a, x0, y0, side, h->var_merge, h->corner_merge, 0);
    return node_cmp(a, x0, y0, side, h->var_split, h->corner_split, 1);
}

int32_t oracle_quadtree_temporal(const float *image, int32_t width, int32_t height, int32_t metric,
                                 uint32_t var_split, uint32_t var_merge, float corner_split,
                                 float corner_merge, int32_t max_step, const uint32_t *prev_mask,
                                 uint32_t *tile_mask, uint8_t *cell_level, uint32_t *hist)
{
    qt_args a = {image, width, height, metric, var_split, corner_split};
    hyst_args hy = {var_split, var_merge, corner_split, corner_merge};
    int Tx = (width + 63) / 64, Ty = (height + 63) / 64;
    for (int ty = 0; ty < Ty; ++ty)
        for (int tx = 0; tx < Tx; ++tx) {
            int X = tx * 64, Y = ty * 64;
            uint32_t prev = prev_mask ? prev_mask[ty * Tx + tx] : 0u, mask = 0;
            if (node_state(&a, &hy, X, Y, 64, (int)(prev & 1u))) {
                mask |= 1u;
                for (int c = 0; c < 4; ++c) {
                    int cx = X + 32 * (c & 1), cy = Y + 32 * (c >> 1);
                    if (!node_state(&a, &hy, cx, cy, 32, (int)((prev >> (1 + c)) & 1u))) continue;
                    mask |= 1u << (1 + c);
                    for (int g = 0; g < 4; ++g) {
                        int gx = cx + 16 * (g & 1), gy = cy + 16 * (g >> 1);
                        if (node_state(&a, &hy, gx, gy, 16, (int)((prev >> (5 + 4 * c + g)) & 1u)))
                            mask |= 1u << (5 + 4 * c + g);
                    }
                }
            }
            if (prev_mask && max_step > 0) {             /* at most max_step levels per frame */
                int pd = mask_depth(prev), d = mask_depth(mask);
                if (d > pd + max_step) {
                    int lim = pd + max_step;             /* truncate below depth lim */
                    mask &= lim == 0 ? 0u : (lim == 1 ? 0x1u : (lim == 2 ? 0x1Fu : 0x1FFFFFu));
                } else if (d < pd - max_step) {
                    int lim = pd - max_step;             /* refine uniformly to depth lim */
                    mask |= lim >= 1 ? 1u : 0u;
                    mask |= lim >= 2 ? 0x1Eu : 0u;
                    mask |= lim >= 3 ? 0x1FFFE0u : 0u;
                }
            }
            tile_mask[ty * Tx + tx] = mask;
        }
    uint64_t h[4];
    levels_and_hist_from_masks(width, height, tile_mask, cell_level, h);
    if (hist) for (int k = 0; k < 4; ++k) hist[k] = (uint32_t)h[k];
    return 0;
}

/* ---------------------------------------------------------------------------------------- */
/* O8 reprojection ("reprojecting pixels using the nearest available depth and the       */
/* previous view-projection matrix"; P:53 first-fragment depth reused).  All fp32, operations  */
/* exactly in this order; every fmaf is a real fused op; nothing else is contracted.           */
/* ---------------------------------------------------------------------------------------- */
int32_t oracle_reproject(int32_t width, int32_t height, const float *M, float depth_threshold,
                         const float *background, const float *prev_trans,
                         const float *prev_depth, const float *cur_depth, float *out_trans,
                         float *out_depth, float *out_final, uint8_t *accept,
                         uint32_t *reject_list, uint32_t *reject_count)
{
    uint32_t nrej = 0;
    float fW = (float)width, fH = (float)height;
    float inv_w = 1.0f / fW, inv_h = 1.0f / fH;
    for (int y = 0; y < height; ++y)
        for (int x = 0; x < width; ++x) {
            size_t p = (size_t)y * width + x;
            float xn = fmaf(2.0f * ((float)x + 0.5f), inv_w, -1.0f);
            float yn = fmaf(2.0f * ((float)y + 0.5f), inv_h, -1.0f);
            float d = cur_depth[p];
            float c[4];
            for (int k = 0; k < 4; ++k)
                c[k] = fmaf(M[4 * k + 0], xn,
                            fmaf(M[4 * k + 1], yn, fmaf(M[4 * k + 2], d, M[4 * k + 3])));
            int ok = c[3] > 0.0f;
            float d_e = 0.0f;
            size_t q = 0;
            if (ok) {
                float xp = c[0] / c[3], yp = c[1] / c[3];
                d_e = c[2] / c[3];
                float fx = floorf((xp + 1.0f) * 0.5f * fW);
                float fy = floorf((yp + 1.0f) * 0.5f * fH);
                ok = (fx >= 0.0f) && (fx < fW) && (fy >= 0.0f) && (fy < fH);
                if (ok) {
                    q = (size_t)(int)fy * width + (size_t)(int)fx;
                    ok = fabsf(prev_depth[q] - d_e) <= depth_threshold;
                }
            }
            if (ok) {
                for (int k = 0; k < 4; ++k) out_trans[4 * p + k] = prev_trans[4 * q + k];
                if (out_depth) out_depth[p] = d_e;
                if (out_final) {
                    float t = prev_trans[4 * q + 3];
                    for (int k = 0; k < 3; ++k)
                        out_final[4 * p + k] =
                            (float)((double)prev_trans[4 * q + k] + (double)t * (double)background[k]);
                    out_final[4 * p + 3] = (float)(1.0 - (double)t);
                }
                if (accept) accept[p] = 1;
            } else {
                if (accept) accept[p] = 0;
                if (reject_list) reject_list[nrej] = (uint32_t)p;
                ++nrej;
            }
        }
    if (reject_count) *reject_count = nrej;
    return 0;
}

/* O8b (NEXT-4, SURVEY 8(f) rank 4 "bilinear-filtered reprojection"; reading A28).  The paper
 * itself fetches the nearest pixel; this variant differs from O8 only in the fetch of
 * the previous result:
 *   - the transform, the nearest previous pixel q, the on-screen test and the disocclusion test
 *     |prev_depth[q] - d_e| <= tau are O8's, unchanged, so accept / reject_list / out_depth are
 *     identical to O8's;
 *   - with (u, v) the continuous previous-frame position (pixel centres at +0.5), the four taps
 *     are x0 = floor(u - 0.5), x1 = x0 + 1 (both clamped to the image), same in y, with weights
 *     wx = (u - 0.5) - floor(u - 0.5), wy likewise;
 *   - the filtered value is used iff ALL FOUR taps pass the disocclusion test against d_e
 *     (no blending across a depth discontinuity); otherwise the nearest pixel is kept (O8);
 *   - fp32 in one fixed order: top = fma(wx, t01 - t00, t00), bot = fma(wx, t11 - t10, t10),
 *     out = fma(wy, bot - top, top), per channel of (C_t, T_tot).
 * Pins (tests/test_oracle_pins.py): whole-pixel shifts reduce to O8 bit for bit; a constant image
 * stays constant; a dyadic linear ramp is reproduced exactly at a quarter-pixel shift; a depth
 * edge falls back to O8 for exactly the pixels whose 2x2 footprint straddles it.               */
int32_t oracle_reproject_bilinear(int32_t width, int32_t height, const float *M,
                                  float depth_threshold, const float *background,
                                  const float *prev_trans, const float *prev_depth,
                                  const float *cur_depth, float *out_trans, float *out_depth,
                                  float *out_final, uint8_t *accept, uint32_t *reject_list,
                                  uint32_t *reject_count, uint8_t *filtered)
{
    uint32_t nrej = 0;
    float fW = (float)width, fH = (float)height;
    float inv_w = 1.0f / fW, inv_h = 1.0f / fH;
    for (int y = 0; y < height; ++y)
        for (int x = 0; x < width; ++x) {
            size_t p = (size_t)y * width + x;
            float xn = fmaf(2.0f * ((float)x + 0.5f), inv_w, -1.0f);
            float yn = fmaf(2.0f * ((float)y + 0.5f), inv_h, -1.0f);
            float d = cur_depth[p];
            float c[4];
            for (int k = 0; k < 4; ++k)
                c[k] = fmaf(M[4 * k + 0], xn,
                            fmaf(M[4 * k + 1], yn, fmaf(M[4 * k + 2], d, M[4 * k + 3])));
            int ok = c[3] > 0.0f;
            float d_e = 0.0f, u = 0.0f, v = 0.0f;
            size_t q = 0;
            if (ok) {
                float xp = c[0] / c[3], yp = c[1] / c[3];
                d_e = c[2] / c[3];
                u = (xp + 1.0f) * 0.5f * fW;
                v = (yp + 1.0f) * 0.5f * fH;
                float fx = floorf(u), fy = floorf(v);
                ok = (fx >= 0.0f) && (fx < fW) && (fy >= 0.0f) && (fy < fH);
                if (ok) {
                    q = (size_t)(int)fy * width + (size_t)(int)fx;
                    ok = fabsf(prev_depth[q] - d_e) <= depth_threshold;
                }
            }
            if (filtered) filtered[p] = 0;
            if (ok) {
                float t[4];
                for (int k = 0; k < 4; ++k) t[k] = prev_trans[4 * q + k];
                /* the 2x2 footprint around (u - 0.5, v - 0.5) */
                float ub = u - 0.5f, vb = v - 0.5f;
                float x0f = floorf(ub), y0f = floorf(vb);
                float wx = ub - x0f, wy = vb - y0f;
                int x0 = (int)x0f, y0 = (int)y0f, x1 = x0 + 1, y1 = y0 + 1;
                if (x0 < 0) x0 = 0;
                if (x1 > width - 1) x1 = width - 1;
                if (y0 < 0) y0 = 0;
                if (y1 > height - 1) y1 = height - 1;
                size_t q00 = (size_t)y0 * width + x0, q01 = (size_t)y0 * width + x1;
                size_t q10 = (size_t)y1 * width + x0, q11 = (size_t)y1 * width + x1;
                int all4 = fabsf(prev_depth[q00] - d_e) <= depth_threshold &&
                           fabsf(prev_depth[q01] - d_e) <= depth_threshold &&
                           fabsf(prev_depth[q10] - d_e) <= depth_threshold &&
                           fabsf(prev_depth[q11] - d_e) <= depth_threshold;
                if (all4) {
                    for (int k = 0; k < 4; ++k) {
                        float t00 = prev_trans[4 * q00 + k], t01 = prev_trans[4 * q01 + k];
                        float t10 = prev_trans[4 * q10 + k], t11 = prev_trans[4 * q11 + k];
                        float top = fmaf(wx, t01 - t00, t00);
                        float bot = fmaf(wx, t11 - t10, t10);
                        t[k] = fmaf(wy, bot - top, top);
                    }
                    if (filtered) filtered[p] = 1;
                }
                for (int k = 0; k < 4; ++k) out_trans[4 * p + k] = t[k];
                if (out_depth) out_depth[p] = d_e;
                if (out_final) {
                    for (int k = 0; k < 3; ++k)
                        out_final[4 * p + k] =
                            (float)((double)t[k] + (double)t[3] * (double)background[k]);
                    out_final[4 * p + 3] = (float)(1.0 - (double)t[3]);
                }
                if (accept) accept[p] = 1;
            } else {
                if (accept) accept[p] = 0;
                if (reject_list) reject_list[nrej] = (uint32_t)p;
                ++nrej;
            }
        }
    if (reject_count) *reject_count = nrej;
    return 0;
}

int32_t oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}
