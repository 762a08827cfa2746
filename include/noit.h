/* noit.h -- C ABI of libnoit.so: B200-native (sm_100a) neural order-independent-transparency
 * resolve, the hot path of STAR-NT (arxiv/paper_2606_16747).
 *
 * Citations: "P:n" = line n of PAPER.md; "S:8(x)" = SURVEY.md section 8(x); readings A1..A24
 * and operation definitions O1..O9 are restated in DESIGN.md.
 *
 * Conventions
 *  - Unless a function name ends in `_host`, every pointer INSIDE a descriptor is a DEVICE
 *    pointer owned by the caller (e.g. a PyTorch tensor).  The library never frees or retains
 *    caller memory.  Descriptors themselves, `M`, `background`, weights are HOST memory.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls enqueue
 *    work on it and return without synchronising (except the `_host` entry points, which
 *    return after their results are in the caller's host buffers).
 *  - Every entry point returns noit_status.  Host-checkable errors (NULL pointers, bad sizes,
 *    unknown enums, missing weights, misalignment) are detected BEFORE any launch and leave all
 *    outputs untouched.  CUDA errors map to NOIT_ERR_CUDA with text in noit_last_error().
 *  - Device-side preconditions are documented, not checked by the hot entry points: offsets
 *    non-decreasing with offsets[0] == 0 and offsets[P] == num_fragments (a malformed CSR drives
 *    the bulk copies out of bounds -- noit_validate_fragbuf checks it on demand); depth finite;
 *    alpha in [0,1]; inputs and outputs do not alias (except noit_reproject's cur_depth ==
 *    prev_depth, which is allowed).
 *  - A context belongs to the device that was current at noit_create; calling a launching entry
 *    point with another device current is NOIT_ERR_CUDA (nothing is launched).
 *  - Allocation and synchronisation: entry points never allocate caller-visible memory.  Context
 *    scratch is allocated with cudaMalloc the FIRST time a call needs it and when a later call
 *    needs more (noit_resolve with cell_level / pass_scales: G buffers and the tile summary;
 *    noit_quadtree_balance: one word per tile; noit_resolve_host: the staging area, two streams
 *    and their events); growing a scratch buffer first synchronises `stream`.  Steady-state calls
 *    (same sizes) neither allocate nor synchronise, and can be captured in a CUDA graph after one
 *    eager call.  noit_resolve_host and noit_validate_fragbuf synchronise by definition.
 *  - A context is not thread-safe; distinct contexts are independent.  Calls on ONE context must
 *    be stream-ordered with respect to each other (same stream, or ordered by events): the
 *    context owns small device scratch (work counters, S7 intermediates) that launches share.
 *  - There is no CPU fallback and no other backend.
 *
 * Fragment buffer layout (S:8(a) S0; stands in for the paper's three raster passes P:55):
 *    offsets u32[P+1]   row-major pixels p = y*W + x, offsets[0] = 0, non-decreasing
 *    depth   f32[F]     smaller = nearer (A9); 16-byte aligned base
 *    rgba    half[F][4] or float[F][4], STRAIGHT colour, .w = alpha (A8); 16-byte aligned base
 *  Fragments of a pixel are contiguous and in submission order; "fragment index" = position.
 */
#ifndef NOIT_H
#define NOIT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct noit_ctx noit_ctx; /* opaque; owns the device copy of the weights + small scratch */

typedef enum {
    NOIT_OK = 0,
    NOIT_ERR_NULL = 1,        /* a required pointer is NULL                                   */
    NOIT_ERR_SIZE = 2,        /* width/height <= 0, P+1 or F overflow u32, count != 771, ...  */
    NOIT_ERR_FORMAT = 3,      /* unknown enum value or misaligned pointer                     */
    NOIT_ERR_NO_WEIGHTS = 4,  /* MLP needed but noit_set_weights was never called             */
    NOIT_ERR_CUDA = 5,        /* a CUDA runtime call failed; see noit_last_error              */
    NOIT_ERR_UNSUPPORTED = 6  /* valid request this build does not implement                  */
} noit_status;

enum { NOIT_RGBA_F16 = 0, NOIT_RGBA_F32 = 1 };     /* fragment colour format                  */
enum { NOIT_MLP_FP32 = 0, NOIT_MLP_BF16 = 1 };     /* weight precision (A6)                   */
enum { NOIT_QT_VARIANCE = 0, NOIT_QT_CORNER = 1 }; /* quadtree split metric (A14)             */

#define NOIT_MLP_PARAMS 771        /* 5->32->16->3 with biases (A4)                     */
#define NOIT_DFAOIT_PARAMS 931     /* 10->32->16->3: the comparison system's network   */
#define NOIT_ABSENT 0xFFFFFFFFu    /* idx1/idx2 of a missing layer                            */

typedef struct {
    int32_t width, height;
    uint32_t num_fragments;        /* F = offsets[P]                                          */
    int32_t color_fmt;             /* NOIT_RGBA_F16 | NOIT_RGBA_F32                           */
    const uint32_t* offsets;       /* [P+1]                                                   */
    const float* depth;            /* [F]                                                     */
    const void* rgba;              /* [F][4]                                                  */
} noit_fragbuf;

/* Optional check of the device-side CSR preconditions (not on the hot path): offsets[0] == 0,
 * offsets non-decreasing, offsets[P] == num_fragments.  Runs a small kernel on `stream`,
 * synchronises it and returns NOIT_OK, or NOIT_ERR_FORMAT with the first offending pixel in
 * noit_last_error.  Pointers as in every noit_fragbuf: device memory.                        */
noit_status noit_validate_fragbuf(noit_ctx* ctx, const noit_fragbuf* fb, void* stream);

/* ---- context ------------------------------------------------------------------------------ */
noit_status noit_create(noit_ctx** out);
void noit_destroy(noit_ctx* ctx);
/* host array of 771 floats: W1[32][5], b1[32], W2[16][32], b2[16], W3[3][16], b3[3] (row =
 * output neuron).  precision NOIT_MLP_BF16 rounds every weight to bf16 (RNE) once, here,
 * and widens it back; activations and accumulation stay fp32 (A6).  Synchronous.             */
noit_status noit_set_weights(noit_ctx* ctx, const float* host_w, int32_t count, int32_t precision);
/* copies the EFFECTIVE weights (after the rounding above) into host_out[771].                */
noit_status noit_get_weights(const noit_ctx* ctx, float* host_out, int32_t count);
/* static or ctx-owned string; never freed by the caller; ctx may be NULL.                    */
const char* noit_last_error(const noit_ctx* ctx);
/* number of kernels this context has launched so far (bench.py's gpu_launches).              */
uint64_t noit_launch_count(const noit_ctx* ctx);
/* Diagnostics.  libnoit_debug.so is the same library with the staged resolve kernel compiled with
 * -DNOIT_DEBUG_BOUNDS: every shared-memory range a scan, a layer fetch or a bulk copy touches is
 * checked against the warp's stage and every fragment range against [0, F), violations are
 * counted on the device (the access is still made).  This call synchronises the device and
 * writes the count since noit_create to *host_count; the release build always reports 0.        */
noit_status noit_debug_bounds_violations(noit_ctx* ctx, uint32_t* host_count);

/* ---- S1-S3: k=2 nearest-layer selection + tail reduction + features
 * Any output pointer may be NULL (skipped); at least one must be set.
 *   idx1, idx2  LOCAL index (j - offsets[p]) of the nearest / 2nd nearest fragment under the
 *               key (depth, index), NOIT_ABSENT if the layer is missing (O1)
 *   count       N = n_p
 *   layer1/2    straight RGBA of the two layers, zeros if absent
 *   depth1      depth of layer 1, 1.0f for an empty pixel (A10)
 *   tail_raw    C_acc.rgb = sum a_i C_i, A_tail = sum a_i, T_tail = prod (1-a_i) over the tail
 *               (every fragment that is not layer 1 or 2) (O2)
 *   features    x = [N, T_tail, C_acc / A_tail] (zeros for the colour if A_tail == 0) (O3)  */
typedef struct {
    uint32_t* idx1; uint32_t* idx2; uint32_t* count;   /* [P] each                            */
    float* layer1; float* layer2;                      /* [P][4]                              */
    float* depth1;                                     /* [P]                                 */
    float* tail_raw;                                   /* [P][5]                              */
    float* features;                                   /* [P][5]                              */
} noit_layers;
noit_status noit_build_features(noit_ctx* ctx, const noit_fragbuf* fb, const noit_layers* out,
                                void* stream);

/* ---- S4 alone: f(x) = relu(W3 relu(W2 relu(W1 x + b1) + b2) + b3) on n rows (A3).
 * No has_tail gating.  features [n][5] -> tail_rgb [n][3].  n == 0 is a no-op.               */
noit_status noit_infer(noit_ctx* ctx, const float* features, uint32_t n, float* tail_rgb,
                       void* stream);

/* ---- NEXT-4 (comparison variant): the network the comparison system DFAOIT evaluates, 10 input
 * features -> 32 -> 16 -> 3 with a SIGMOID output ("differs only in the output activation",
 * P:99-104), 931 parameters laid out W1[32][10], b1[32], W2[16][32], b2[16], W3[3][16], b3[3]
 * in HOST memory (fp32, used as given).  It exists to measure the inference-cost ratio of the
 * 10 -> 5 feature reduction with the same kernel shape as noit_infer; how DFAOIT forms
 * its ten features is only summarised in the paper, so nothing here computes them.
 * features [n][10] -> rgb [n][3] (device).  n == 0 is a no-op.                               */
noit_status noit_infer_dfaoit(noit_ctx* ctx, const float* host_w, int32_t count, const float* features,
                              uint32_t n, float* rgb, void* stream);

/* ---- S1-S5 fused resolve (Eq. 4; O5); S7 when cell_level is set (O7);
 * S9 when pixel_list is set (O9).
 *   C_t   = a1 C1 + (1-a1) a2 C2 + [A_tail > 0] T_2 f(x),  T_2 = (1-a1)(1-a2)
 *   T_tot = T_2 T_tail;  C_p = C_t + T_tot C_b
 *   out_trans  [P][4] = (C_t, T_tot)      out_final [P][4] = (C_p, 1 - T_tot)
 *   out_depth1 [P]    = depth of layer 1, 1.0f if empty.   No clamping anywhere (A11).
 * At least one output must be non-NULL; out_trans/out_final need 16-byte alignment.
 * Adaptive (S7): cell_level[ceil(H/8)*ceil(W/8)] from noit_quadtree gives each 8x8 cell its
 * leaf level; lod = level_to_lod[level] in {0,1,2}; lod 1 reads `half` (ceil(W/2) x
 * ceil(H/2)), lod 2 reads `quarter`; layer 1 always comes from `full`; layer 2
 * (premultiplied) and the raw tail accumulators of the coarse pixels are bilinearly upsampled
 * with taps clamped to the pixel's own leaf, then features, MLP and composite run at full
 * resolution (A18-A20).  A level that maps to lod k > 0 requires the matching buffer.
 * pixel_list/pixel_count (device): resolve only the listed pixels (count read on the device),
 * leave the others untouched; not combinable with cell_level.
 * Frame-global resolution control (NEXT-1, the paper's own scheme P:78-87; O7g, A27): when
 * pass_scales (device, float[3] = {w, s_2, s_3} as written by noit_quadtree_balance) is set,
 * pass 2 (layer 2) is taken at lod2 and pass 3 (tail statistics, N) at lod3 for the WHOLE
 * frame, lod_p = 0 if s_p > 2^-0.5, 1 if s_p > 2^-1.5, else 2, decided on the device (no host
 * round trip); lod 0 = the pixel's own full-resolution list, lod 1 / 2 = bilinear upsample from
 * `half` / `quarter` (both required), taps clamped to the image.  Not combinable with
 * cell_level or pixel_list.                                                                  */
typedef struct {
    noit_fragbuf full;
    const noit_fragbuf* half;        /* NULL => no S7                                          */
    const noit_fragbuf* quarter;
    const uint8_t* cell_level;       /* NULL => plain resolve                                  */
    uint8_t level_to_lod[4];         /* default {2,1,0,0}: 64-leaf->1/4, 32->1/2, 16/8->full   */
    float background[3];             /* C_b (A11)                                              */
    const uint32_t* pixel_list;      /* [<= P] pixel indices, or NULL                          */
    const uint32_t* pixel_count;     /* device scalar: entries of pixel_list to process        */
    float* out_trans; float* out_final; float* out_depth1;
    const float* pass_scales;        /* device {w, s_2, s_3}, or NULL                          */
    const float* background_image;   /* device [P][4] per-pixel C_b (.xyz used; NEXT-4) or NULL:
                                        replaces `background` in out_final; 16-byte aligned    */
} noit_resolve_desc;
noit_status noit_resolve(noit_ctx* ctx, const noit_resolve_desc* desc, void* stream);

/* Same as noit_resolve (plain, no S7/S9) but EVERY pointer in `desc` is a HOST pointer: the
 * call stages the fragment buffer into context-owned device memory (grown on demand, kept
 * between calls), runs the fused kernel and copies the requested outputs back.  Returns after
 * the outputs are in host memory.  Pinned host memory makes the copies asynchronous DMA.
 * Frames above 32 MB are pipelined in up to 8 bands of whole 32-pixel tiles: the host->device
 * copies, the kernels (on `stream`) and the device->host copies run on three streams chained by
 * events, so the outputs travel back while later inputs still arrive; results are bit-identical
 * to the single launch.  The call reads host_desc->full.offsets on the host to cut the bands
 * (NOIT_ERR_FORMAT if they are not monotone within [0, F]).                                    */
noit_status noit_resolve_host(noit_ctx* ctx, const noit_resolve_desc* host_desc, void* stream);

/* ---- NEXT-4: the DFAOIT resolve, the method STAR-NT starts from and is compared with (P:99-104,
 * Eq. 3; O12, reading A29).  Same fragment buffer, same k = 2 selection and tail scan as
 * noit_resolve (plain, whole frame), but
 *   x (10)  = [ a1 C1 + (1-a1) a2 C2 (3),  C_avg (3) and alpha_avg (1) of the n-2 tail fragments,
 *               C_acc = sum_tail a_i C_i (3) ]          (all tail entries 0 when n <= 2)
 *   C_t     = sigmoid network 10 -> 32 -> 16 -> 3 (931 parameters, host_w as in noit_infer_dfaoit)
 *             evaluated on x for every pixel with n >= 1; 0 for an empty pixel
 *   T_tot   = prod over ALL fragments (1 - a_i);  C_p = C_t + T_tot C_b          (Eq. 3)
 *   out_trans [P][4] = (C_t, T_tot), out_final [P][4] = (C_p, 1 - T_tot), out_depth1 [P] as in
 *   noit_resolve; features10 [P][10] (optional, 8-byte aligned) receives x.
 * The two exact layers are NOT decoupled from the prediction (the limitation P:106 names): this
 * entry point exists to measure the cost of the 10-feature resolve against the 5-feature one
 * and as the reference point of Eq. 4.  host_w: 931 floats, host memory.               */
noit_status noit_resolve_dfaoit(noit_ctx* ctx, const noit_fragbuf* fb, const float* host_w, int32_t count,
                                const float* background /*[3], host*/, float* out_trans, float* out_final,
                                float* out_depth1, float* features10, void* stream);

/* ---- S6 quadtree split (sizes 64->8 per BASELINE.json cfg4, A13; O6).
 * Base tiles 64x64 anchored at (0,0), Tx = ceil(W/64), Ty = ceil(H/64).  A node at level
 * l < 3 with >= 1 in-image pixel splits iff metric(node) > threshold (strict); evaluated
 * top-down.
 *   NOIT_QT_VARIANCE: q_c = rint(255 clamp(c,0,1)); split iff
 *       sum_c (n S2_c - S1_c^2) > var_threshold_q n^2  (exact integers) (A14, A16)
 *   NOIT_QT_CORNER: D = (1/6) sum over the 6 pairs of the node's 4 in-image corner
 *       pixels of the Euclidean RGB distance (fp32, fixed order); split iff D > corner_threshold
 *   tile_mask [Ty*Tx]: bit 0 root; bit 1+c level-1 child c = cx+2cy; bit 5+4c+g level-2 child
 *   cell_level [ceil(H/8)*ceil(W/8)]: level 0..3 of the leaf containing the 8x8 cell
 *   level_hist [4] (overwritten by the call): leaves per level with >= 1 in-image pixel */
typedef struct {
    int32_t metric;
    uint32_t var_threshold_q;      /* summed-over-channels variance, 8-bit units squared      */
    float corner_threshold;
} noit_qt_params;
noit_status noit_quadtree(noit_ctx* ctx, const float* image /*[P][4]*/, int32_t width,
                          int32_t height, const noit_qt_params* params, uint32_t* tile_mask,
                          uint8_t* cell_level, uint32_t* level_hist, void* stream);

/* ---- NEXT-3: noit_quadtree in the paper's own geometry: 16x16 base tiles, four levels
 * down to 2x2 leaves; same metrics, mask layout and top-down rule.
 *   tile_mask [ceil(H/16)*ceil(W/16)], cell_level [ceil(H/2)*ceil(W/2)] (leaf level of every 2x2
 *   cell), level_hist [4] (zeroed by the call).                                              */
noit_status noit_quadtree16(noit_ctx* ctx, const float* image /*[P][4]*/, int32_t width,
                            int32_t height, const noit_qt_params* params, uint32_t* tile_mask,
                            uint8_t* cell_level, uint32_t* level_hist, void* stream);

/* ---- NEXT-2: temporal tile state ("tiles computed in frame F_t guide ... F_t+1", P:61
 * split / merge thresholds, "tiles may change by only one level per frame"; O11, A26).
 * noit_quadtree with a memory: a node that was NOT split in prev_tile_mask splits iff
 * metric > split threshold; a node that WAS split merges iff metric < merge threshold.  The
 * rule is defined for either order of the two thresholds: merge <= split is the stabilising
 * order (inside the band a node keeps its state, reading A26); merge > split is P:61's sentence
 * read literally ("split thresholds being smaller than the merge thresholds"): a node whose
 * metric lies strictly between the two then changes state every frame.  Then the depth of every base tile
 * is limited to its previous depth +- max_level_step (deeper: truncated; shallower: refined
 * uniformly).  prev_tile_mask == NULL: no history, identical to noit_quadtree with the split
 * thresholds.  prev_tile_mask must not alias tile_mask.  max_level_step in [0, 3], 0 = no
 * limit (the paper: 1).  Outputs as in noit_quadtree.                                       */
typedef struct {
    int32_t metric;
    uint32_t var_split_q, var_merge_q;      /* summed-over-channels variance, 8-bit units squared */
    float corner_split, corner_merge;
    int32_t max_level_step;
} noit_qt_temporal_params;
noit_status noit_quadtree_temporal(noit_ctx* ctx, const float* image /*[P][4]*/, int32_t width,
                                   int32_t height, const noit_qt_temporal_params* params,
                                   const uint32_t* prev_tile_mask, uint32_t* tile_mask,
                                   uint8_t* cell_level, uint32_t* level_hist, void* stream);

/* ---- NEXT-1: quadtree consistency + demand index (O10, reading A25).
 * "neighboring tiles may differ by at most one refinement level ... two relaxation iterations
 * (k=2) are sufficient": the level of a base tile is the depth of its subtree (0 = not
 * split .. 3 = a grandchild split); one iteration is the Jacobi step L_i <- max(L_i, max over the
 * 4 edge neighbours of L_j - 1); a tile that rises to level L is refined uniformly to depth L.
 *   tile_mask  [Ty*Tx] in/out (device): masks from noit_quadtree, updated in place
 *   tile_level [Ty*Tx] out, optional: balanced level of every base tile
 *   cell_level, level_hist: as in noit_quadtree, recomputed from the balanced masks (optional;
 *              level_hist is zeroed by the call)
 *   scales     [3] out, optional (needs level_hist): w = sum l N_l / sum N_l,
 *              s_2 = clamp(2^(w - delta2), 0.25, 1), s_3 likewise with delta3 (Eq. 2 P:80;
 *              the paper's delta2 = 2.2, delta3 = 3.0), fp32
 * iterations in [0, 16] (the paper's k = 2).                                                  */
noit_status noit_quadtree_balance(noit_ctx* ctx, int32_t width, int32_t height, int32_t iterations,
                                  float delta2, float delta3, uint32_t* tile_mask,
                                  uint8_t* tile_level, uint8_t* cell_level, uint32_t* level_hist,
                                  float* scales, void* stream);

/* The same pass for callers that cannot allocate (CUDA-graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): arguments, outputs and results are exactly noit_quadtree_balance's, but the
 * kernel's scratch (balanced masks before they are published, finish ticket, histogram accumulators)
 * lives in a file-scope device array of the library instead of context scratch.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine, on its first use or later.
 *   limit   ceil(W/64) * ceil(H/64) <= NOIT_BALANCE_STATIC_MAX_TILES (16384 base tiles, e.g.
 *           8192 x 8192 pixels); beyond it NOIT_ERR_SIZE and nothing is launched
 *   cost    64.25 KB of device memory on every GPU that loads the library, until the process exits
 *   sharing ALL calls on a device share the array, whatever context or stream they come from: two
 *           calls that overlap on the GPU race (order them on one stream or with events).  The
 *           array keeps the last call's contents; the call clears what must start at zero itself.  */
#define NOIT_BALANCE_STATIC_MAX_TILES 16384
noit_status noit_quadtree_balance_static(noit_ctx* ctx, int32_t width, int32_t height, int32_t iterations,
                                         float delta2, float delta3, uint32_t* tile_mask,
                                         uint8_t* tile_level, uint8_t* cell_level, uint32_t* level_hist,
                                         float* scales, void* stream);

/* ---- S8 depth-based reprojection with disocclusion test (O8, A21-A23).
 * Per pixel, fp32 in a fixed order: NDC of the pixel centre and cur_depth -> M -> previous
 * pixel q and expected depth d_e; accept iff w > 0, q on screen and
 * |prev_depth[q] - d_e| <= depth_threshold.  Accepted: out_trans[p] = prev_trans[q] (bit
 * copy), out_depth[p] = d_e, accept[p] = 1, out_final[p] = (C_t + T_tot C_b, 1 - T_tot).
 * Rejected: accept[p] = 0, p appended to reject_list (order unspecified), outputs untouched.
 * M = VP_prev * VP_cur^-1, row-major, column vectors.  out_depth/out_final/accept/reject_list
 * may be NULL; reject_count (required) is zeroed by the call.
 * filter (NEXT-4, O8b / A28): NOIT_REPROJECT_NEAREST is the paper's fetch
 * (P:121).  NOIT_REPROJECT_BILINEAR changes only the value fetched for an ACCEPTED pixel: the
 * 2x2 footprint of prev_trans around the continuous previous position (taps clamped to the
 * image, weights wx, wy in fp32, top = fma(wx, t01 - t00, t00), bot likewise,
 * out = fma(wy, bot - top, top)) where all four taps pass the disocclusion test against d_e,
 * the nearest pixel elsewhere; accept, reject_list and out_depth are the same for both filters.
 * Any other value: NOIT_ERR_FORMAT.                                                            */
enum { NOIT_REPROJECT_NEAREST = 0, NOIT_REPROJECT_BILINEAR = 1 };
typedef struct {
    int32_t width, height;
    float M[16];
    float depth_threshold;
    float background[3];
    const float* prev_trans; const float* prev_depth; const float* cur_depth;
    float* out_trans; float* out_depth; float* out_final;
    uint8_t* accept;
    uint32_t* reject_list; uint32_t* reject_count;
    int32_t filter;
} noit_reproject_desc;
noit_status noit_reproject(noit_ctx* ctx, const noit_reproject_desc* desc, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* NOIT_H */
