/* gabsplat.h -- C ABI of libgabsplat: the differentiable tile-based rasterizer for 3D Gabor-based
 * primitives (3DGabSplat, arXiv 2508.05343), hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations are /root/reference/PAPER.md line numbers plus the equation they fall in.
 *
 * The four calls follow the paper's statement of the renderer ("transformation ...
 * splat ... tile-based colour-alpha blending"; :160 "tile-based rasterizer"):
 *
 *   gabsplat_preprocess       projection of every primitive to the image plane
 *                             (Eq.2 :91, Eq.3 :101, Eq.9 :145/:414, Eq.10-11 :150-154, SH colour :83)
 *   gabsplat_bin_sort         (tile | depth) instance keys, stable sort, per-tile ranges (:103, :160)
 *   gabsplat_render_forward   per-pixel front-to-back blend of 2D Gabor primitives (Eq.12 :158, Eq.13 :162)
 *   gabsplat_render_backward  the same computation in reverse: gradients of sum_p <dL/dC(p), C(p)> with
 *                             respect to every primitive parameter, including f and omega (:48, :129)
 *
 * General rules
 *   - Every pointer inside the structs below is a DEVICE pointer unless its name ends in _host.
 *     The structs themselves are HOST structs, read during the call (they may be freed afterwards).
 *   - All device buffers are allocated, owned and freed by the caller.  The library allocates only
 *     inside gabsplat_create (a few KB of device scratch) and frees it in gabsplat_destroy.
 *   - Inputs are never written.  Outputs are fully overwritten (gradients are zeroed by the library
 *     before accumulation).
 *   - Calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL = the legacy default
 *     stream) and return without synchronising, except where stated.
 *   - Return value: one of the GABSPLAT_* status codes.  Nothing is printed, nothing aborts.
 *   - There is no CPU fallback: on a machine without a usable sm_100 device gabsplat_create fails.
 *   - All floating-point storage is IEEE binary32, contiguous, row-major in the index order written.
 *   - Every device pointer must be 16-byte aligned (the kernels use 128-bit loads and stores).
 *
 * Value contract (activated inputs): scales > 0, rotations are unit quaternions (w,x,y,z)
 * and are not re-normalised, opacities in (0,1), weights omega_k in [0,1) (omega >= 0 is relied on by the
 * envelope reject), freqs in cycles per world unit (Eq.7 :127).  Gradients are with respect to these
 * activated values.
 */
#ifndef GABSPLAT_H_
#define GABSPLAT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GABSPLAT_OK 0
#define GABSPLAT_INVALID_ARG 1 /* null pointer, N < 0, K outside [0,8], sh_degree outside [0,3], variant outside [0,3], bad size/focal */
#define GABSPLAT_CAPACITY 2    /* instance buffers or workspace too small */
#define GABSPLAT_CUDA 3        /* a CUDA call failed; see gabsplat_last_error */
#define GABSPLAT_UNSUPPORTED 4 /* no sm_100 device */

#define GABSPLAT_MAX_K 8
#define GABSPLAT_TILE 16       /* tiles are 16x16 pixels */
#define GABSPLAT_CHUNK 1024    /* primitives per CTA of the projection kernel */
#define GABSPLAT_SH_COEFFS 16  /* storage stride of SH coefficients per primitive (degree 3) */

typedef struct gabsplat_ctx gabsplat_ctx;

/* Create / destroy a context bound to CUDA device `device`.  Host calls; create synchronises. */
int32_t gabsplat_create(gabsplat_ctx** out, int32_t device);
void gabsplat_destroy(gabsplat_ctx* ctx);
/* Static description of the last non-OK status on this context (never NULL). */
const char* gabsplat_last_error(const gabsplat_ctx* ctx);

/* Pinhole camera ("viewing transformation W", "Jacobian J of the affine approximation of the
 * projective transformation").  Pixel (x,y) is sampled at integer coordinates (x,y). */
typedef struct {
  int32_t width, height;
  float fx, fy, cx, cy;
  float world_to_cam[12]; /* row-major 3x4 [W | tau]:  t = W mu + tau */
  float z_near;           /* > 0 (INVALID_ARG otherwise: the depth key orders the bit patterns of positive
                             floats); primitives with t_z <= z_near are culled */
  float bg[3];            /* background colour, composited as C + T_final * bg */
} gabsplat_camera;

/* Variants of the primitive, bit flags of gabsplat_scene.variant:
 *  LINE_INTEGRAL  keep the per-component amplitude of the exact line integral along the ray that Eq.12 drops
 *                 (Eq.25-27; constants as corrected in DESIGN.md reading C4):
 *                 M = (1 - sum w_k) + sum w_k C2_k cos(phi_k),  C2_k = exp(-2 pi^2 f_z''^2 / S22)
 *  MIP_FILTER     Mip-Splatting's 2D filter in place of the 0.3 px^2 dilation: dilation 0.1 px^2 and
 *                 opacity scaled by sqrt(det Sigma2D / det(Sigma2D + 0.1 I)).
 * Both fold into the per-primitive record the blend kernels gather; conic_opacity[.][3] stays the input opacity. */
#define GABSPLAT_VARIANT_LINE_INTEGRAL 1
#define GABSPLAT_VARIANT_MIP_FILTER 2

/* The primitives.  N primitives, K Gabor components each. */
typedef struct {
  int32_t N, K, sh_degree;
  int32_t variant;        /* 0, or GABSPLAT_VARIANT_* flags or'ed; must be the same in every call of a pass */
  const float* means;     /* [N][3]                                                  */
  const float* scales;    /* [N][3]   Sigma = R diag(s^2) R^T  (:87)                 */
  const float* rotations; /* [N][4]   unit quaternion (w,x,y,z)                      */
  const float* opacities; /* [N]                                                     */
  const float* sh;        /* [N][16][3]  only the first (sh_degree+1)^2 rows are read */
  const float* freqs;     /* [N][K][3]  f_{k,i}  (Eq.7)                              */
  const float* weights;   /* [N][K]     omega_{k,i}  (Eq.7)                          */
} gabsplat_scene;

/* Outputs of gabsplat_preprocess, one entry per primitive.  tiles_touched and radius are written for every
 * primitive (0 = culled); every other array is written for the VISIBLE primitives only -- rows of culled primitives
 * are left untouched (unspecified; nothing in the library reads them).  `packed` is the record the blend kernels
 * gather. */
typedef struct {
  float* mean2d;           /* [N][2]  mu2D in pixels (:99)                                         */
  float* depth;            /* [N]     camera-space t_z; its bit pattern is the low half of the key */
  int32_t* radius;         /* [N]     ceil(3 sqrt(lambda_max)) of the dilated 2D covariance        */
  float* conic_opacity;    /* [N][4]  (a,b,c) = (Sigma2D + 0.3 I)^-1 (Eq.3), opacity               */
  float* rgb;              /* [N][3]  SH colour, clamped at 0 from below                           */
  uint8_t* rgb_clamped;    /* [N][4]  1 where the channel was clamped (4th byte 0)                 */
  float* freq2d;           /* [N][K][2]  f2D in cycles per pixel (Eq.10-11)                        */
  uint32_t* tiles_touched; /* [N]     number of tiles in the primitive's rectangle                */
  int32_t* rect;           /* [N][4]  xmin,ymin,xmax,ymax in tiles, max exclusive                  */
  float* packed;           /* [N][gabsplat_packed_floats(K)]  gather record, 16-byte aligned       */
  uint32_t* chunk_visible; /* [gabsplat_chunk_visible_count(N)] = [3][ceil(N / GABSPLAT_CHUNK)] (+1), all of it written
                              by gabsplat_preprocess -- size it with that function, the layout has grown before.
                              Per chunk of consecutive primitives: the number of
                              visible ones (what the binning needs to compact them in index order), then the
                              smallest and the largest bits(depth) among them (0xffffffff / 0 if none): the
                              depth range the binning buckets its sort by                               */
} gabsplat_projected;

/* Number of uint32 elements gabsplat_projected.chunk_visible must hold for N primitives. */
uint64_t gabsplat_chunk_visible_count(int32_t N);

/* Number of floats per primitive in gabsplat_projected.packed (a multiple of 4). */
int32_t gabsplat_packed_floats(int32_t K);

/* Tile binning state.  capacity = number of (key,id) slots the caller allocated. */
typedef struct {
  uint32_t* offsets;          /* [N]  scratch of the binning, one entry per visible primitive in depth order:
                                 the inclusive prefix of tiles_touched on images of more than 26000 tiles, of the
                                 estimated placement cost otherwise; the rest is not written             */
  uint64_t* keys;             /* [capacity]  sorted on return: (tile_id << 32) | bits(depth).  No later stage
                                 reads the keys: for images of at most 26000 tiles the pointer may be NULL
                                 and the keys are then not materialised                                */
  uint32_t* ids;              /* [capacity]  primitive index of each instance, same order            */
  uint32_t* tile_ranges;      /* [tiles_y*tiles_x][2]  [start,end) into keys/ids; (0,0) if empty     */
  uint32_t* tile_order;       /* [tiles_y*tiles_x]  the order in which the forward blend launches its CTAs:
                                 the tiles by descending list length, or by tile_work_hint (below)      */
  uint64_t capacity;
  uint32_t* num_instances;    /* [1]  device: D = total instance count                               */
  void* workspace;            /* device scratch, >= gabsplat_sort_workspace_bytes(N, capacity, W, H) bytes */
  uint64_t workspace_bytes;
  const uint32_t* tile_work_hint; /* optional (NULL: none), [tiles_y*tiles_x]: gabsplat_fwd_out.tile_work of an
                                 earlier render of (about) this view.  tile_order then follows min(hint, list
                                 length) instead of the list length.  A tile's time is set by how far it walks
                                 its list before its last pixel saturates, which the list length does not
                                 predict; a trainer that revisits its views keeps one hint array per view.
                                 It changes the launch order of the forward blend and nothing else.  It is
                                 IGNORED (tile_order = descending list length) for images of more than 26 000
                                 tiles, which take the one-byte radix path, and when capacity == 0.  What it
                                 gains was measured on an unchanged scene re-rendered from the same view, its
                                 best case; bench.py's headline step does not use it          */
} gabsplat_binning;

uint64_t gabsplat_sort_workspace_bytes(int32_t N, uint64_t capacity, int32_t width, int32_t height);

/* Forward outputs.  n_contrib[p] = 1-based position, within the tile list of pixel p, of the last
 * primitive that was blended at p (0 = none); its id is ids[tile_ranges[tile][0] + n_contrib - 1]. */
typedef struct {
  float* image;        /* [3][H][W] */
  float* final_T;      /* [H][W]    */
  uint32_t* n_contrib; /* [H][W]    */
  /* Optional (NULL for inference): device scratch of >= gabsplat_blend_state_bytes(...) bytes in which the
   * forward records, per half tile (one warp's 16x8 pixels), the list of primitives that were blended at one
   * of its pixels and a 128-bit mask of those pixels.  gabsplat_render_backward replays these lists in
   * reverse and REQUIRES them: it neither re-walks the tile lists nor re-takes any skip/stop decision. */
  void* blend_state;
  uint64_t blend_state_bytes;
  uint32_t* tile_work; /* optional (NULL: not written), [tiles_y*tiles_x]: list entries the tile consumed before all of
                          its pixels were finished (a multiple of the staging batch, at most the list length):
                          the tile_work_hint of a later gabsplat_bin_sort of the same view                      */
} gabsplat_fwd_out;

/* Bytes of gabsplat_fwd_out.blend_state for an image of this size and `capacity` instance slots
 * (worst case: every instance of a tile's list is blended in both half tiles; 40 bytes per slot). */
uint64_t gabsplat_blend_state_bytes(int32_t width, int32_t height, uint64_t capacity);

/* Gradient outputs (all required except d_mean2d / d_mean2d_abs, which may be NULL). */
typedef struct {
  float* d_means;      /* [N][3]     */
  float* d_scales;     /* [N][3]     */
  float* d_rotations;  /* [N][4]     */
  float* d_opacities;  /* [N]        */
  float* d_sh;         /* [N][16][3] */
  float* d_freqs;      /* [N][K][3]  */
  float* d_weights;    /* [N][K]     */
  float* d_mean2d;     /* [N][2] optional: dL/dmu2D in pixel units (densification statistic, :175) */
  float* d_mean2d_abs; /* [N][2] optional: sum over pixels of |per-pixel dL/dmu2D| (AbsGS variant, :224) */
} gabsplat_grads;

/* Bytes of device scratch gabsplat_render_backward needs for N primitives with K components.  The scratch must
 * be ALL ZERO when gabsplat_render_backward is called; the call returns it all zero again (it clears exactly the
 * records it wrote), so the caller zeroes it once, after allocating it. */
uint64_t gabsplat_grad_workspace_bytes(int32_t N, int32_t K);

/* S1.  Writes tiles_touched, radius and chunk_visible for all N primitives and every other array of
 * `out` for the visible ones (see gabsplat_projected). */
int32_t gabsplat_preprocess(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                            gabsplat_projected* out, void* stream);

/* S2.  Builds the list of (key,id) instances, one per (primitive, tile of its rectangle), ordered by key with
 * ties by primitive index -- the result of a stable LSD radix sort on one-byte digits of the keys emitted in
 * primitive-major order (the depth digits are sorted on the primitives before duplication, the tile digits on
 * the instances after it) -- and extracts tile ranges.
 * If D > capacity nothing is emitted, *num_instances still holds D, and (when num_instances_host is
 * given) GABSPLAT_CAPACITY is returned.  num_instances_host != NULL makes the call synchronise the
 * stream once to read D back; with NULL the call is fully asynchronous and the caller must have sized
 * capacity from an earlier run. */
int32_t gabsplat_bin_sort(gabsplat_ctx* ctx, int32_t N, const gabsplat_projected* proj, const gabsplat_camera* cam,
                          gabsplat_binning* bin, uint64_t* num_instances_host, void* stream);

/* S1 + S2 in one call: the same results as gabsplat_preprocess followed by gabsplat_bin_sort, with the fp64 value
 * track of the projection (needed only by the blend) running on the context's side stream beside the binning
 * (which needs only the indexing track).  All outputs are ready, in the order of `stream`, when later work
 * enqueued on `stream` runs. */
int32_t gabsplat_preprocess_bin_sort(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                     gabsplat_projected* proj, gabsplat_binning* bin, uint64_t* num_instances_host,
                                     void* stream);

/* S3.  One CTA per tile; Eq.12-13 with the alpha rules of DESIGN.md (alpha = min(0.99, o G M),
 * skip alpha < 1/255, stop before T(1-alpha) < 1e-4). */
int32_t gabsplat_render_forward(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                const gabsplat_projected* proj, const gabsplat_binning* bin, gabsplat_fwd_out* out,
                                void* stream);

/* S4a + S4b.  dL_dimage is [3][H][W] on the device.  `bin` must be exactly what gabsplat_bin_sort returned for this
 * view, workspace included (the projection backward walks the list of visible primitives it holds); `fwd` must
 * carry the blend state. */
int32_t gabsplat_render_backward(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                                 const gabsplat_projected* proj, const gabsplat_binning* bin,
                                 const gabsplat_fwd_out* fwd, const float* dL_dimage, gabsplat_grads* grads,
                                 void* grad_workspace, uint64_t grad_workspace_bytes, void* stream);

/* Auxiliary renders (the frequency-map diagnostic of PAPER.md:764): the forward blend of S3 -- same
 * lists, same alpha rules -- with the colour of primitive i replaced by (sum_k omega_k |f2D_k| in cycles per pixel,
 * camera depth t_z, 1) over a zero background.  aux_image: [3][H][W] device = (blended frequency map, blended
 * depth, accumulated alpha = 1 - final T).  workspace: device scratch of >= gabsplat_aux_workspace_bytes bytes. */
uint64_t gabsplat_aux_workspace_bytes(int32_t N, int32_t width, int32_t height);
int32_t gabsplat_render_aux(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                            const gabsplat_projected* proj, const gabsplat_binning* bin, float* aux_image,
                            void* workspace, uint64_t workspace_bytes, void* stream);

/* The training loss of PAPER.md:171 Eq.14 on the device:
 *     L = (1 - lambda) mean|image - target| + lambda (1 - mean SSIM(image, target)),
 * SSIM per channel with the 11x11 Gaussian window (sigma 1.5, normalised, zero padding) and C1 = 0.01^2, C2 = 0.03^2
 * of the 3DGS loss the paper adopts.  image, target: [3][H][W] device.  loss_out: device [3] = (L, mean L1, mean SSIM).
 * dL_dimage (may be NULL: forward only): [3][H][W] device, fully overwritten -- the dL_dimage argument of
 * gabsplat_render_backward.  Deterministic (fixed-order reductions).  lambda in [0,1]. */
uint64_t gabsplat_loss_workspace_bytes(int32_t width, int32_t height);
int32_t gabsplat_loss(gabsplat_ctx* ctx, int32_t width, int32_t height, const float* image, const float* target, float lambda,
                      float* loss_out, float* dL_dimage, void* workspace, uint64_t workspace_bytes, void* stream);

/* gabsplat_loss_static -- the loss above for callers that cannot allocate device memory.
 *
 * gabsplat_loss wants a workspace, and somebody has to cudaMalloc it.  Not every caller can: code that runs as a
 * plugin inside another engine and is given only its input and output buffers; a real-time loop whose rules forbid
 * allocator calls once it is running (cudaMalloc serialises the whole process and may stall the GPU); a process that
 * shares a nearly full GPU and cannot count on a free block being there.  This entry point needs no workspace, no
 * context and no gabsplat_create: its scratch (the nine derivative maps and the per-block partial sums of Eq.14 :171)
 * is a fixed array compiled into the library.  It never calls cudaMalloc, cudaFree or any routine that allocates.
 *
 * Same arithmetic, same kernels, same results bit for bit as gabsplat_loss; same arguments minus ctx and workspace.
 * image, target, loss_out [3], dL_dimage (may be NULL) are DEVICE pointers owned by the caller, on the device that is
 * CURRENT on the calling thread, which must also be the device of `stream`.
 *
 * Limit: width * height <= gabsplat_loss_static_max_pixels() = 262 144 (512 x 512) and each side <= 2048.  A larger
 *   image returns GABSPLAT_CAPACITY and launches nothing; use gabsplat_loss for it.
 * Cost: the array is 9 MiB and is resident on EVERY GPU on which this library's module is loaded, from then until
 *   the process exits, whether or not this function is ever called.
 * First call on each device: looks up the array's address on that device (cudaGetSymbolAddress; host-side, cached
 *   afterwards).  Make that first call before starting any stream capture on the device.
 * Sharing: all calls on one GPU use the same array.  It keeps whatever the previous call left; that is harmless here
 *   because each call writes every scratch value before reading it, so nothing has to be cleared.  But two calls whose
 *   kernels can overlap on the GPU -- different streams without an ordering between them, or two host threads -- race
 *   on it and both results are garbage.  Order such calls yourself (one stream, or events).
 * Errors: GABSPLAT_INVALID_ARG / GABSPLAT_CAPACITY / GABSPLAT_CUDA; gabsplat_loss_static_last_error() returns the
 *   text of the calling thread's last non-OK status (never NULL).  Asynchronous like gabsplat_loss. */
uint64_t gabsplat_loss_static_max_pixels(void);
const char* gabsplat_loss_static_last_error(void);
int32_t gabsplat_loss_static(int32_t width, int32_t height, const float* image, const float* target, float lambda,
                             float* loss_out, float* dL_dimage, void* stream);

/* Convenience for callers with HOST buffers (bench.py's end-to-end leg): one forward (and, if
 * dL_dimage_host != NULL, backward) pass with host->device copies of the scene / image gradient and
 * device->host copies of the image / gradients inside the call; synchronises.  All pointers in
 * `scene_host` and `grads_host` are HOST pointers here; grads_host may be NULL when dL_dimage_host is.
 * Device memory is taken from `device_arena` (device pointer, arena_bytes long; query the size with
 * gabsplat_host_arena_bytes; zero it once after allocating it -- it holds the gradient scratch, see
 * gabsplat_grad_workspace_bytes). */
uint64_t gabsplat_host_arena_bytes(int32_t N, int32_t K, int32_t width, int32_t height, uint64_t capacity);
int32_t gabsplat_render_host(gabsplat_ctx* ctx, const gabsplat_scene* scene_host, const gabsplat_camera* cam,
                             uint64_t capacity, float* image_host, const float* dL_dimage_host,
                             gabsplat_grads* grads_host, void* device_arena, uint64_t arena_bytes, void* stream);

/* ---- instrumentation (used by bench.py and the tests; none of it is needed to render) ----------------
 *
 * Per-stage device timing.  While enabled, every stage launched by the four calls above is bracketed by a
 * pair of CUDA events recorded on the stream of the call.  gabsplat_timing_read waits for the recorded
 * events, writes up to max_records (stage id, elapsed milliseconds) pairs in launch order, stores the
 * number of records that existed in *n_records, and clears the record list.  Host calls. */
#define GABSPLAT_STAGE_PREPROCESS 0      /* S1  projection kernel                                   */
#define GABSPLAT_STAGE_SCAN 1            /* S2a prefix sum of tiles_touched over the depth-ordered visible primitives */
#define GABSPLAT_STAGE_DUPLICATE 2       /* S2b chunk bounds + per-(chunk, tile) counts (<= 26 000 tiles); key emission (radix path) */
#define GABSPLAT_STAGE_SORT 3            /* S2c the tile digit: one counting placement pass; one-byte radix passes over the
                                            instances on the radix path                                          */
#define GABSPLAT_STAGE_RANGES 4          /* S2d tile ranges (prefix of the count table; from the sorted keys on the radix path) */
#define GABSPLAT_STAGE_BLEND_FORWARD 5   /* S3                                                      */
#define GABSPLAT_STAGE_BLEND_BACKWARD 6  /* S4a (incl. zeroing the 2D gradient records)             */
#define GABSPLAT_STAGE_PREPROCESS_BACKWARD 7 /* S4b (incl. zeroing the gradient outputs)             */
#define GABSPLAT_STAGE_DEPTH_SORT 8      /* S2c depth order of the visible primitives (bucketed; radix passes as fallback) */
#define GABSPLAT_STAGE_COUNT 9
int32_t gabsplat_timing_enable(gabsplat_ctx* ctx, int32_t on);
int32_t gabsplat_timing_read(gabsplat_ctx* ctx, int32_t* stage_ids_host, float* ms_host, int32_t max_records,
                             int32_t* n_records_host);

/* Number of CUDA kernels this library has launched in this process so far (host counter). */
uint64_t gabsplat_kernel_launches(void);

/* Per-pixel work counters of the forward blend, the numerators of the blend kernels' roofline
 * (DESIGN.md "Rooflines"): counters is a DEVICE array [H][W][4] of
 *   [0] pairs examined  -- list entries visited before the pixel stopped (the stopping entry included),
 *   [1] pairs that pass the envelope test o G >= 1/255 (the ones whose K cosines must be evaluated),
 *   [2] pairs blended,
 *   [3] envelope-passing pairs at list positions <= the last contributor (what the backward re-evaluates).
 * Same arguments as gabsplat_render_forward; runs a counting variant of the blend kernel. */
int32_t gabsplat_count_pairs(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                             const gabsplat_projected* proj, const gabsplat_binning* bin, uint32_t* counters,
                             void* stream);

/* The forward blend's decisions at n selected pixels (instrumentation of the parity tests; reading C18: at a
 * pixel where a skip / stop / clamp decision sits within fp32 error of its threshold both outcomes are correct, and
 * the tests hand the CUDA path's decisions at exactly those pixels to the oracle).  One thread per pixel walks the
 * pixel's tile list with the operation sequence of gabsplat_render_forward (Eq.12-13 :158-162; bit-identical alpha).
 *   pixels   device [n][2] int32 (x, y); a pixel outside the image is not traced: its colour_T is 0 and its info is
 *            (0, 0, 0, 1)
 *   offsets  device [n+1] uint32, ascending: pixel i may write entries[offsets[i] .. offsets[i+1]) (an inverted pair
 *            gives the pixel an empty slice)
 *   entries  device: for every entry blended at pixel i, in order: its 1-based position in the tile list, bit 31 set
 *            when min(0.99, .) was active (zero derivative in the backward); entries beyond the slice are dropped
 *   colour_T device [n][4] float: the pixel's (r, g, b) incl. background and final T -- equal bit for bit to
 *            gabsplat_fwd_out.image / final_T
 *   info     device [n][4] uint32: n_contrib, number of blended entries (may exceed the slice), 1-based position of
 *            the entry at which the pixel stopped (T (1 - alpha) < 1e-4; 0 = never), 1 if the pixel is outside the image else 0 */
int32_t gabsplat_trace_pixels(gabsplat_ctx* ctx, const gabsplat_scene* scene, const gabsplat_camera* cam,
                              const gabsplat_projected* proj, const gabsplat_binning* bin, int32_t n, const int32_t* pixels,
                              const uint32_t* offsets, uint32_t* entries, float* colour_T, uint32_t* info, void* stream);

/* cos and sin of n raw radian phases (device arrays) exactly as the blend kernels evaluate the phases of Eq.12
 * (:158): the MUFU path, no explicit range reduction.  For the committed measurement of its error bound
 * (DESIGN.md "Tolerances"). */
int32_t gabsplat_probe_sincos(gabsplat_ctx* ctx, int32_t n, const float* phase, float* cos_out, float* sin_out, void* stream);

/* The placement pass of gabsplat_bin_sort works on bands of tile rows; bands > 0 forces that many bands (so that a
 * test can run the multi-band code on a small image), 0 restores the automatic choice.  Results never depend on it. */
int32_t gabsplat_set_place_bands(gabsplat_ctx* ctx, int32_t bands);

/* The ALU rooflines of the blend kernels measured on this device: results_host[16] (HOST) =
 *   [0] FFMA lane-instructions/s   [1] packed FFMA2 lane-instructions/s   [2] MUFU.EX2 lane-ops/s
 *   [3] MUFU.COS lane-ops/s        [4] 4 FFMA : 1 MUFU mix, lane-instructions/s   [5] integer ALU-pipe lane-instr/s
 *   [6] SM clock (Hz) seen by the kernels   [7] number of SMs   [8..13] entries 0..5 per SM per clock.
 * Dependency-free chains, 64 warps per SM, best of 3 after a warm-up.  Synchronises; takes a few milliseconds. */
int32_t gabsplat_measure_peaks(gabsplat_ctx* ctx, float* results_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* GABSPLAT_H_ */
