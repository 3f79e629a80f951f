/* ddf.h - C ABI of libddf: batched Directed Distance Field queries on one B200 (sm_100a).
 *
 * The operation: PAPER.md:58-62 (Sec. III-A, Eq. 1)  f(x, d) = (t, xi): for a ray with origin
 * x and unit direction d, t is the distance to the first surface along d and xi the predicted
 * probability that the ray hits at all; "Every query is one forward pass" (PAPER.md:80,
 * Sec. III-C).  The network family is the paper's "sinusoidal encoding with a wide MLP"
 * (Sec. IV-C) in the shapes BASELINE.json's configs fix:
 *
 *   gamma(v) = [v, sin(2^0 pi v), cos(2^0 pi v), ..., sin(2^(L-1) pi v), cos(2^(L-1) pi v)]
 *              (3 sines then 3 cosines per band), gamma = [gamma_Lo(origin) ; gamma_Ld(dir)]
 *   h_0 = gamma;  h_{l+1} = ReLU(W_l in_l + b_l),  in_l = [h_l ; gamma] if l == skip_layer else h_l
 *   z = W_out h_last + b_out;  t = softplus(z_0);  xi = sigmoid(z_1)          (n_out == 2)
 *   s = z_0                                                                   (n_out == 1, SDF)
 *
 * Arithmetic: weights and activations are bf16 operands (fp32 blobs are rounded to bf16 RNE at
 * create), products accumulate in fp32, bias + ReLU in fp32, gamma and every hidden activation
 * but the last are rounded to bf16 RNE; the head reads the last activation un-rounded.
 *
 * General rules
 *  - Every function returns 0 (DDF_OK) or a negative ddf_status; none throws, aborts or prints.
 *  - Pointers marked [device] are CUDA device pointers on the current device, caller-owned,
 *    contiguous, 4-byte aligned (16-byte alignment enables the vectorised path); [host] are
 *    host pointers.  Inputs and outputs must not alias.
 *  - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = default stream);
 *    no call synchronises the stream except ddf_create / ddf_destroy / ddf_trainer_create /
 *    ddf_trainer_export / the *_host variants, and - only for models served by the CUDA-core path -
 *    sdf_sphere_trace with early_exit and ddf_query_shadowed[_lights] (their grids are sized on the host),
 *    and ddf_query_ao_wavefront / ddf_query_shaded when spp does not divide 32 or only the CUDA-core path
 *    serves the model (one host read of the hit count; such a call cannot be captured).
 *    Results are valid once the stream reaches the point after the call.
 *  - n == 0 is DDF_OK and a no-op; n < 0 or a NULL pointer with n > 0 is DDF_E_INVALID_ARG.
 *  - Results are a pure function of (weights, ray): independent of n and of the ray's position
 *    in the batch, bit-reproducible run to run (training steps accumulate gradients with atomics
 *    and are reproducible to rounding only).  Directions must be unit length (not checked).
 *  - A model (and a trainer) lives on the CUDA device that was current when it was created: its weights, workspaces,
 *    tensor maps and kernel attributes exist there only.  Every call that takes one (ddf_destroy included; not
 *    ddf_set_path / ddf_get_info / ddf_trainer_steps, which touch host state only) must be made with that device
 *    current (cudaSetDevice) and with pointers and a stream of that device; with another device current it returns
 *    DDF_E_INVALID_ARG and launches nothing.  Multi-GPU use is one model per device (bench.py --gpus N: one process per
 *    GPU); ddf_get_info(model, 4) tells which device a model belongs to.
 *  - A model (and a trainer) owns device workspaces that its calls reuse: use one model from one
 *    stream / host thread at a time; different models are independent.  On a fused path ddf_query,
 *    ddf_query_logits and ddf_query_ao with an spp that divides 32 never allocate (their workspace is sized
 *    at ddf_create).  The calls that need a per-batch workspace - ddf_query_host, ddf_query_camera /
 *    ddf_query_ao_points on models that read rays from memory, ddf_query_ao with any other spp,
 *    sdf_sphere_trace, the wavefront calls, and every query of a model served by the CUDA-core path
 *    (also one forced there by ddf_set_path(model, 1): reserve after that call) - take it from ddf_reserve; without a reservation that covers the batch they size
 *    it themselves on first use (a synchronising cudaFree / cudaMalloc).  Once the workspace covers
 *    the batch a call issues only stream-ordered work, so it can be recorded by
 *    stream capture and replayed as a CUDA graph (ddf_trainer_step bakes that step's learning
 *    rate into the capture; ddf_trainer_loss_grads and every query are replayable as they are).
 *  - Every wait inside the tensor-core kernels is bounded: if a barrier is not reached within one minute of wall-clock
 *    time (only a bug in the library, or a context frozen from outside for that long, can cause it) the kernel traps
 *    instead of hanging the device.  A trap is a sticky CUDA error - the context is unusable afterwards and every call
 *    returns DDF_E_CUDA; the process has to reset the device or exit.
 *  - There is no CPU fallback: without a CUDA device of compute capability 10.x the calls
 *    return DDF_E_UNSUPPORTED / DDF_E_CUDA.
 */
#ifndef DDF_H
#define DDF_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum ddf_status {
  DDF_OK = 0,
  DDF_E_INVALID_ARG = -1,   /* NULL pointer, negative count, bad enum value                 */
  DDF_E_BAD_LAYOUT  = -2,   /* ddf_layout fields inconsistent or struct_size/version wrong  */
  DDF_E_UNSUPPORTED = -3,   /* shape or device not supported by any kernel                  */
  DDF_E_CUDA        = -4,   /* a CUDA call failed; see ddf_last_cuda_error()                */
  DDF_E_NOMEM       = -5,   /* host or device allocation failed                             */
  DDF_E_TOO_LARGE   = -6    /* batch larger than the fixed capacity of a *_static entry point */
} ddf_status;

#define DDF_LAYOUT_VERSION 1u

/* POD, caller-owned, copied by ddf_create. */
typedef struct ddf_layout {
  uint32_t struct_size;        /* sizeof(ddf_layout)                                        */
  uint32_t version;            /* DDF_LAYOUT_VERSION                                        */
  uint32_t input_kind;         /* 0 = ray (origin + direction), 1 = point (SDF networks)    */
  uint32_t n_freq_origin;      /* L_o >= 0 (identity always included)                       */
  uint32_t n_freq_dir;         /* L_d >= 0; ignored for input_kind 1                        */
  uint32_t n_hidden;           /* number of Linear+ReLU layers, >= 1                        */
  uint32_t width;              /* output width of every hidden layer                        */
  int32_t  skip_layer;         /* 0-based layer whose input is [h ; gamma]; -1 none; else 1..n_hidden-1 */
  uint32_t n_out;              /* 2 = (distance logit, visibility logit); 1 = linear value  */
  uint32_t weight_dtype;       /* 0 = fp32, 1 = bf16 (raw uint16)                           */
  uint32_t weights_on_device;  /* 0 = `weights` is a host pointer, 1 = device pointer       */
} ddf_layout;

/* Weight blob: layers 0..n_hidden-1 then the head; each layer is W[out][in] row-major followed
 * by b[out], all in `weight_dtype`.  in(layer 0) = E = (3+6 L_o) + (3+6 L_d) (ray) or 3+6 L_o
 * (point); in(skip layer) = width + E ordered [h ; gamma]; head rows are (distance, visibility). */

typedef struct ddf_model ddf_model;            /* opaque; owns a pre-tiled device copy of the weights */

typedef struct ddf_camera { float pos[3]; float look_at[3]; float fov_deg; } ddf_camera;
typedef struct ddf_scene  { float sphere_c[3]; float sphere_r; float box_min[3]; float box_max[3]; } ddf_scene;

/* ---------------------------------------------------------------- model life cycle
 * ddf_create copies `weights` (host or device per layout->weights_on_device), rounds fp32 to
 * bf16, builds the tiled device copy and the per-model workspace; the caller may free `weights`
 * on return.  Synchronises the device.  *out is NULL on failure. */
int  ddf_create(const void* weights, const ddf_layout* layout, ddf_model** out);
int  ddf_destroy(ddf_model* model);                       /* NULL is DDF_OK */
const char* ddf_status_string(int status);
int  ddf_last_cuda_error(void);                           /* cudaError_t of the last DDF_E_CUDA on this thread */
/* Which kernel serves a layout: width a multiple of 256 (up to 2048): the persistent tcgen05 kernel;
 * width 64 or 128 with a weight set that fits in shared memory: the shared-memory-resident tcgen05
 * kernel; any other width up to 2048 is zero-padded at create to the next such width (padded units
 * have zero weights and bias, so every result is unchanged); everything else: the CUDA-core path. */
/* kernel selection: 0 = automatic (tcgen05 path when the layout allows, else the SIMT path),
 * 1 = force the SIMT path, 2 = force the tcgen05 path (DDF_E_UNSUPPORTED if it cannot run).
 * The persistent tcgen05 kernel answers a batch in one launch; a batch of at most 40 of its 256-ray
 * tiles (n <= 10,240) is instead answered as n_hidden + 2 launches chained by programmatic dependent
 * launch - encoding, one launch per hidden layer with the layer's output columns split over the
 * CTA pairs, heads - which keeps the whole chip busy on a small batch (2.5x faster at n <= 2,048).
 * Both return the same bits.  3 = tcgen05 path, always the single persistent launch; 4 = tcgen05
 * path, column-split whenever the batch fits the split scratch (n <= 18,944), else persistent.
 * 5 = tcgen05 path, activation-resident kernel for every batch size: the same forward pass with the layer hand-off kept
 * in shared and tensor memory (64 rays per CTA resident as the MMA's B operand; no activation is written to global
 * memory - BASELINE.json north_star (b) "Activations stay on-chip between layers"), for widths that are a multiple of
 * 256 up to 1280 with an encoding of at most 128 values; other layouts fall back to the persistent kernel.  Its results
 * agree with the persistent kernel's up to the order in which the same products are added (not bit for bit).
 * 3, 4 and 5 are DDF_E_UNSUPPORTED for models the persistent kernel does not serve. */
int  ddf_set_path(ddf_model* model, int path);
/* Sizes the per-batch workspaces ahead of time so that no later call with at most max_rays rays allocates
 * (SURVEY.md 8(b) "the library never allocates in ddf_query (workspace, if any, sized at create)").  `what` selects
 * which: DDF_RESERVE_HOST - staging of ddf_query_host (32 B per ray, plus its two copy streams and events);
 * DDF_RESERVE_RAYS - the ray buffer of ddf_query_camera / ddf_query_ao_points (24 B per ray; max_rays counts
 * width * height or n_pts * spp), and, when the reduce of ddf_query_ao cannot be fused into the query (spp does not
 * divide 32, or only the CUDA-core path serves the model), its per-ray results (8 B per ray); DDF_RESERVE_TRACE - sdf_sphere_trace (37 B per ray); DDF_RESERVE_WAVE - the
 * wavefront calls on max_rays primary rays, with room for spp ambient-occlusion rays per hit (40 B per primary ray,
 * or 32 + 24 spp if that is more; spp = 0: shadow calls only).  For a model only the CUDA-core path serves, the
 * activation workspace of its queries is sized too, whatever `what` is: that path answers a batch in passes of 16,384
 * rays, so the workspace holds min(max_rays, 16,384) rows (about 2 E_pad + 8 width bytes each) however large the batch.  Synchronises the device when
 * it (re)allocates; reservations only grow.  max_rays == 0 is a no-op; unknown bits in `what`: DDF_E_INVALID_ARG. */
#define DDF_RESERVE_HOST  1u
#define DDF_RESERVE_RAYS  2u
#define DDF_RESERVE_TRACE 4u
#define DDF_RESERVE_WAVE  8u
#define DDF_RESERVE_ALL   15u
int  ddf_reserve(ddf_model* model, uint32_t what, int64_t max_rays, int spp);
/* which = 0: 1 if the tcgen05 path serves this model, else 0; 1: kernels launched by the
 * last query call on this model; 2: E (encoded input width); 3: rays per tile of the path;
 * 4: ordinal of the CUDA device the model was created on. */
int64_t ddf_get_info(const ddf_model* model, int which);

/* ---------------------------------------------------------------- the paper's own field
 * PAPER.md:64 (Sec. III-A) / PAPER.md:84 (Sec. III-D): "a multiresolution hash grid that encodes
 * the point x, following [8] ... 16 levels, two features per level, a table of 2^19 entries per
 * level, base resolution 16, and growth 1.5, over a box that bounds the normalized object",
 * direction d with "four sinusoidal bands", "a two-layer MLP of width 64 reads the joined code
 * and outputs t and xi".  Definition used here (readings H1-H7):
 *   N_l = floor(base_resolution * growth^l); the level stores (N_l+1)^3 vertices when that fits
 *   T = 2^log2_table_size entries (index ix + (N_l+1)(iy + (N_l+1) iz)), else T hashed entries
 *   (index (ix ^ iy*2654435761 ^ iz*805459861) mod T, 32-bit products);
 *   x01 = clamp((x - box_min)/(box_max - box_min), 0, 1); pos = x01 * N_l; cell = min(floor(pos),
 *   N_l - 1); trilinear interpolation of the 8 cell corners, n_features values per vertex;
 *   MLP input = [level 0 features, level 1 features, ... ; gamma_{L_d}(d)], then Linear+ReLU
 *   layers and the same heads as above.
 * table: entries of all levels back to back, n_features values each, fp32 or fp16 (raw uint16).
 * mlp: layers 0..n_hidden-1 then the head, W[out][in] row-major then b[out], fp32 (rounded to
 * bf16 at create) or bf16.  Arithmetic: interpolation in fp32, bf16 MLP operands, fp32 accumulate.
 * This build serves n_features == 2, n_levels <= 16, L_d <= 4, width == 64, n_hidden 1..4.
 * The resulting model is used with ddf_query / ddf_query_host / ddf_query_logits / ddf_query_ao. */
typedef struct ddf_hashgrid_layout {
  uint32_t struct_size;        /* sizeof(ddf_hashgrid_layout) */
  uint32_t version;            /* DDF_LAYOUT_VERSION */
  uint32_t n_levels, n_features, log2_table_size, base_resolution;
  float    growth;
  float    box_min[3], box_max[3];
  uint32_t n_freq_dir, n_hidden, width, n_out;
  uint32_t table_dtype;        /* 0 = fp32, 2 = fp16 */
  uint32_t mlp_dtype;          /* 0 = fp32, 1 = bf16 */
  uint32_t weights_on_device;  /* both pointers: 0 = host, 1 = device */
} ddf_hashgrid_layout;
/* total number of table entries (vertices stored over all levels), or a negative ddf_status */
int64_t ddf_hashgrid_table_entries(const ddf_hashgrid_layout* layout);
int  ddf_create_hashgrid(const void* table, const void* mlp, const ddf_hashgrid_layout* layout,
                         ddf_model** out);

/* ---------------------------------------------------------------- the query
 * origins, dirs: [device] float[n][3].  out_dist, out_vis: [device] float[n]
 * (out_vis may be NULL; for n_out == 1 models out_dist receives the linear value z_0). */
int  ddf_query(ddf_model* model, const float* origins, const float* dirs, int64_t n,
               float* out_dist, float* out_vis, void* stream);
/* Same through [host] buffers (pinned for full speed): H2D copies, query, D2H copies, and a
 * stream synchronise, all inside the call.  The end-to-end entry point bench.py times.  Batches of
 * 2^18 rays or more are cut into 4 (8 from 2^21) tile-aligned chunks: uploads run ahead on a
 * stream owned by the model, chunk i is answered on `stream` once it has landed, and its results
 * return on a third stream while chunk i+1 is being answered; results are bit-identical to one
 * ddf_query over the whole batch. */
int  ddf_query_host(ddf_model* model, const float* origins, const float* dirs, int64_t n,
                    float* out_dist, float* out_vis, void* stream);
/* Primary rays ("To trace a primary ray we evaluate f at the camera and read t and
 * xi"): the width x height rays of ddf_gen_camera answered in one call, row-major, bit-identical
 * to ddf_gen_camera + ddf_query.  For a hash-grid model the rays are generated inside the query
 * kernel and the level features of the shared origin are computed once per CTA (8 bytes of HBM
 * traffic per ray instead of 32 and no per-ray gathers); other models use a workspace. */
int  ddf_query_camera(ddf_model* model, const ddf_camera* cam, int width, int height,
                      float* out_dist, float* out_vis, void* stream);
/* Debug/parity aid: raw logits z[n][n_out] instead of the head nonlinearities. */
int  ddf_query_logits(ddf_model* model, const float* origins, const float* dirs, int64_t n,
                      float* out_z, void* stream);

/* ---------------------------------------------------------------- ray generators
 * All pointers [device]; rays are float[.][3]. */
/* Host helper (A13): camera at `radius` on the sphere, position drawn from the counter
 * generator (seed, stream, indices 0,1), looking at the origin, 50 degree field of view. */
int  ddf_camera_from_seed(uint64_t seed, uint64_t stream, float radius, ddf_camera* out);
/* Pinhole primary rays, row-major, all origins = cam->pos ("evaluate f at the camera"). */
int  ddf_gen_camera(const ddf_camera* cam, int width, int height, float* o, float* d, void* stream);
/* n points uniform on the sphere |p| = radius with outward normals (counters 2i, 2i+1). */
int  ddf_gen_sphere_points(uint64_t seed, uint64_t rng_stream, int64_t n, float radius,
                           float* p, float* nrm, void* stream);
/* Shadow rays: o = p + eps n, d = normalise(light - o), tmax = |light - o| (tmax may be NULL). */
int  ddf_gen_shadow(const float* p, const float* nrm, int64_t n, const float light[3], float eps,
                    float* o, float* d, float* tmax, void* stream);
/* G-buffer: first hit of every camera ray against a sphere inside an axis-aligned room seen
 * from inside (inward wall normals).  t_hit may be NULL. */
int  ddf_gen_gbuffer(const ddf_camera* cam, const ddf_scene* scene, int width, int height,
                     float* p, float* nrm, float* t_hit, void* stream);
/* AO rays: spp cosine-weighted hemisphere directions per point, pixel-major; o = p + eps n. */
int  ddf_gen_ao(const float* p, const float* nrm, int64_t n_pts, int spp, uint64_t seed,
                uint64_t rng_stream, float eps, float* o, float* d, void* stream);
/* ao[i] = 1 - mean_s( vis > 0.5 and dist < ao_radius ) ("average the hit flag"). */
int  ddf_ao_reduce(const float* vis, const float* dist, int64_t n_pts, int spp, float ao_radius,
                   float* ao, void* stream);
/* Query + reduce in one call; the per-ray results never reach global memory when spp divides
 * 32 (a pixel's rays then sit in one warp of a tile); otherwise a workspace of 8 bytes per ray
 * owned by the model is used and ddf_ao_reduce runs as a second launch. */
int  ddf_query_ao(ddf_model* model, const float* o, const float* d, int64_t n_pts, int spp,
                  float ao_radius, float* ao, void* stream);
/* The same from surface points: the spp rays of point i are ddf_gen_ao's (same seed, rng_stream, eps: ray
 * k = i * spp + s), ao[i] as ddf_query_ao.  For a hash-grid field with spp dividing 32 the rays are generated
 * inside the query kernel and never exist in memory (12 B of point + 12 B of normal per spp rays instead of
 * 24 B per ray, and the spp rays of a point share one set of level look-ups); every other model generates
 * them into a workspace owned by `model` and calls ddf_query_ao.  Bit for bit ddf_gen_ao + ddf_query_ao.
 * p, nrm [n_pts][3] [device], ao [n_pts] [device]; n_pts * spp <= 2^31 - 1. */
int  ddf_query_ao_points(ddf_model* model, const float* p, const float* nrm, int64_t n_pts, int spp,
                         uint64_t seed, uint64_t rng_stream, float eps, float ao_radius, float* ao,
                         void* stream);
/* shadow[i] = 1 if vis > 0.5 and dist < tmax ("occluded within the distance to the light"). */
int  ddf_shadow_test(const float* vis, const float* dist, const float* tmax, int64_t n,
                     uint8_t* shadow, void* stream);

/* ---------------------------------------------------------------- wavefront secondary rays
 * PAPER.md:13 (the field answers "what a surface point sees in some direction")
 * ("The hit point is x + t d when xi is high"), PAPER.md:80 (shadow test: evaluate f from the
 * surface point toward the light; occluded within the distance to the light => shadow).
 * ddf_gen_shadow_from_hits turns the results of a primary query into a COMPACTED batch of shadow
 * rays: for every primary ray i with vis[i] > 0.5, in increasing i (stable),
 *   o2 = o_i + (dist_i - eps) d_i     (the hit point, stepped back by eps along the ray - the
 *                                      field returns no normal to offset along),
 *   d2 = normalise(light - o2),  tmax = |light - o2|,  index[k] = i.
 * All pointers [device]; o2, d2 [n][3], tmax [n], index [n] must hold n entries; *count (int64,
 * [device]) receives the number of secondary rays.  Uses a workspace owned by `model`. */
int  ddf_gen_shadow_from_hits(ddf_model* model, const float* o, const float* d, const float* dist,
                              const float* vis, int64_t n, const float light[3], float eps,
                              float* o2, float* d2, float* tmax, int32_t* index, int64_t* count,
                              void* stream);
/* ddf_gen_shadow_from_hits for callers that must not allocate device memory.  Same inputs, same outputs, same
 * bits as ddf_gen_shadow_from_hits (it launches the same three kernels), but it takes no model: the few numbers
 * the compaction keeps between its launches (one int32 per 256 primary rays) sit in a fixed 256 KB array inside
 * the library image instead of a cudaMalloc'ed workspace.  It is meant for hosts that gave all device memory to
 * their own pool when they started (a renderer with a fixed budget, a training framework's caching allocator), so
 * that a cudaMalloc made on the library's behalf would fail, and for frame loops that cannot take the device-wide
 * stall of a cudaMalloc / cudaFree.  What to know before using it:
 *  - n may be at most DDF_STATIC_MAX_RAYS (2^24 = 16,777,216); a larger n returns DDF_E_TOO_LARGE and nothing is
 *    launched.  Split a larger batch and add the offsets yourself, or use ddf_gen_shadow_from_hits.
 *  - The call itself never calls cudaMalloc, cudaFree or any library routine that allocates.  The array costs its
 *    256 KB on every GPU on which the process loads libddf.so, from load until exit, used or not.
 *  - The first call on each device looks the array's device address up (cudaGetSymbolAddress, with the caller's
 *    current device; a failure comes back as DDF_E_CUDA) and keeps it.  Make that first call during start-up, on
 *    the device you will use, before any stream capture is begun; later calls on that device only launch kernels.
 *  - There is one array per device and every call on that device uses it.  Two calls whose kernels can be on the
 *    GPU at the same time (different streams, or different host threads on different streams) overwrite each
 *    other's numbers and return garbage: issue them on one stream, or order the streams with events.  Calls that
 *    follow one another on a stream need no clearing in between - each call rewrites every entry it reads, so a
 *    larger earlier batch leaves nothing behind that a smaller later one could pick up.
 * All pointers [device] except light [host]; sizes and meaning as for ddf_gen_shadow_from_hits. */
#define DDF_STATIC_MAX_RAYS 16777216
int  ddf_gen_shadow_from_hits_static(const float* o, const float* d, const float* dist, const float* vis,
                                     int64_t n, const float light[3], float eps, float* o2, float* d2,
                                     float* tmax, int32_t* index, int64_t* count, void* stream);
/* The whole loop in one call: primary query -> hit compaction -> shadow rays -> second query on
 * the compacted batch (its size never leaves the device on the tcgen05 and hash-grid paths) ->
 * lit[i] = 1 if ray i hit (vis > 0.5) and its shadow ray is NOT occluded (not (vis2 > 0.5 and
 * dist2 < tmax)), else 0.  out_dist / out_vis [n] receive the primary results; out_count
 * (int64 [device], may be NULL) the number of shadow rays traced. */
int  ddf_query_shadowed(ddf_model* model, const float* o, const float* d, int64_t n,
                        const float light[3], float eps, float* out_dist, float* out_vis,
                        uint8_t* out_lit, int64_t* out_count, void* stream);
/* The same loop for several point lights (PAPER.md:80 evaluates f "toward the light"; a scene has
 * more than one): lights [host] float[n_lights][3], 1 <= n_lights <= 8.  The primary query and the
 * ranking of the hits run once; every light then gets its own shadow rays from the same hit points,
 * its own second query and bit j of out_lit_mask[i] (1 = ray i hit and light j is not occluded).
 * out_count receives the number of shadow rays traced, hits x n_lights.  With n_lights == 1 this is
 * ddf_query_shadowed bit for bit. */
int  ddf_query_shadowed_lights(ddf_model* model, const float* o, const float* d, int64_t n,
                               const float* lights, int n_lights, float eps, float* out_dist,
                               float* out_vis, uint8_t* out_lit_mask, int64_t* out_count, void* stream);

/* Ambient occlusion at the field's OWN hits (AO "along a set of hemisphere directions"
 * from a surface point "offset slightly along its normal"; the field as the renderer's
 * secondary-ray oracle, "no mesh in the pipeline").  The field returns no normal, so it is estimated
 * from the hit-point image of the primary batch (reading W5): the batch is a
 * width x height image, ray i = y * width + x; for every i with vis[i] > 0.5, P_i = o_i + dist_i d_i;
 * along x the difference goes to the neighbour that also hit (both hit: the one with the smaller
 * |dist_j - dist_i|, forward on ties), forward P_{i+1} - P_i, backward P_i - P_{i-1}; along y likewise
 * with +-width; n = normalise(du x dv) turned so that n . d_i <= 0; n = -d_i if an axis has no hit
 * neighbour or the product vanishes.
 * ddf_gen_ao_from_hits: stable compaction of the hits in increasing i: p_c, nrm_c [n][3], index [n]
 * (all must hold n = width * height entries), *count (int64 [device]) the number of hits; when o2 / d2
 * (both or neither; [n * spp][3]) are given they receive spp cosine-weighted rays per hit from
 * p_c + eps * nrm_c, exactly ddf_gen_ao(p_c, nrm_c, count, ...) with the count read on the device.
 * All pointers [device]; asynchronous on `stream`; uses a workspace owned by `model`.
 * width * height * spp must not exceed 2^31 - 1 (DDF_E_INVALID_ARG). */
int  ddf_gen_ao_from_hits(ddf_model* model, const float* o, const float* d, const float* dist,
                          const float* vis, int width, int height, int spp, uint64_t seed,
                          uint64_t rng_stream, float eps, float* p_c, float* nrm_c, int32_t* index,
                          float* o2, float* d2, int64_t* count, void* stream);
/* The whole loop in one call: primary query -> hit points and normals -> compacted AO rays -> second
 * query with the 16 -> 1 reduce fused (batch size read on the device on the tcgen05 and hash-grid paths
 * when spp divides 32; otherwise one host read of the count) -> out_ao[i] = 1 - mean over the spp rays of
 * (vis2 > 0.5 and dist2 < ao_radius) where ray i hit, 1 where it missed.  out_dist / out_vis [n] receive
 * the primary results, out_nrm ([n][3], may be NULL) the normal per pixel (0 where the ray missed),
 * out_count (int64 [device], may be NULL) the number of AO rays traced, hits x spp. */
int  ddf_query_ao_wavefront(ddf_model* model, const float* o, const float* d, int width, int height,
                            int spp, uint64_t seed, uint64_t rng_stream, float eps, float ao_radius,
                            float* out_dist, float* out_vis, float* out_nrm, float* out_ao,
                            int64_t* out_count, void* stream);
/* Shadows and ambient occlusion of one frame from ONE primary query (PAPER.md:155 / Table VI: the field as
 * the renderer's secondary-ray oracle for exactly these two effects): ddf_query, then the shadow loop of
 * ddf_query_shadowed_lights (n_lights = 0: skipped, out_lit_mask may be NULL) and the AO loop of
 * ddf_query_ao_wavefront (spp = 0: skipped, out_ao / out_nrm may be NULL) on the same primary results;
 * every output is bit for bit what those two calls return.  out_counts (int64[2] [device], may be NULL)
 * receives {shadow rays traced, AO rays traced}. */
int  ddf_query_shaded(ddf_model* model, const float* o, const float* d, int width, int height,
                      const float* lights, int n_lights, int spp, uint64_t seed, uint64_t rng_stream,
                      float eps, float ao_radius, float* out_dist, float* out_vis, uint8_t* out_lit_mask,
                      float* out_nrm, float* out_ao, int64_t* out_counts, void* stream);

/* ---------------------------------------------------------------- training the hash-grid field
 * PAPER.md:70 / 86: "an L1 term on distance, clamped at the box scale, plus a cross-entropy term
 * on the hit weighted at 0.3"; "Adam for 30,000 steps, a batch of 16,384 rays, and a learning rate
 * of 3e-3 decayed by cosine to five percent of its value"; 30 percent of each batch are ray-march
 * shifted points.  Readings T1-T6:
 *   per ray  l = hit * min(|softplus(z0) - t|, dist_clamp) + ce_weight * CE(sigmoid(z1), hit),
 *   loss = mean over the batch; Adam as published, bias-corrected, dense over every parameter;
 *   lr(s) = lr0 (f + (1-f)(1 + cos(pi min(s,S)/S))/2);  fp32 master parameters; the arithmetic of the
 *   hidden layers' products is ddf_train_params.arithmetic.
 * The trainer owns fp32 copies of the table and the MLP (+ Adam moments and a gradient buffer:
 * 4 x the field size) and, for DDF_TRAIN_BF16X3, a workspace of 256 bytes per ray of the largest
 * batch seen (it grows, synchronising the device, when a larger batch arrives).  This build trains
 * n_features == 2, width == 64, n_hidden <= 2.  A step is 4 kernels (gather, MLP, scatter, Adam),
 * the first three (and ddf_gen_train_batch) chained on `stream` by programmatic dependent launch;
 * like every call here it is ordered after the work already in `stream` and needs no
 * synchronisation. */
typedef struct ddf_train_params {
  uint32_t struct_size;        /* sizeof(ddf_train_params) */
  float lr0, lr_final_frac; int32_t total_steps;
  float beta1, beta2, adam_eps, dist_clamp, ce_weight;
  uint32_t arithmetic;         /* how the MLP products of the forward / backward pass are formed.
                                * DDF_TRAIN_BF16X3: on the tensor cores; each fp32 operand is split into two
                                * bf16 terms (16 mantissa bits together) and a product is three bf16 MMAs with
                                * fp32 accumulation, relative error ~2^-16 per term.  DDF_TRAIN_FP32: on the
                                * CUDA cores.  Parameters, moments, gradients, the loss, the head and the table
                                * interpolation are fp32 either way (the paper trains in half precision,
                                * PAPER.md:86; both choices here are tighter). */
} ddf_train_params;
#define DDF_TRAIN_BF16X3 0u
#define DDF_TRAIN_FP32 1u
typedef struct ddf_trainer ddf_trainer;
/* table, mlp: [host] fp32 blobs in the ddf_create_hashgrid order (layout dtypes must be 0). */
int  ddf_trainer_create(const float* table, const float* mlp, const ddf_hashgrid_layout* layout,
                        const ddf_train_params* params, ddf_trainer** out);
int  ddf_trainer_destroy(ddf_trainer* trainer);
/* One optimisation step on a batch: forward, loss, backward, Adam update (step counter + 1).
 * o, d [device] float[n][3]; t [device] float[n] target distance; hit [device] uint8[n];
 * loss [device] float (may be NULL) receives the batch loss BEFORE the update. */
int  ddf_trainer_step(ddf_trainer* trainer, const float* o, const float* d, const float* t,
                      const uint8_t* hit, int64_t n, float* loss, void* stream);
/* Parity aid: loss and gradients of the mean loss, no update.  grad_table [device] float
 * [entries * 2], grad_mlp [device] float [mlp parameters, blob order]; either may be NULL. */
int  ddf_trainer_loss_grads(ddf_trainer* trainer, const float* o, const float* d, const float* t,
                            const uint8_t* hit, int64_t n, float* loss, float* grad_table,
                            float* grad_mlp, void* stream);
/* Current parameters to [host] fp32 blobs (synchronises); feed them to ddf_create_hashgrid. */
int  ddf_trainer_export(ddf_trainer* trainer, float* table, float* mlp);
int64_t ddf_trainer_steps(const ddf_trainer* trainer);
/* Analytic supervision (stands in for the paper's mesh ray cast): distance to the
 * FIRST SURFACE along d of a solid sphere and a solid axis-aligned box, from any
 * origin (from inside an object that is where the ray leaves it).  t [n] (0 for a miss), hit [n]. */
int  ddf_scene_raycast(const ddf_scene* scene, const float* o, const float* d, int64_t n,
                       float* t, uint8_t* hit, void* stream);
/* One training batch (reading T6): origins uniform in [-sample_half, sample_half]^3 aimed at a
 * uniform point of [-1,1]^3; half of them re-anchored on the surface they hit (stepped back 1e-3,
 * new direction uniform on the sphere); targets from ddf_scene_raycast's rule; 30 % of the hit
 * rays moved forward by u * t with target t - u t (PAPER.md:70 self-consistency).  Ray k of step
 * s draws counters (s n + k) * 16 + j of (seed, rng_stream). */
int  ddf_gen_train_batch(const ddf_scene* scene, uint64_t seed, uint64_t rng_stream, int64_t step,
                         int64_t n, float sample_half, float* o, float* d, float* t, uint8_t* hit,
                         void* stream);

/* ---------------------------------------------------------------- sphere-tracing comparison
 * (BASELINE.json configs[4]).  `model` must have input_kind 1, n_out 1.
 * Traces s(p) = (|p| - base_radius) + alpha * MLP(p):
 *   t = 0; for step < max_steps: p = o + t d; s = s(p); if |s| < eps: hit, stop;
 *          t += s; if t > t_max or t < 0: miss, stop.   Unconverged: miss.
 * early_exit 0: every ray is evaluated max_steps times (finished rays keep their state);
 * early_exit 1: finished rays are compacted away between steps (stable: the live list keeps ray order).
 * omega in (1, 2): over-relaxed steps, t += omega * s; when the spheres at the previous and at the current point do
 * not touch (|s| + |s_prev| < t - t_prev) the step may have jumped a surface: the ray goes back to t_prev + s_prev
 * (that evaluation counted) and takes plain steps from then on.  omega <= 1 (0 included): the plain rule above,
 * bit for bit; omega >= 2, negative or NaN: DDF_E_INVALID_ARG.
 * out_t [n], out_hit [n] (0/1), out_steps [n] (SDF evaluations that counted for the ray).
 * trace_p / trace_s (may be NULL): [n][max_steps][3] / [n][max_steps] visited points and values
 * (unvisited entries are NaN).  total_evals [device] int64 (may be NULL): MLP evaluations made. */
typedef struct sdf_trace_params {
  int32_t max_steps; float eps; float t_max; float base_radius; float alpha; int32_t early_exit; float omega;
} sdf_trace_params;
int  sdf_sphere_trace(ddf_model* model, const float* o, const float* d, int64_t n,
                      const sdf_trace_params* params, float* out_t, uint8_t* out_hit,
                      int32_t* out_steps, float* trace_p, float* trace_s, int64_t* total_evals,
                      void* stream);

#ifdef __cplusplus
}
#endif
#endif
