/* farm.h -- C ABI of the B200-native FARM mapping hot path (libfarm_map.so).
 *
 * The library implements the data-parallel part of FARM's per-batch synchronous memory update
 *     M_t = f(M_{t-1}, o_t)                    ("Online construction", steps 1-5)
 * in the voxel-overlap formulation fixed by BASELINE.json `north_star`:
 *   (1) back-project masked RGB-D detections to world points        ("masked depth points")
 *   (2) quantise the points to voxel keys, one key set V_d per detection
 *   (3) count voxel overlap |V_d ∩ V_o| of every detection with every map object
 *   (4) cosine similarity of detection descriptors against all map descriptors
 *                                                   ("a single batched detection-by-entity similarity matrix")
 *   (5) score = w_geo*|V_d∩V_o|/min(|V_d|,|V_o|) + w_sem*cos, argmax, `> tau` else new object
 *                                                   (BASELINE.json rule), then merge voxels,
 *       AABBs, count-weighted descriptors and view evidence into the map.
 * The exact rules (R1..R26) are listed in DESIGN.md section 3.  Every step runs in hand-written sm_100a
 * CUDA kernels; there is no CPU fallback -- without a CUDA device every call below except the option
 * setters fails with FARM_ERR_CUDA.
 *
 * Conventions
 *   - "DEVICE pointer": caller-owned CUDA device memory, must stay valid until the map's stream has
 *     executed the call.  "HOST pointer": ordinary host memory, consumed/filled before the call returns.
 *   - integrate calls are asynchronous on the map's stream and never synchronise the device.  Only
 *     host-visible arguments are validated at call time.  Data-dependent failures (hash table full,
 *     object capacity, per-call scratch overflow) set a sticky device error word that the next
 *     farm_map_sync / farm_map_read / farm_map_last_assoc returns as FARM_ERR_CAPACITY; after that the
 *     map content is unspecified.
 *   - one host thread per map handle.
 *   - K: row-major 3x3, fx=K[0], fy=K[4], cx=K[2], cy=K[5], skew ignored.  T_world_cam: row-major 4x4,
 *     camera (x right, y down, z forward; depth = camera z, not ray length) -> world; top 3x4 is read.
 *   - instance_mask: 0 = background, k in 1..n_det = detection k-1 of that frame (descriptor row k-1),
 *     k > n_det = ignored (counted in stats).
 *   - voxel key: ix = floor(X * (1/voxel_size)) etc. in fp32, each in [-2^20, 2^20);
 *     key = (ix+2^20)<<42 | (iy+2^20)<<21 | (iz+2^20);  0xFFFFFFFFFFFFFFFF = no key.
 */
#ifndef FARM_H_
#define FARM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FARM_OK 0
#define FARM_ERR_INVALID_ARG (-1)
#define FARM_ERR_CUDA (-2)
#define FARM_ERR_CAPACITY (-3)
#define FARM_ERR_STATE (-4)
#define FARM_ERR_RANGE (-5) /* reserved: points outside the key range are dropped and counted (stats), never an error */

#define FARM_KEY_EMPTY 0xFFFFFFFFFFFFFFFFull

/* descriptor storage dtypes (one per map; detection rows and the map's similarity operands use it) */
#define FARM_DTYPE_F32 0
#define FARM_DTYPE_F16 1
#define FARM_DTYPE_BF16 2

/* integer options (farm_map_set_option_i); legal only before the first integrate / import / debug call */
#define FARM_OPT_DESC_DTYPE 1        /* FARM_DTYPE_*, default F32                                              */
#define FARM_OPT_MAX_OBJECTS 2       /* object capacity, default 65536                                         */
#define FARM_OPT_MAX_VOXELS 3        /* owned-voxel capacity, default 1<<22; sizes the block table unless MAX_BLOCKS is set */
#define FARM_OPT_IMG_W 4             /* image width  (required)                                                */
#define FARM_OPT_IMG_H 5             /* image height (required)                                                */
#define FARM_OPT_MAX_DET_PER_CALL 6  /* sum of n_det over the frames of one call, default 4096, max 65535        */
#define FARM_OPT_STREAM 7            /* cudaStream_t as integer, default 0 (legacy default stream)             */
#define FARM_OPT_MAX_PAIRS_PER_CALL 8 /* distinct (detection, voxel) pairs per call; default = pixels per call  */
#define FARM_OPT_MAX_FRAMES_PER_CALL 9 /* default 16, max 64                                                    */
#define FARM_OPT_SIM_PATH 10         /* 0 auto, 1 force CUDA-core fp32 FMA, 2 force tcgen05 tensor path, 3 tcgen05 with CTA pairs (cta_group::2) */
#define FARM_OPT_TIMING 11           /* 0 off; 1 CUDA events around the similarity kernel only; 2 around every kernel (this
                                        serialises the programmatically chained kernels).  May be changed at any time    */
#define FARM_OPT_OVERLAP 12          /* 1 (default): similarity on an internal side stream, concurrent with lift+probe;
                                        0 one stream; 2 / 3 experimental orders (see farm_api.cu).  Mode 1 needs the grids of
                                        one call to be co-resident (device-side waits between them, bounded: on expiry the
                                        sticky error reports FARM_ERR_STATE); with CUDA_LAUNCH_BLOCKING set the library
                                        uses mode 0                                                                    */
#define FARM_OPT_MAX_BLOCKS 13       /* capacity in 4x4x4 voxel blocks (256 B each); table = next pow2 >= 2x;
                                        default MAX_VOXELS / 4.  Exceeding it sets the sticky capacity error           */
#define FARM_OPT_GAUSSIAN 14         /* 1: also carry the paper's geometry: a 3-D Gaussian per
                                        detection and per object and the Hellinger distance of every match; default 0.
                                        The association rule is unchanged                                              */
#define FARM_OPT_COVISIBILITY 15     /* 1: maintain the N x ceil(N/64) covisibility bitset of PAPER.md:354 (step 7): all pairs
                                        of distinct objects that received a detection in one call; default 0            */
#define FARM_OPT_VIEWS 16            /* k in 0..8: keep up to k representative views per object (PAPER.md:63 item (iii),
                                        PAPER.md:353 step 6 "High-quality view selection"); default 0 = off               */
#define FARM_OPT_CORRESPONDENCE 17    /* 1: correspondence by union-find over the sparse match graph with entity-entity merges
                                        (steps 3-5; rules U1-U4 of DESIGN.md): every entity whose score
                                        exceeds tau is retained, a detection retaining two or more entities bridges them, the
                                        lowest id wins, same-call duplicate spawns are joined.  Needs tau >= 0.  Default 0 */
#define FARM_OPT_GEOMETRY 18          /* 0 (default): voxel overlap (BASELINE.json rule);  1: the paper's geometry -- similarity
                                        prefilter, then g = 1 - Hellinger distance between the detection's and the entity's
                                        Gaussian (rules H1-H3).  Needs FARM_OPT_GAUSSIAN = 1            */
#define FARM_OPT_EDGES 19             /* k in 0..16: maintain the weighted covisibility edge dictionary of PAPER.md:354 (rules
                                        W1-W4 of DESIGN.md; see farm_map_read_edges); default 0 = off.  Needs
                                        FARM_OPT_GAUSSIAN = 1; not available together with FARM_OPT_CORRESPONDENCE          */
#define FARM_OPT_INPUTS_READY 20      /* 1: the caller guarantees that the inputs of every integrate call are COMPLETE in device memory
                                        when the call is made -- not merely ordered before it on the map's stream -- and stay
                                        untouched until the call's work is done.  From the third call on, the similarity kernel of
                                        a call then no longer waits for the previous call's merge: it starts when the previous
                                        similarity kernel ends, computes the rows that merge does not write, and the rows it does
                                        write afterwards (split schedule).  Results are identical.  Takes
                                        effect with the 16-bit dtypes on the tensor-core path (FARM_OPT_SIM_PATH 0 or 2),
                                        FARM_OPT_OVERLAP = 1, and without FARM_OPT_CORRESPONDENCE / FARM_OPT_GEOMETRY; otherwise it
                                        is accepted and changes nothing.  farm_map_integrate_batch_host orders its own staging
                                        copies and may always be used with it.  Measured: single-frame
                                        calls 22-25 % shorter (33 / 49 / 45 us on configs 1-3); 16-frame batches of configs[4]
                                        no faster than the stream-ordered schedule (the board is power-managed there).  With FARM_OPT_TIMING = 1 only every
                                        eighth similarity kernel is bracketed by events and the sum is scaled.  Default 0      */
/* float options (farm_map_set_option_f) */
#define FARM_OPTF_Z_MIN 101          /* exclusive lower depth bound, default 0                                  */
#define FARM_OPTF_Z_MAX 102          /* inclusive upper depth bound, default +inf                               */
#define FARM_OPTF_VIEW_COS 103       /* a viewing direction is new if its cosine with every kept direction is below this;
                                        default cos(30 deg) = 0.8660254 (the paper's "fixed angular threshold" is unstated)  */
#define FARM_OPTF_PREFILTER_COS 105   /* H1: candidates are the entities with cosine > this; default 0.5 (the paper's
                                        "sufficiently similar" is unstated)                                              */
#define FARM_OPTF_HELLINGER_BUDGET 106 /* H2: candidates with H > this are dropped; default 1 (no gate; the paper's "fixed
                                        Hellinger budget" is unstated)                                                   */
#define FARM_OPTF_EDGE_DECAY 107      /* W4: weight discount per integrate call, in (0, 1]; default 0.9 (the paper's "temporal
                                        decay" is unstated)                                                              */
#define FARM_OPTF_EDGE_CUTOFF 108     /* W3: a neighbour farther than this multiple of the median kNN distance is dropped;
                                        >= 0, default 2 (the paper's "soft median cutoff" is unstated)                    */
#define FARM_OPTF_VIEW_CLOSER 104    /* or the view is kept if its distance is below this ratio x the closest kept view;
                                        default 0.8 (the paper's "sufficiently closer" is unstated)                        */

typedef struct farm_map farm_map; /* opaque; the library owns all map memory */

/* One map object as exported / imported.  (PAPER.md:63 entity attributes reduced to BASELINE.json's fields.) */
typedef struct {
  int32_t id;               /* dense 0..N-1, creation order                                                  */
  uint32_t n_voxels;        /* |V_o|, number of owned voxel keys                                             */
  uint32_t n_obs;           /* detections merged so far                                                      */
  float aabb_min[3];        /* AABB over all merged world points (fp32, exact min/max)                       */
  float aabb_max[3];
  int32_t best_frame;       /* best view: frame sequence number (0-based over all integrated frames)         */
  int32_t best_det;         /*            detection index inside that frame                                  */
  uint32_t best_pixels;     /*            its valid masked pixel count (the view quality measure)            */
  float best_cam_pos[3];    /*            camera position (translation of T_world_cam)                       */
  uint64_t n_points;        /* total valid masked pixels merged                                              */
} farm_object;

typedef struct {
  uint64_t valid_points;    /* valid masked pixels of the call (R4 and key in range)                         */
  uint64_t dropped_points;  /* valid pixels whose voxel index left [-2^20, 2^20)                             */
  uint64_t ignored_pixels;  /* pixels with label > n_det                                                     */
  uint64_t unique_voxels;   /* sum over detections of |V_d|                                                  */
  uint32_t matches, spawns, skipped, n_det;
} farm_frame_stats;

typedef struct {
  uint64_t frames, calls, valid_points, unique_voxels, matches, spawns;
} farm_totals; /* cumulative since create / import */

/* Create an empty map.  BASELINE.json: farm_map_create(voxel_size, D, w_geo, w_sem, tau).
 * voxel_size > 0 metres; 1 <= D <= 8192; w_geo >= 0, w_sem >= 0.  *out receives the handle.
 * Device memory is allocated at the first integrate / import, when the options are frozen. */
int farm_map_create(float voxel_size, int D, float w_geo, float w_sem, float tau, farm_map **out);
int farm_map_destroy(farm_map *m);

int farm_map_set_option_i(farm_map *m, int key, long long value);
int farm_map_set_option_f(farm_map *m, int key, float value);

/* One frame.  BASELINE.json: farm_map_integrate(depth, instance_mask, K, T_world_cam, det_descriptors, n_det).
 * depth [H,W] fp32 metres, instance_mask [H,W] u16, K [9], T_world_cam [16], det_descriptors [n_det, D] in
 * the map's storage dtype: all DEVICE pointers (det_descriptors may be NULL iff n_det == 0).
 * Equivalent to farm_map_integrate_batch with one frame. */
int farm_map_integrate(farm_map *m, const float *depth, const uint16_t *instance_mask, const float *K,
                       const float *T_world_cam, const void *det_descriptors, int n_det);

/* F frames scored against ONE snapshot of the map (the paper's "RGB-D batch").
 * depth [F,H,W], mask [F,H,W], K [F,9], T [F,16], desc [sum n_det, D]: DEVICE pointers.  n_det: HOST array [F].
 * Global detection index j = position in the concatenation of the frames' detection lists. */
int farm_map_integrate_batch(farm_map *m, int n_frames, const float *depth, const uint16_t *instance_mask,
                             const float *K, const float *T_world_cam, const void *det_descriptors,
                             const int *n_det);

/* Same call with HOST buffers (pinned memory recommended): the library copies the batch into one of its two
 * device staging sets with cudaMemcpyAsync on an internal copy stream, then runs the identical kernels on the
 * map's stream.  The call does not block: the copy of call t+1 overlaps the kernels of call t.  The host
 * buffers may be reused once the map's stream has passed the call (farm_map_sync / farm_map_last_assoc). */
int farm_map_integrate_batch_host(farm_map *m, int n_frames, const float *depth, const uint16_t *instance_mask,
                                  const float *K, const float *T_world_cam, const void *det_descriptors,
                                  const int *n_det);

/* Results of the LAST integrate call, HOST buffers of M = sum n_det entries (any may be NULL).
 * obj_id: object the detection was merged into (-1 = skipped, R8); is_new: 1 if that object was spawned by it;
 * best_score: R18.  Synchronises the stream; returns the sticky device error if set. */
int farm_map_last_assoc(farm_map *m, int32_t *obj_id, uint8_t *is_new, float *best_score, farm_frame_stats *stats);

/* Non-blocking form of farm_map_last_assoc: enqueues the device->host copies of the LAST call's results on the
 * map's stream and returns.  The HOST buffers (pinned memory, else the copy blocks) are valid after the next
 * farm_map_sync / farm_map_last_assoc / farm_map_read; the sticky device error is reported there. */
int farm_map_last_assoc_async(farm_map *m, int32_t *obj_id, uint8_t *is_new, float *best_score,
                              farm_frame_stats *stats);

/* Paper-faithful geometry (needs FARM_OPT_GAUSSIAN = 1; HOST buffers, any may be NULL; both calls synchronise).
 * "Each detection is lifted into a 3D Gaussian (mu_d, Sigma_d) over the masked depth points, with
 * Sigma_d stored in a 6-vector packed form" -- mu [.,3], cov [.,6] = population covariance packed xx xy xz yy yz zz.
 * the entity Gaussian is the sufficient-statistics merge M1 = w mu, M2 = w (Sigma + mu mu^T) over its
 * detections, w = number of points (weight [N], 0 for imported objects that have not been observed).
 * hellinger [M] = Hellinger distance in [0,1] between the detection's Gaussian and the Gaussian
 * of the object it was matched to, as that object was at entry of the call; -1 for spawned / skipped detections
 * and for objects without a Gaussian.  voxel_size^2 is added to both covariance diagonals (reading G3). */
int farm_map_last_gaussians(farm_map *m, float *mu, float *cov, float *hellinger);
int farm_map_read_gaussians(farm_map *m, double *weight, float *mu, float *cov);

/* Covisibility bitset (needs FARM_OPT_COVISIBILITY = 1; "A bitset adjacency (N x ceil(N/64) blocks) marks
 * all pairs of entities that were jointly visible in the current batch").  Two-call pattern: rows == NULL writes only
 * *words = ceil(N/64); else rows is a HOST buffer [N, *words] of uint64; bit b of row a is set iff objects a != b both
 * received a detection in one integrate call.  Bits are never cleared.  Synchronises. */
int farm_map_read_covisibility(farm_map *m, uint64_t *rows, int *words);

/* Identity history of the entity merges (needs FARM_OPT_CORRESPONDENCE; HOST buffers; synchronises).  alias [N]: the live
 * entity every id stands for now (itself while alive); an absorbed entity keeps its id as a dead record (no observations,
 * no voxels, zero descriptor).  farm_map_last_merges: the (loser, winner) pairs of the LAST integrate call, arbitrary
 * order; pass loser == NULL to get only *n. */
int farm_map_read_alias(farm_map *m, int32_t *alias);
int farm_map_last_merges(farm_map *m, int32_t *loser, int32_t *winner, int *n);

/* Retained views (needs FARM_OPT_VIEWS = k > 0; HOST buffers; synchronises).  PAPER.md:353: "A new viewpoint is retained
 * for an entity only if its viewing direction differs from all existing retained viewpoints by more than a fixed
 * angular threshold, or if it is sufficiently closer than the closest existing viewpoint."  Readings (V1-V2):
 * direction = unit vector from the camera position to the centre of the detection's point box, all decisions in fp32;
 * merged detections offer their view in index order; a full set replaces its farthest view (earliest on ties) if the
 * new view is closer than that one, else the new view is dropped.  views: [N, k] records, counts: [N] (<= k). */
typedef struct {
  int32_t frame, det;       /* frame sequence number and detection index inside the frame      */
  uint32_t n_px;            /* valid masked pixels of that detection                            */
  float cam[3], dir[3];     /* camera position; unit viewing direction camera -> object         */
  float dist;               /* distance camera -> centre of the detection's point box           */
} farm_view;
int farm_map_read_views(farm_map *m, farm_view *views, int32_t *counts);

/* Weighted covisibility edges (needs FARM_OPT_EDGES = k > 0; HOST buffers; synchronises).  PAPER.md:354: "a parallel
 * weighted edge dictionary accumulates their co-occurrence, restricted to spatially proximal pairs (a k-nearest-neighbor
 * graph in Gaussian Hellinger distance with a soft median cutoff) and discounted by a temporal decay".  Readings
 * (W1-W4): per call, S = the distinct entities that received a detection; for a in S, N_k(a) = its k nearest
 * members of S in Hellinger distance between the entity Gaussians after the call's merge (ordered through the
 * Bhattacharyya distance DB, of which H = sqrt(1 - exp(-DB)) is an increasing function that saturates at 1 in floating
 * point; fp32 value, ties -> lower id); b in N_k(a) is kept iff DB(a, b) <= cutoff x the lower median of a's kNN
 * distances; every unordered pair kept from either side gets w <- w * decay^(calls since its last update) + 1.
 * Writes the n edges (a < b, sorted by (a, b)) with w discounted to the last integrate call; *n_out = n even when
 * capacity < n (then only the first `capacity` are written and FARM_ERR_CAPACITY is returned).  a, b, w may be NULL. */
int farm_map_read_edges(farm_map *m, uint32_t *a, uint32_t *b, double *w, uint64_t capacity, uint64_t *n_out);

/* Step 4 alone, for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the dense cosine of M rows of A against N rows of B with the fused row maximum / argmax of R14-R16, R18
 * ("a single batched detection-by-entity similarity matrix") -- the arithmetic of the CUDA-core similarity
 * kernel, operands and results given by the caller, no map.
 *   A DEVICE [M, D], B DEVICE [N, D], row-major, both in `dtype` (FARM_DTYPE_*); rows need not be normalised
 *   max_cos DEVICE f32 [M]: max over B rows of clamp(cos, -1, 1); argmax DEVICE i32 [M]: its row, lowest index on ties;
 *   (0, -1) when N = 0; a zero-norm row has cosine 0 with everything.  Either output may be NULL.
 *   stream: cudaStream_t (as void*); the kernels are enqueued on it, the call does not synchronise.
 * The scratch of the kernels (inverse row norms, one packed word per row of A) is a file-scope device array of
 * FARM_NOALLOC_SCRATCH_BYTES that every GPU using the library holds until the process exits; the call allocates nothing
 * (no cudaMalloc / cudaFree / allocating library routine).  Limits: M <= FARM_NOALLOC_MAX_M, N <= FARM_NOALLOC_MAX_N,
 * 1 <= D <= 8192; beyond them FARM_ERR_INVALID_ARG and nothing is enqueued.  ALL calls of the process on one GPU share the
 * array, which keeps the last call's contents (each call clears what it needs): calls that overlap on the GPU -- different
 * streams without an ordering between them -- race; calls on one stream are safe. */
#define FARM_NOALLOC_MAX_M 4096
#define FARM_NOALLOC_MAX_N 65536
#define FARM_NOALLOC_SCRATCH_BYTES 311296 /* 4 * MAX_M + 4 * MAX_N + 8 * MAX_M */
int farm_cosine_rowmax_noalloc(const void *A, int M, const void *B, int N, int D, int dtype, float *max_cos, int32_t *argmax,
                               void *stream);

/* Retrieval-side scoring over the finished memory (a second workload beside the mapper, rules Q1-Q5 of
 * DESIGN.md).  The three per-entity retrieval embedding matrices of PAPER.md:356 (caption text, image, image-VL), the
 * class ids and the query vectors are INPUTS; parser, encoders and the VLM reranker are out of scope.
 *   emb0/1/2  DEVICE [N, d0/d1/d2] in emb_dtype (FARM_DTYPE_*), N = current number of objects; cls DEVICE [N] or NULL
 *   q_target  HOST fp32 [2*d0 + d1 + d2]: the four query channels of the target -- description in space 0 (w = 1.0),
 *             raw utterance in space 0 (w = 0.5), prompt-ensemble mean in space 1 (w = 0.75), description in space 2
 *             (w = 1.0) ("each channel contributes w/(mu+rank) with offset mu = 5")
 *   n_pred predicates, pred_type HOST [n_pred] in FARM_PRED_*, each with its own landmark variable q_landmarks HOST
 *             [n_pred, 2*d0 + d1 + d2]; the landmark is bound to its top-scoring live entity
 *   Near / NextTo: exp(-d^2 / (2 sigma^2)) of the inter-centroid distance, sigma = 0.5 m / 1.0 m; Closest / Farthest:
 *             1 / (|rank - r*| + 1), rank by that distance among the live entities; centroid = Gaussian mean where the
 *             entity has one (FARM_OPT_GAUSSIAN), else the centre of its AABB
 *   s = s_sem * (0.5 + 0.5 * gbar), gbar = geometric mean of the predicate scores, s_sem * 0.3 on a class mismatch
 *             (target_class < 0: no class factor)
 * Outputs (HOST, any may be NULL): top_ids / top_scores [topk] by s (ties -> lower id, -1 past the live entities),
 * landmarks [n_pred], s_sem / gbar / s [N] (0 for entities without observations).  Synchronises. */
#define FARM_PRED_NEAR 0
#define FARM_PRED_NEXTTO 1
#define FARM_PRED_CLOSEST 2
#define FARM_PRED_FARTHEST 3
int farm_map_query(farm_map *m, const void *emb0, const void *emb1, const void *emb2, int d0, int d1, int d2, int emb_dtype,
                   const int32_t *cls, const float *q_target, int target_class, int n_pred, const int32_t *pred_type,
                   const float *q_landmarks, int topk, int32_t *top_ids, float *top_scores, int32_t *landmarks, float *s_sem,
                   float *gbar, float *s);

/* Export (HOST buffers) -- with farm_map_import the "scene state" persistence of PAPER.md:597 ("the memory is persisted
 * as a scene state") reduced to this path's fields.  Two-call pattern: with objects == NULL only *n_objects / *n_voxels are written.
 * descriptors: [N, D] fp32 masters (may be NULL).  voxel_keys / voxel_owner: [n_voxels] pairs in arbitrary
 * order (may be NULL).  Synchronises; returns the sticky device error if set. */
int farm_map_read(farm_map *m, farm_object *objects, int *n_objects, float *descriptors, uint64_t *voxel_keys,
                  uint32_t *voxel_owner, long long *n_voxels);

/* Bulk load into an EMPTY map (PAPER.md:597 scene-state resume; pre-populated maps).  HOST pointers.  Objects are
 * installed verbatim (ids must be 0..n-1 in order), descriptors are renormalised and shadowed (R26), every
 * voxel key must be unique, its owner < n_objects, and objects[i].n_voxels must equal the number of voxels listed
 * for i, else FARM_ERR_INVALID_ARG.  The frame counter is not part of the object records: a resumed map continues
 * its numbering with farm_map_set_frame_seq (else new frames start at 0 and tie with imported best views). */
int farm_map_import(farm_map *m, const farm_object *objects, int n_objects, const float *descriptors,
                    const uint64_t *voxel_keys, const uint32_t *voxel_owner, long long n_voxels);

/* Stream sync + sticky device error.  totals may be NULL. */
int farm_map_sync(farm_map *m, farm_totals *totals);

/* Per-stage device time accumulated since the last reset (needs FARM_OPT_TIMING >= 1; stages that are not
 * bracketed report 0) and kernel launches per stage.  ms / launches: HOST arrays [FARM_N_STAGES], may be
 * NULL.  Synchronises the stream. */
#define FARM_N_STAGES 6
#define FARM_STAGE_PREP 0        /* reset of per-call state + detection row norms            */
#define FARM_STAGE_LIFT 1        /* steps 1-2: back-project, voxelise, tile-level dedupe       */
#define FARM_STAGE_SIMILARITY 2  /* step 4: dense cosine with fused row max / argmax          */
#define FARM_STAGE_PROBE 3       /* step 3: voxel hash probe / insert, exact dedupe, overlap   */
#define FARM_STAGE_ASSOCIATE 4   /* step 5a: candidate scores, argmax, threshold, new ids     */
#define FARM_STAGE_MERGE 5       /* step 5b: voxel commit, descriptors, AABB, view evidence   */
int farm_map_stage_times(farm_map *m, float *ms, long long *launches, int reset);

/* Number of kernels this library has launched for the map so far (host counter). */
long long farm_map_kernel_launches(const farm_map *m);

/* Frame sequence number the next integrated frame will get (R23 best-view records carry it).  It starts at 0, advances
 * by the number of frames of every integrate call, can only be moved forward, and must stay <= INT32_MAX
 * (farm_object.best_frame is 32-bit): integrate returns FARM_ERR_STATE beyond that. */
int farm_map_get_frame_seq(farm_map *m, long long *frame_seq);
int farm_map_set_frame_seq(farm_map *m, long long frame_seq);

/* Thread-local description of the last error returned on this thread. */
const char *farm_last_error(void);

/* ---- parity / debug entry points (not on the production path) ---- */
/* Dense per-pixel world point (NaN where invalid) and voxel key (FARM_KEY_EMPTY where invalid or out of
 * range) of one frame.  All DEVICE pointers; xyz [H,W,3], keys [H,W].  n_det bounds the valid labels. */
int farm_debug_backproject(farm_map *m, const float *depth, const uint16_t *instance_mask, const float *K,
                           const float *T_world_cam, int n_det, float *xyz, uint64_t *keys);
/* For the LAST integrate call, HOST buffers; pass keys == NULL first to obtain offsets[M] = total.
 * offsets [M+1]; keys: the distinct voxel keys of each detection (arbitrary order inside a detection);
 * n_px [M]; box [M,6] = min xyz, max xyz of the detection's world points. */
int farm_debug_last_voxels(farm_map *m, long long *offsets, uint64_t *keys, uint32_t *n_px, float *box);
/* Sparse overlap histogram of the LAST call: offsets [M+1]; obj_id/count: (object, |V_d ∩ V_o|) with
 * count > 0, arbitrary order inside a detection.  Pass obj_id == NULL first to size. */
int farm_debug_last_overlaps(farm_map *m, long long *offsets, int32_t *obj_id, uint32_t *count);
/* Dense pass of the LAST call: per detection the maximum clamped cosine over all objects at entry and
 * its argmax (lowest id on ties; -1 when the map was empty).  HOST buffers [M]. */
int farm_debug_last_dense(farm_map *m, float *max_cos, int32_t *argmax);

#ifdef __cplusplus
}
#endif
#endif /* FARM_H_ */
