// farm_oracle.cpp -- CPU ORACLE for the FARM mapping hot path.  TEST INFRASTRUCTURE, NOT PRODUCT.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, load
// or call this file.  It shares no source, header, table or helper with paper_2606_15476_b200/csrc and
// neither side includes the other.
//
// What it is: a plain, slow, single-threaded C++17 re-statement of the per-batch object-level memory
// update M_t = f(M_{t-1}, o_t) ("Per-frame synchronous update") in the
// voxel-overlap formulation that BASELINE.json `north_star` fixes, executed literally with std::map /
// std::set and double accumulators.  Rule numbers R1..R26 are those of SURVEY.md §8(c) / DESIGN.md §3;
// each function cites the rule and the passage it follows.  No blocking, fusion or reordering.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fno-fast-math -shared -fPIC   (see oracle/build.py)
// `-ffp-contract=off` matters: R5 requires every fp32 multiply and add to be rounded individually.
//
// Pins (tests/test_oracle_pins.py, `-m "not gpu"`): P1..P12 of DESIGN.md §4 -- closed-form
// back-projection of hand-placed points, floor-vs-truncate voxel cases, brute-force set intersection,
// library GEMM for the cosine matrix, closed-form running mean, conservation / containment /
// idempotence invariants.  No function here is "parity unpinned".
//
// Paper-faithful geometry carried beside the voxel rule (rules G1-G4 of DESIGN.md §11):
// per-detection 3D Gaussian over the masked depth points, entity Gaussian by sufficient-
// statistics merge, Hellinger distance between Gaussians.  Pins G-P1..G-P4 in
// tests/test_oracle_gaussian.py (covisibility bitset of PAPER.md:354, rule C1, pinned there as well by brute-force
// pair enumeration, symmetry and monotonicity): numpy mean/cov of the same points, union-of-halves, textbook closed forms
// of the Hellinger distance and numpy.linalg for the general formula.  The association decision is NOT changed.
//
// Round 2 additions (SURVEY.md §8(f) NEXT-1..4; readings in DESIGN.md §10-§13), every one off by default:
//   U1-U4  correspondence by union-find over the sparse match graph with entity-entity merges
//   H1-H3  the paper's geometry as the geometric term of the decision: similarity prefilter, then Hellinger distance
//          between the detection's and the entity's Gaussian within a budget
//   V1-V3  high-quality view selection: up to k views per entity, kept if the viewing direction is new or the view is
//          sufficiently closer (PAPER.md:63 item (iii))
//   Q1-Q5  retrieval-side scoring: reciprocal-rank fusion over four query channels, closed-form predicates over the
//          entity centroids, composite score, top-K
// Pins: tests/test_oracle_next.py (brute-force union-find, conservation laws, hand cases, closed forms, numpy ranks).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <map>
#include <set>
#include <vector>

namespace {

constexpr uint64_t KEY_EMPTY = 0xFFFFFFFFFFFFFFFFull;
constexpr int KEY_BIAS = 1 << 20;  // R6: 21 bits per axis, index range [-2^20, 2^20)

enum { DT_F32 = 0, DT_F16 = 1, DT_BF16 = 2 };

// ---- storage dtype <-> fp32 (R14/R25).  f16 uses the compiler's _Float16 (IEEE binary16, RNE);
// bf16 is the upper half of an fp32 with round-to-nearest-even.  Pinned against torch in the tests.
float bf16_to_f32(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  std::memcpy(&f, &u, 4);
  return f;
}
uint16_t f32_to_bf16(float f) {
  uint32_t u;
  std::memcpy(&u, &f, 4);
  if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x40);  // NaN stays NaN
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}
float f16_to_f32(uint16_t h) {
  _Float16 x;
  std::memcpy(&x, &h, 2);
  return (float)x;
}
uint16_t f32_to_f16(float f) {
  _Float16 x = (_Float16)f;
  uint16_t h;
  std::memcpy(&h, &x, 2);
  return h;
}
float load_storage(const void *p, int dtype, size_t i) {
  if (dtype == DT_F32) return ((const float *)p)[i];
  if (dtype == DT_F16) return f16_to_f32(((const uint16_t *)p)[i]);
  return bf16_to_f32(((const uint16_t *)p)[i]);
}
float round_to_storage(float f, int dtype) {  // value of the dtype shadow, as fp32
  if (dtype == DT_F32) return f;
  if (dtype == DT_F16) return f16_to_f32(f32_to_f16(f));
  return bf16_to_f32(f32_to_bf16(f));
}

struct BestView {  // R23
  int32_t frame = -1, det = -1;
  uint32_t n_px = 0;
  float cam[3] = {0, 0, 0};
};

struct View {  // V1: one retained viewpoint of an entity
  int32_t frame = -1, det = -1;
  uint32_t n_px = 0;
  float cam[3] = {0, 0, 0}, dir[3] = {0, 0, 0}, dist = 0;
};

struct Object {  // R1
  bool alive = true;     // U4: false once the entity has been absorbed by another one
  int32_t alias = -1;    // U4: the entity that absorbed this one (-1 while alive)
  std::vector<View> views;  // V2: at most views_k retained viewpoints, in the order they were retained
  uint32_t n_voxels = 0, n_obs = 0;
  uint64_t n_points = 0;
  float amin[3], amax[3];
  std::vector<float> f;       // fp32 master descriptor, unit norm
  std::vector<float> shadow;  // round_to_storage(f), carried as fp32
  BestView best;
  // G2: sufficient statistics of the entity Gaussian, M1 = w*mu, M2 = w*(Sigma + mu mu^T),
  // w = number of merged points; packed symmetric order xx, xy, xz, yy, yz, zz ("6-vector")
  double gW = 0.0, gM1[3] = {0, 0, 0}, gM2[6] = {0, 0, 0, 0, 0, 0};
};

struct Stats {  // per call
  uint64_t valid_points = 0, dropped_points = 0, ignored_pixels = 0, unique_voxels = 0;
  uint32_t matches = 0, spawns = 0, skipped = 0;
};

struct Map {
  float voxel_size, inv_vs, w_geo, w_sem, tau, z_min, z_max;
  int D, dtype, H, W;
  // options (oracle_set_option); all off by default
  int edges_k = 0;               // W: weighted covisibility edges over a kNN graph in Hellinger distance (0 = off)
  float edge_decay = 0.9f;       // W4: temporal decay per call
  float edge_cutoff = 2.0f;      // W3: soft median cutoff, as a multiple of the median kNN distance
  long long call_index = 0;      // integrate calls so far (W4: the clock of the decay)
  std::map<std::pair<int, int>, std::pair<double, long long>> edges;  // W4: {a < b} -> (weight, call of the last update)
  int opt_corr = 0;              // U: union-find correspondence with entity-entity merges
  int opt_geom = 0;              // H: 0 = voxel overlap (BASELINE.json rule), 1 = Hellinger distance between Gaussians
  float prefilter_cos = 0.5f;    // H1: candidates are the entities with cos > prefilter_cos
  float hell_budget = 1.0f;      // H2: candidates with H > hell_budget are dropped (1 = no gate: H <= 1 always)
  int views_k = 0;               // V: views kept per entity (0 = off)
  float view_cos = 0.8660254f;   // V2: a direction is new if its cosine with every kept direction is below this (30 degrees)
  float view_closer = 0.8f;      // V2: or the view is closer than view_closer x the closest kept view
  std::vector<int32_t> merged_from, merged_into;  // U4: (loser, winner) pairs of the last call
  std::map<uint64_t, uint32_t> owner;  // R11: one owner per key
  std::vector<Object> objs;
  int64_t frame_seq = 0;
  // results of the last call
  int M = 0;
  std::vector<int32_t> assoc;
  std::vector<uint8_t> is_new;
  std::vector<float> best_score, second_score;
  std::vector<float> tau_gap;                        // min over all scored pairs of |score - tau| (tests: margin filter)
  std::vector<float> dense_max, dense_second;        // R16: max_o clamp(cos(a_d, shadow_o)) over ALL entry objects; runner-up
  std::vector<int32_t> dense_arg;                    //      and its argmax (lowest id on ties), -1 if N = 0 / skipped
  std::vector<std::set<uint64_t>> V;                 // R7
  std::vector<uint32_t> n_px;                        // R7
  std::vector<float> box;                            // R7, [M,6]
  std::vector<std::map<uint32_t, uint32_t>> overlap; // R9
  std::vector<double> gS1, gS2;                      // G1: per detection sum p [M,3], sum p p^T [M,6]
  std::vector<float> hell;                           // G4: Hellinger distance to the matched entity, -1 if none
  // C1 ("A bitset adjacency (N x ceil(N/64) blocks) marks all pairs of entities that were jointly
  // visible in the current batch"): row a, bit b set iff a != b and both received a detection in one call.
  // Rows grow with N; bits are never cleared.
  std::vector<std::vector<uint64_t>> covis;
  Stats stats;
};

// G1/G2: mean and population covariance from (w, M1, M2); packed order xx, xy, xz, yy, yz, zz
void gaussian_from_moments(double w, const double *M1, const double *M2, double mu[3], double cov[6]) {
  for (int a = 0; a < 3; ++a) mu[a] = M1[a] / w;
  static const int ia[6] = {0, 0, 0, 1, 1, 2}, ib[6] = {0, 1, 2, 1, 2, 2};
  for (int k = 0; k < 6; ++k) cov[k] = M2[k] / w - mu[ia[k]] * mu[ib[k]];
}

double det3(const double c[6]) {  // symmetric 3x3 from packed xx, xy, xz, yy, yz, zz
  return c[0] * (c[3] * c[5] - c[4] * c[4]) - c[1] * (c[1] * c[5] - c[4] * c[2]) + c[2] * (c[1] * c[4] - c[3] * c[2]);
}

// G3 ("the Hellinger distance between two Gaussians is unitless and bounded in [0,1]"):
//   H^2 = 1 - |S1|^(1/4) |S2|^(1/4) / |Sbar|^(1/2) * exp(-1/8 dmu^T Sbar^-1 dmu),  Sbar = (S1 + S2)/2,
// with S = Sigma + eps2 * I on both sides (reading G3: masked depth patches are near-planar, their sample
// covariance is near-singular; the paper does not say how it conditions it; eps = voxel_size is the only
// length scale of this formulation).
double hellinger(const double mu1[3], const double c1[6], const double mu2[3], const double c2[6], double eps2) {
  double s1[6], s2[6], sb[6];
  for (int k = 0; k < 6; ++k) {
    const double reg = (k == 0 || k == 3 || k == 5) ? eps2 : 0.0;
    s1[k] = c1[k] + reg;
    s2[k] = c2[k] + reg;
    sb[k] = 0.5 * (s1[k] + s2[k]);
  }
  const double d1 = det3(s1), d2 = det3(s2), db = det3(sb);
  // inverse of Sbar by the adjugate (symmetric)
  const double inv[6] = {(sb[3] * sb[5] - sb[4] * sb[4]) / db, (sb[2] * sb[4] - sb[1] * sb[5]) / db,
                         (sb[1] * sb[4] - sb[2] * sb[3]) / db, (sb[0] * sb[5] - sb[2] * sb[2]) / db,
                         (sb[1] * sb[2] - sb[0] * sb[4]) / db, (sb[0] * sb[3] - sb[1] * sb[1]) / db};
  const double d[3] = {mu1[0] - mu2[0], mu1[1] - mu2[1], mu1[2] - mu2[2]};
  const double q = d[0] * (inv[0] * d[0] + inv[1] * d[1] + inv[2] * d[2]) + d[1] * (inv[1] * d[0] + inv[3] * d[1] + inv[4] * d[2]) +
                   d[2] * (inv[2] * d[0] + inv[4] * d[1] + inv[5] * d[2]);
  const double bc = std::pow(d1, 0.25) * std::pow(d2, 0.25) / std::sqrt(db) * std::exp(-0.125 * q);
  const double h2 = 1.0 - bc;
  return h2 > 0.0 ? std::sqrt(h2) : 0.0;
}

// W2: Bhattacharyya distance DB = 1/8 dmu^T Sbar^-1 dmu + 1/2 ln(|Sbar| / sqrt(|S1| |S2|)) of the same regularised
// Gaussians.  The Hellinger distance is a strictly increasing function of it, H = sqrt(1 - exp(-DB)), so "nearest in
// Hellinger distance" and "nearest in DB" are the same order -- but H rounds to 1 for every pair more than a few object
// sizes apart, where DB still separates them.
double bhattacharyya(const double mu1[3], const double c1[6], const double mu2[3], const double c2[6], double eps2) {
  double s1[6], s2[6], sb[6];
  for (int k = 0; k < 6; ++k) {
    const double reg = (k == 0 || k == 3 || k == 5) ? eps2 : 0.0;
    s1[k] = c1[k] + reg;
    s2[k] = c2[k] + reg;
    sb[k] = 0.5 * (s1[k] + s2[k]);
  }
  const double d1 = det3(s1), d2 = det3(s2), db = det3(sb);
  const double inv[6] = {(sb[3] * sb[5] - sb[4] * sb[4]) / db, (sb[2] * sb[4] - sb[1] * sb[5]) / db,
                         (sb[1] * sb[4] - sb[2] * sb[3]) / db, (sb[0] * sb[5] - sb[2] * sb[2]) / db,
                         (sb[1] * sb[2] - sb[0] * sb[4]) / db, (sb[0] * sb[3] - sb[1] * sb[1]) / db};
  const double d[3] = {mu1[0] - mu2[0], mu1[1] - mu2[1], mu1[2] - mu2[2]};
  const double q = d[0] * (inv[0] * d[0] + inv[1] * d[1] + inv[2] * d[2]) + d[1] * (inv[1] * d[0] + inv[3] * d[1] + inv[4] * d[2]) +
                   d[2] * (inv[2] * d[0] + inv[4] * d[1] + inv[5] * d[2]);
  return 0.125 * q + 0.5 * std::log(db / std::sqrt(d1 * d2));
}

// R5 (BASELINE.json "same fp32 operation order and FMA contraction disabled"):
// back-projection of pixel (u = column, v = row) at depth z.  Every * and + is an individually rounded
// fp32 operation in exactly this order; no +0.5 pixel-centre offset.
void backproject(const float *K, const float *T, int u, int v, float z, float out[3]) {
  const float fx = K[0], fy = K[4], cx = K[2], cy = K[5];
  const float inv_fx = 1.0f / fx, inv_fy = 1.0f / fy;
  const float xn = ((float)u - cx) * inv_fx;
  const float yn = ((float)v - cy) * inv_fy;
  const float xc = xn * z, yc = yn * z, zc = z;
  out[0] = ((T[0] * xc + T[1] * yc) + T[2] * zc) + T[3];
  out[1] = ((T[4] * xc + T[5] * yc) + T[6] * zc) + T[7];
  out[2] = ((T[8] * xc + T[9] * yc) + T[10] * zc) + T[11];
}

// R6: voxel index = floor(X * inv_vs) per axis (fp32 multiply, then floor), valid iff in [-2^20, 2^20);
// key packs the three biased 21-bit indices.  Returns false when the point is out of range (dropped).
bool voxel_key(const Map &m, const float p[3], uint64_t *key) {
  int64_t idx[3];
  for (int a = 0; a < 3; ++a) {
    const float q = std::floor(p[a] * m.inv_vs);
    if (!(q >= (float)-KEY_BIAS && q < (float)KEY_BIAS)) return false;  // also rejects NaN
    idx[a] = (int64_t)q;
  }
  *key = ((uint64_t)(idx[0] + KEY_BIAS) << 42) | ((uint64_t)(idx[1] + KEY_BIAS) << 21) | (uint64_t)(idx[2] + KEY_BIAS);
  return true;
}

// R4: valid pixel = finite depth in (z_min, z_max]
bool depth_valid(const Map &m, float z) { return std::isfinite(z) && z > m.z_min && z <= m.z_max; }

// R21 helper: normalise a double vector; returns false for the zero vector
bool normalise(std::vector<double> &v) {
  double s = 0;
  for (double x : v) s += x * x;
  if (!(s > 0)) return false;
  const double inv = 1.0 / std::sqrt(s);
  for (double &x : v) x *= inv;
  return true;
}

void refresh_shadow(const Map &m, Object &o) {
  o.shadow.resize(m.D);
  for (int i = 0; i < m.D; ++i) o.shadow[i] = round_to_storage(o.f[i], m.dtype);
}

// R15: cosine of two fp32 operand rows, double accumulation, explicit norms, clamp to [-1,1]
float cosine(const float *a, const float *b, int D) {
  double dot = 0, na = 0, nb = 0;
  for (int i = 0; i < D; ++i) {
    dot += (double)a[i] * (double)b[i];
    na += (double)a[i] * (double)a[i];
    nb += (double)b[i] * (double)b[i];
  }
  if (!(na > 0) || !(nb > 0)) return 0.0f;
  double c = dot / (std::sqrt(na) * std::sqrt(nb));
  if (c > 1.0) c = 1.0;
  if (c < -1.0) c = -1.0;
  return (float)c;
}

// U3: union-find with path compression; the root of a set is its smallest node index
int uf_find(std::vector<int> &parent, int x) {
  int r = x;
  while (parent[r] != r) r = parent[r];
  while (parent[x] != r) {
    const int nx = parent[x];
    parent[x] = r;
    x = nx;
  }
  return r;
}
void uf_union(std::vector<int> &parent, int a, int b) {
  a = uf_find(parent, a), b = uf_find(parent, b);
  if (a == b) return;
  if (a < b) parent[b] = a; else parent[a] = b;
}

// V1-V2 ("A new viewpoint is retained for an entity only if its viewing direction differs from all
// existing retained viewpoints by more than a fixed angular threshold, or if it is sufficiently closer than the
// closest existing viewpoint"; "up to k representative views").  All arithmetic in fp32, one rounded
// operation at a time, because it decides which views are kept (both implementations take the decision in fp32).
// Readings: the viewing direction is the unit vector from the camera position to the centre of the detection's point
// box; a full set replaces its farthest view (earliest on ties) if the new view is closer than that one, else the
// new view is dropped.
bool make_view(const float *box, const float *cam, int32_t frame, int32_t det, uint32_t n_px, View *out) {
  float d[3];
  for (int k = 0; k < 3; ++k) {
    const float c = 0.5f * (box[k] + box[3 + k]);
    d[k] = c - cam[k];
  }
  const float d2 = (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
  const float dist = std::sqrt(d2);
  if (!(dist > 0.0f)) return false;
  out->frame = frame, out->det = det, out->n_px = n_px, out->dist = dist;
  for (int k = 0; k < 3; ++k) out->cam[k] = cam[k], out->dir[k] = d[k] / dist;
  return true;
}
bool offer_view(const Map &m, Object &ob, const View &v) {
  bool fresh = true;
  float closest = std::numeric_limits<float>::infinity();
  for (const View &k : ob.views) {
    const float dot = (v.dir[0] * k.dir[0] + v.dir[1] * k.dir[1]) + v.dir[2] * k.dir[2];
    if (!(dot < m.view_cos)) fresh = false;
    closest = std::fmin(closest, k.dist);
  }
  const bool closer = !ob.views.empty() && v.dist < m.view_closer * closest;
  if (!ob.views.empty() && !fresh && !closer) return false;
  if ((int)ob.views.size() < m.views_k) {
    ob.views.push_back(v);
    return true;
  }
  size_t far = 0;
  for (size_t i = 1; i < ob.views.size(); ++i)
    if (ob.views[i].dist > ob.views[far].dist) far = i;
  if (!(v.dist < ob.views[far].dist)) return false;
  ob.views[far] = v;
  return true;
}

}  // namespace

extern "C" {

typedef struct {
  int32_t id;
  uint32_t n_voxels, n_obs;
  float aabb_min[3], aabb_max[3];
  int32_t best_frame, best_det;
  uint32_t best_pixels;
  float best_cam_pos[3];
  uint64_t n_points;
} oracle_object;

typedef struct {
  uint64_t valid_points, dropped_points, ignored_pixels, unique_voxels;
  uint32_t matches, spawns, skipped, n_det;
} oracle_stats;

void *oracle_create(float voxel_size, int D, float w_geo, float w_sem, float tau, int dtype, int H, int W,
                    float z_min, float z_max) {
  Map *m = new Map();
  m->voxel_size = voxel_size;
  m->inv_vs = 1.0f / voxel_size;  // R6: fp32 reciprocal computed once
  m->D = D;
  m->w_geo = w_geo;
  m->w_sem = w_sem;
  m->tau = tau;
  m->dtype = dtype;
  m->H = H;
  m->W = W;
  m->z_min = z_min;
  m->z_max = z_max;
  return m;
}
void oracle_destroy(void *h) { delete (Map *)h; }
void *oracle_clone(void *h) { return new Map(*(Map *)h); }  // deep copy (tests: margin filter, what-if runs)

// options: 1 correspondence (U), 2 geometry (H), 3 prefilter cosine, 4 Hellinger budget, 5 views k, 6 view cosine, 7 view closer
int oracle_set_option(void *h, int key, double v) {
  Map &m = *(Map *)h;
  switch (key) {
    case 1: if (v != 0 && !(m.tau >= 0.0f)) return -1; m.opt_corr = v != 0; return 0;
    case 2: m.opt_geom = (int)v; return 0;
    case 3: m.prefilter_cos = (float)v; return 0;
    case 4: m.hell_budget = (float)v; return 0;
    case 5: m.views_k = (int)v; return 0;
    case 6: m.view_cos = (float)v; return 0;
    case 7: m.view_closer = (float)v; return 0;
    case 8: m.edges_k = (int)v; return 0;
    case 9: m.edge_decay = (float)v; return 0;
    case 10: m.edge_cutoff = (float)v; return 0;
  }
  return -1;
}

// Debug: dense per-pixel world point (NaN where invalid) and key (KEY_EMPTY where invalid or dropped). R3-R6.
void oracle_backproject(void *h, const float *depth, const uint16_t *mask, const float *K, const float *T,
                        int n_det, float *xyz, uint64_t *keys) {
  Map &m = *(Map *)h;
  const float nanv = std::numeric_limits<float>::quiet_NaN();
  for (int v = 0; v < m.H; ++v)
    for (int u = 0; u < m.W; ++u) {
      const size_t i = (size_t)v * m.W + u;
      xyz[3 * i] = xyz[3 * i + 1] = xyz[3 * i + 2] = nanv;
      keys[i] = KEY_EMPTY;
      const uint16_t lab = mask[i];
      if (lab == 0 || lab > n_det || !depth_valid(m, depth[i])) continue;
      float p[3];
      backproject(K, T, u, v, depth[i], p);
      xyz[3 * i] = p[0];
      xyz[3 * i + 1] = p[1];
      xyz[3 * i + 2] = p[2];
      uint64_t key;
      if (voxel_key(m, p, &key)) keys[i] = key;
    }
}

// The update M_t = f(M_{t-1}, o_t) for one batch of F frames (batch snapshot semantics R2,
// PAPER.md:350 "a single batched detection-by-entity similarity matrix").
int oracle_integrate_batch(void *h, int F, const float *depth, const uint16_t *mask, const float *K,
                           const float *T, const void *desc, const int *n_det) {
  Map &m = *(Map *)h;
  const int D = m.D;
  const size_t HW = (size_t)m.H * m.W;
  int M = 0;
  std::vector<int> base(F + 1, 0);
  for (int f = 0; f < F; ++f) {
    base[f] = M;
    M += n_det[f];
  }
  base[F] = M;
  const int N = (int)m.objs.size();  // R2: snapshot size at entry
  m.M = M;
  m.assoc.assign(M, -1);
  m.is_new.assign(M, 0);
  m.best_score.assign(M, 0.0f);
  m.second_score.assign(M, -std::numeric_limits<float>::infinity());
  m.tau_gap.assign(M, std::numeric_limits<float>::infinity());
  m.dense_max.assign(M, 0.0f);
  m.dense_second.assign(M, -std::numeric_limits<float>::infinity());
  m.dense_arg.assign(M, -1);
  m.V.assign(M, {});
  m.n_px.assign(M, 0);
  m.box.assign((size_t)M * 6, 0.0f);
  m.overlap.assign(M, {});
  m.gS1.assign((size_t)M * 3, 0.0);
  m.gS2.assign((size_t)M * 6, 0.0);
  m.hell.assign(M, -1.0f);
  m.stats = Stats();
  std::vector<int> det_frame(M), det_local(M);

  // ---- steps 1-2 (R3-R8): back-project every valid masked pixel, quantise, build V_d, n_px_d, box_d
  for (int f = 0; f < F; ++f) {
    const float *Kf = K + 9 * f, *Tf = T + 16 * f;
    for (int d = 0; d < n_det[f]; ++d) {
      det_frame[base[f] + d] = f;
      det_local[base[f] + d] = d;
    }
    for (int v = 0; v < m.H; ++v)
      for (int u = 0; u < m.W; ++u) {
        const size_t i = f * HW + (size_t)v * m.W + u;
        const uint16_t lab = mask[i];
        if (lab == 0) continue;                                   // R3: background
        if (lab > n_det[f]) { m.stats.ignored_pixels++; continue; }  // R3: label without a descriptor row
        if (!depth_valid(m, depth[i])) continue;                  // R4
        float p[3];
        backproject(Kf, Tf, u, v, depth[i], p);                   // R5
        uint64_t key;
        if (!voxel_key(m, p, &key)) { m.stats.dropped_points++; continue; }  // R6: out of range -> dropped
        const int j = base[f] + lab - 1;                          // R2: global detection index
        float *b = &m.box[(size_t)j * 6];
        if (m.n_px[j] == 0) {
          for (int a = 0; a < 3; ++a) b[a] = b[3 + a] = p[a];
        } else {
          for (int a = 0; a < 3; ++a) {
            b[a] = std::fmin(b[a], p[a]);
            b[3 + a] = std::fmax(b[3 + a], p[a]);
          }
        }
        m.n_px[j]++;
        m.V[j].insert(key);                                       // R7
        {                                                         // G1: moments of the detection's points
          const double x = p[0], y = p[1], z = p[2];
          double *s1 = &m.gS1[(size_t)j * 3], *s2 = &m.gS2[(size_t)j * 6];
          s1[0] += x, s1[1] += y, s1[2] += z;
          s2[0] += x * x, s2[1] += x * y, s2[2] += x * z, s2[3] += y * y, s2[4] += y * z, s2[5] += z * z;
        }
        m.stats.valid_points++;
      }
  }
  for (int j = 0; j < M; ++j) m.stats.unique_voxels += m.V[j].size();

  // ---- step 3 (R9): overlap c[d][o] = |V_d ∩ V_o(entry)| through the key -> owner map
  for (int j = 0; j < M; ++j)
    for (uint64_t key : m.V[j]) {
      auto it = m.owner.find(key);
      if (it != m.owner.end()) m.overlap[j][it->second]++;
    }

  // ---- steps 4-5a (R10, R14-R20): dense cosine, score, argmax, threshold
  std::vector<float> a(D);
  std::vector<int> target(M, -1);
  std::vector<int> best_obj(M, -1);
  std::vector<std::vector<int>> retained(M);  // U1: entities with score > tau (the sparse match graph)
  const double eps2 = (double)m.voxel_size * (double)m.voxel_size;
  for (int j = 0; j < M; ++j) {
    if (m.n_px[j] == 0) {  // R8: empty detection is skipped
      m.stats.skipped++;
      continue;
    }
    for (int i = 0; i < D; ++i) a[i] = load_storage(desc, m.dtype, (size_t)j * D + i);  // R14
    float best = 0.0f, second = -std::numeric_limits<float>::infinity();
    int best_o = -1;
    double mu_d[3], c_d[6];
    if (m.opt_geom == 1) gaussian_from_moments((double)m.n_px[j], &m.gS1[(size_t)j * 3], &m.gS2[(size_t)j * 6], mu_d, c_d);
    for (int o = 0; o < N; ++o) {                                // R16: every pair
      const float c = cosine(a.data(), m.objs[o].shadow.data(), D);  // R15
      if (m.dense_arg[j] < 0 || c > m.dense_max[j]) {            // R16 dense row max, ties -> lowest id
        if (m.dense_arg[j] >= 0) m.dense_second[j] = std::fmax(m.dense_second[j], m.dense_max[j]);
        m.dense_max[j] = c;
        m.dense_arg[j] = o;
      } else {
        m.dense_second[j] = std::fmax(m.dense_second[j], c);
      }
      float g = 0.0f;
      if (m.opt_geom == 0) {                                     // R10
        auto it = m.overlap[j].find((uint32_t)o);
        const uint32_t cnt = it == m.overlap[j].end() ? 0u : it->second;
        const uint32_t mn = std::min<uint32_t>((uint32_t)m.V[j].size(), m.objs[o].n_voxels);
        if (mn > 0) g = (float)cnt / (float)mn;
      } else {
        // H1 ("restrict candidates to active entities whose per-detection feature is sufficiently
        // similar"): only entities with cos > prefilter_cos are candidates at all.
        if (!(c > m.prefilter_cos)) continue;
        // H2 ("then compute the Hellinger distance between the detection's 3D Gaussian and each candidate entity's
        // Gaussian, retaining every candidate entity within a fixed Hellinger budget"); H3: g = 1 - H.  An entity
        // without a Gaussian (imported, never observed) stays a candidate with g = 0.
        if (m.objs[o].gW > 0.0) {
          double mu_o[3], c_o[6];
          gaussian_from_moments(m.objs[o].gW, m.objs[o].gM1, m.objs[o].gM2, mu_o, c_o);
          const float hf = (float)hellinger(mu_d, c_d, mu_o, c_o, eps2);
          if (hf > m.hell_budget) continue;
          g = 1.0f - hf;
        }
      }
      const float score = m.w_geo * g + m.w_sem * c;             // R17 (fp32: two mul, one add)
      m.tau_gap[j] = std::fmin(m.tau_gap[j], std::fabs(score - m.tau));
      if (m.opt_corr && score > m.tau) retained[j].push_back(o); // U1
      if (best_o < 0 || score > best) {                          // R18: ties -> lowest id
        if (best_o >= 0) second = std::fmax(second, best);
        best = score;
        best_o = o;
      } else {
        second = std::fmax(second, score);
      }
    }
    m.best_score[j] = best_o >= 0 ? best : 0.0f;
    m.second_score[j] = second;
    best_obj[j] = (best_o >= 0 && best > m.tau) ? best_o : -1;   // R18: strict
    if (best_obj[j] >= 0 && m.objs[best_o].gW > 0.0) {  // G4: distance to the matched entity's Gaussian as it was at entry (R2)
      double mu_d2[3], c_d2[6], mu_o[3], c_o[6];
      gaussian_from_moments((double)m.n_px[j], &m.gS1[(size_t)j * 3], &m.gS2[(size_t)j * 6], mu_d2, c_d2);
      gaussian_from_moments(m.objs[best_o].gW, m.objs[best_o].gM1, m.objs[best_o].gM2, mu_o, c_o);
      m.hell[j] = (float)hellinger(mu_d2, c_d2, mu_o, c_o, eps2);
    }
  }

  int next_id = N;
  std::vector<int> loser_of;  // U4: entities absorbed in this call, ascending
  std::vector<int> parent;
  m.merged_from.clear();
  m.merged_into.clear();
  if (!m.opt_corr) {
    for (int j = 0; j < M; ++j) {
      if (m.n_px[j] == 0) continue;
      if (best_obj[j] >= 0) {
        target[j] = best_obj[j];
        m.assoc[j] = best_obj[j];
        m.stats.matches++;
      } else {  // R20: new ids in order of j
        target[j] = next_id++;
        m.assoc[j] = target[j];
        m.is_new[j] = 1;
        m.stats.spawns++;
      }
    }
  } else {
    // U2 (reading; repairs the duplicate spawns that R2 makes possible): a detection d that retained no entity is
    // linked to an earlier detection e of the same call when they see the same new space and look alike:
    //   c_dd(d, e) = number of keys of V_d that are unowned at entry and whose R12 claimant (the lowest-index detection
    //   of the call containing the key) is e;  g = c_dd / min(|V_d|, |V_e|);  score = w_geo*g + w_sem*cos(a_d, a_e) > tau.
    std::map<uint64_t, int> claim;
    for (int j = 0; j < M; ++j) {
      if (m.n_px[j] == 0) continue;
      for (uint64_t key : m.V[j])
        if (m.owner.find(key) == m.owner.end()) claim.emplace(key, j);
    }
    parent.resize(N + M);
    for (int i = 0; i < N + M; ++i) parent[i] = i;
    std::vector<float> b(D);
    for (int j = 0; j < M; ++j) {
      if (m.n_px[j] == 0) continue;
      for (int o : retained[j]) uf_union(parent, N + j, o);      // U1 edges; a detection retaining two entities bridges them
      if (!retained[j].empty()) continue;
      std::map<int, uint32_t> cdd;
      for (uint64_t key : m.V[j]) {
        auto it = claim.find(key);
        if (it != claim.end() && it->second != j) cdd[it->second]++;
      }
      for (int i = 0; i < D; ++i) a[i] = load_storage(desc, m.dtype, (size_t)j * D + i);
      for (auto &kv : cdd) {
        const int e = kv.first;
        const uint32_t mn = std::min<uint32_t>((uint32_t)m.V[j].size(), (uint32_t)m.V[e].size());
        const float g = mn ? (float)kv.second / (float)mn : 0.0f;
        for (int i = 0; i < D; ++i) b[i] = load_storage(desc, m.dtype, (size_t)e * D + i);
        const float score = m.w_geo * g + m.w_sem * cosine(a.data(), b.data(), D);
        m.tau_gap[j] = std::fmin(m.tau_gap[j], std::fabs(score - m.tau));
        if (score > m.tau) uf_union(parent, N + j, N + e);
      }
    }
    // U3 ("A union-find pass over the match graph with path compression resolves the case where multiple
    // detections claim the same entity, and the case where one detection bridges two previously separate entities"):
    // the root of a component is its smallest node; entities are numbered before detections, so a component that holds
    // an entity is won by its lowest-id entity (reading: the oldest identity survives), and a component of detections
    // only becomes ONE new entity, numbered in the order of its lowest detection index (R20).
    std::map<int, int> new_id_of_root;
    for (int j = 0; j < M; ++j) {
      if (m.n_px[j] == 0) continue;
      const int r = uf_find(parent, N + j);
      if (r < N) {
        target[j] = r;
        m.stats.matches++;
      } else {
        auto it = new_id_of_root.find(r);
        if (it == new_id_of_root.end()) {
          it = new_id_of_root.emplace(r, next_id++).first;
          m.is_new[j] = 1;  // the component's lowest detection creates the entity
          m.stats.spawns++;
        } else {
          m.stats.matches++;
        }
        target[j] = it->second;
      }
      m.assoc[j] = target[j];
    }
    for (int o = 0; o < N; ++o)
      if (uf_find(parent, o) != o) loser_of.push_back(o);
  }

  // ---- step 5b: merge, after all decisions (R12, R13, R21-R23)
  m.objs.resize(next_id);
  for (int o = N; o < next_id; ++o) {
    m.objs[o].f.assign(D, 0.0f);
    m.objs[o].shadow.assign(D, 0.0f);
    for (int k = 0; k < 3; ++k) {
      m.objs[o].amin[k] = std::numeric_limits<float>::infinity();
      m.objs[o].amax[k] = -std::numeric_limits<float>::infinity();
    }
  }
  // U4 ("Entity-level merges flagged by the correspondence pass are also executed here, absorbing the
  // loser's covisibility, captions, view records, and identity history into the winner"): before the call's detections
  // are fused, every loser L is absorbed by its winner W -- voxels re-owned, counts summed, boxes united, best view by
  // R23, Gaussian statistics summed, views offered under V2, covisibility row ORed in and column renamed.  The
  // count-weighted descriptors of the losers enter the winner's R21 fold below.  L stays as a dead id (alias -> W).
  std::vector<std::vector<int>> losers_of_winner(next_id);
  if (!loser_of.empty()) {
    std::map<uint32_t, uint32_t> win;
    for (int L : loser_of) win[(uint32_t)L] = (uint32_t)uf_find(parent, L);
    for (auto &kv : m.owner) {
      auto it = win.find(kv.second);
      if (it != win.end()) kv.second = it->second;
    }
    for (int L : loser_of) {
      const int Wn = uf_find(parent, L);
      Object &lo = m.objs[L], &wo = m.objs[Wn];
      losers_of_winner[Wn].push_back(L);
      m.merged_from.push_back(L);
      m.merged_into.push_back(Wn);
      wo.n_voxels += lo.n_voxels;
      wo.n_points += lo.n_points;
      for (int k = 0; k < 3; ++k) {
        wo.amin[k] = std::fmin(wo.amin[k], lo.amin[k]);
        wo.amax[k] = std::fmax(wo.amax[k], lo.amax[k]);
      }
      if (lo.best.n_px > wo.best.n_px ||
          (lo.best.n_px == wo.best.n_px && lo.best.n_px > 0 &&
           (lo.best.frame < wo.best.frame || (lo.best.frame == wo.best.frame && lo.best.det < wo.best.det))))
        wo.best = lo.best;
      wo.gW += lo.gW;
      for (int k = 0; k < 3; ++k) wo.gM1[k] += lo.gM1[k];
      for (int k = 0; k < 6; ++k) wo.gM2[k] += lo.gM2[k];
      for (const View &v : lo.views) offer_view(m, wo, v);
      // covisibility: row W |= row L; every bit L becomes bit W; no diagonal
      if ((size_t)L < m.covis.size() && (size_t)Wn < m.covis.size()) {
        for (size_t w = 0; w < m.covis[L].size(); ++w) m.covis[Wn][w] |= m.covis[L][w];
        for (size_t r = 0; r < m.covis.size(); ++r) {
          auto &row = m.covis[r];
          if (row.empty()) continue;
          if (row[(size_t)L >> 6] >> (L & 63) & 1ull) {
            row[(size_t)L >> 6] &= ~(1ull << (L & 63));
            if ((int)r != Wn) row[(size_t)Wn >> 6] |= 1ull << (Wn & 63);
          }
        }
        m.covis[Wn][(size_t)Wn >> 6] &= ~(1ull << (Wn & 63));
        std::fill(m.covis[L].begin(), m.covis[L].end(), 0ull);
      }
    }
  }
  // R12: keys unowned at entry go to the lowest-j detection of this call that contains them
  for (int j = 0; j < M; ++j) {
    if (target[j] < 0) continue;
    for (uint64_t key : m.V[j])
      if (m.owner.emplace(key, (uint32_t)target[j]).second) m.objs[target[j]].n_voxels++;
  }
  // R21: f_o <- normalise(n_obs * f_o + sum over matched detections of a_d/|a_d|); R22; R23
  std::vector<std::vector<int>> by_target(next_id);
  for (int j = 0; j < M; ++j)
    if (target[j] >= 0) by_target[target[j]].push_back(j);
  for (int o = 0; o < next_id; ++o) {
    if (by_target[o].empty()) continue;
    Object &ob = m.objs[o];
    std::vector<double> sum(D);
    for (int i = 0; i < D; ++i) sum[i] = (double)ob.n_obs * (double)ob.f[i];
    for (int L : losers_of_winner[o]) {  // U4: the losers' descriptors, weighted by their detection counts
      for (int i = 0; i < D; ++i) sum[i] += (double)m.objs[L].n_obs * (double)m.objs[L].f[i];
      ob.n_obs += m.objs[L].n_obs;
    }
    for (int j : by_target[o]) {
      std::vector<double> ad(D);
      for (int i = 0; i < D; ++i) ad[i] = (double)load_storage(desc, m.dtype, (size_t)j * D + i);
      if (normalise(ad))
        for (int i = 0; i < D; ++i) sum[i] += ad[i];
    }
    if (normalise(sum)) {
      for (int i = 0; i < D; ++i) ob.f[i] = (float)sum[i];
      refresh_shadow(m, ob);
    }
    for (int j : by_target[o]) {
      ob.n_obs += 1;
      ob.n_points += m.n_px[j];
      ob.gW += (double)m.n_px[j];                                  // G2: sufficient-statistics merge
      for (int k = 0; k < 3; ++k) ob.gM1[k] += m.gS1[(size_t)j * 3 + k];
      for (int k = 0; k < 6; ++k) ob.gM2[k] += m.gS2[(size_t)j * 6 + k];
      const float *b = &m.box[(size_t)j * 6];
      for (int k = 0; k < 3; ++k) {  // R22
        ob.amin[k] = std::fmin(ob.amin[k], b[k]);
        ob.amax[k] = std::fmax(ob.amax[k], b[3 + k]);
      }
      const float *Tf = T + 16 * det_frame[j];
      const float cam[3] = {Tf[3], Tf[7], Tf[11]};
      if (m.n_px[j] > ob.best.n_px) {  // R23: strict > keeps the earliest (frame_seq, det) on ties
        ob.best.n_px = m.n_px[j];
        ob.best.frame = (int32_t)(m.frame_seq + det_frame[j]);
        ob.best.det = det_local[j];
        ob.best.cam[0] = cam[0];
        ob.best.cam[1] = cam[1];
        ob.best.cam[2] = cam[2];
      }
      if (m.views_k > 0) {  // V: detections offer their view in index order
        View v;
        if (make_view(b, cam, (int32_t)(m.frame_seq + det_frame[j]), det_local[j], m.n_px[j], &v)) offer_view(m, ob, v);
      }
    }
  }
  for (int L : loser_of) {  // U4: the absorbed entities stay as dead ids
    Object &lo = m.objs[L];
    lo.alive = false;
    lo.alias = uf_find(parent, L);
    lo.n_voxels = lo.n_obs = 0;
    lo.n_points = 0;
    std::fill(lo.f.begin(), lo.f.end(), 0.0f);
    std::fill(lo.shadow.begin(), lo.shadow.end(), 0.0f);
    for (int k = 0; k < 3; ++k) {
      lo.amin[k] = std::numeric_limits<float>::infinity();
      lo.amax[k] = -std::numeric_limits<float>::infinity();
    }
    lo.best = BestView();
    lo.gW = 0.0;
    for (int k = 0; k < 3; ++k) lo.gM1[k] = 0.0;
    for (int k = 0; k < 6; ++k) lo.gM2[k] = 0.0;
    lo.views.clear();
  }
  // C1: every pair of distinct entities observed in this call (matched or spawned) becomes covisible
  {
    std::set<int> seen;
    for (int j = 0; j < M; ++j)
      if (target[j] >= 0) seen.insert(target[j]);
    const size_t words = ((size_t)next_id + 63) / 64;
    m.covis.resize(next_id);
    for (auto &row : m.covis) row.resize(words, 0);
    for (int a : seen)
      for (int b : seen)
        if (a != b) m.covis[a][(size_t)b >> 6] |= 1ull << (b & 63);
  }
  // W1-W4 ("a parallel weighted edge dictionary accumulates their co-occurrence, restricted to spatially
  // proximal pairs (a k-nearest-neighbor graph in Gaussian Hellinger distance with a soft median cutoff) and discounted
  // by a temporal decay").  Readings (none of the constants is printed):
  //   W1 S = the distinct entities that received a detection in this call (they all carry a Gaussian afterwards);
  //   W2 N_k(a) = the k entities of S \ {a} nearest to a in Hellinger distance between the entity Gaussians after this
  //      call's merge, ordered through the Bhattacharyya distance d = DB (fp32; H = sqrt(1 - exp(-DB)) is increasing
  //      in it and saturates at 1 in floating point where DB still separates pairs), ties -> lower id;
  //   W3 "soft median cutoff": b in N_k(a) is kept iff d(a, b) <= cutoff * (lower median of a's kNN distances);
  //   W4 every unordered pair {a, b} with b kept for a or a kept for b: w <- w * decay^(calls since its last update) + 1.
  m.call_index++;
  if (m.edges_k > 0) {
    std::set<int> seen;
    for (int j = 0; j < M; ++j)
      if (target[j] >= 0 && m.objs[target[j]].gW > 0.0) seen.insert(target[j]);
    std::vector<int> S(seen.begin(), seen.end());
    std::set<std::pair<int, int>> touched;
    for (int a : S) {
      double mu_a[3], c_a[6];
      gaussian_from_moments(m.objs[a].gW, m.objs[a].gM1, m.objs[a].gM2, mu_a, c_a);
      std::vector<std::pair<float, int>> dist;
      for (int b : S) {
        if (b == a) continue;
        double mu_b[3], c_b[6];
        gaussian_from_moments(m.objs[b].gW, m.objs[b].gM1, m.objs[b].gM2, mu_b, c_b);
        dist.push_back({(float)bhattacharyya(mu_a, c_a, mu_b, c_b, eps2), b});
      }
      std::sort(dist.begin(), dist.end());  // by distance, then by id
      const size_t kk = std::min<size_t>((size_t)m.edges_k, dist.size());
      if (kk == 0) continue;
      const float med = dist[(kk - 1) / 2].first;
      for (size_t i = 0; i < kk; ++i)
        if (dist[i].first <= m.edge_cutoff * med) touched.insert({std::min(a, dist[i].second), std::max(a, dist[i].second)});
    }
    for (auto &e : touched) {
      auto &rec = m.edges[e];
      rec.first = rec.first * std::pow((double)m.edge_decay, (double)(m.call_index - rec.second)) + 1.0;
      rec.second = m.call_index;
    }
  }
  m.frame_seq += F;
  return 0;
}

// ---- results of the last call
int oracle_last_M(void *h) { return ((Map *)h)->M; }
void oracle_last_assoc(void *h, int32_t *assoc, uint8_t *is_new, float *best, float *second, oracle_stats *st) {
  Map &m = *(Map *)h;
  for (int j = 0; j < m.M; ++j) {
    if (assoc) assoc[j] = m.assoc[j];
    if (is_new) is_new[j] = m.is_new[j];
    if (best) best[j] = m.best_score[j];
    if (second) second[j] = m.second_score[j];
  }
  if (st) {
    st->valid_points = m.stats.valid_points;
    st->dropped_points = m.stats.dropped_points;
    st->ignored_pixels = m.stats.ignored_pixels;
    st->unique_voxels = m.stats.unique_voxels;
    st->matches = m.stats.matches;
    st->spawns = m.stats.spawns;
    st->skipped = m.stats.skipped;
    st->n_det = (uint32_t)m.M;
  }
}
// R16 / R19: dense row maximum of the clamped cosine over all entry objects and its argmax (lowest id on ties);
// (0, -1) for skipped detections and for an empty map.
void oracle_last_dense(void *h, float *max_cos, int32_t *argmax, float *second) {
  Map &m = *(Map *)h;
  for (int j = 0; j < m.M; ++j) {
    if (max_cos) max_cos[j] = m.dense_max[j];
    if (argmax) argmax[j] = m.dense_arg[j];
    if (second) second[j] = m.dense_second[j];  // runner-up value (-inf when N < 2); used by tests for margins only
  }
}
// CSR of V_d (keys ascending inside a detection), n_px, box.  offsets has M+1 entries.
void oracle_last_voxels(void *h, int64_t *offsets, uint64_t *keys, uint32_t *n_px, float *box) {
  Map &m = *(Map *)h;
  int64_t pos = 0;
  for (int j = 0; j < m.M; ++j) {
    offsets[j] = pos;
    for (uint64_t k : m.V[j]) {
      if (keys) keys[pos] = k;
      pos++;
    }
    if (n_px) n_px[j] = m.n_px[j];
    if (box) std::memcpy(box + 6 * j, &m.box[6 * (size_t)j], 24);
  }
  offsets[m.M] = pos;
}
// CSR of the sparse overlap histogram (objects ascending inside a detection), zero counts omitted.
void oracle_last_overlaps(void *h, int64_t *offsets, int32_t *obj, uint32_t *count) {
  Map &m = *(Map *)h;
  int64_t pos = 0;
  for (int j = 0; j < m.M; ++j) {
    offsets[j] = pos;
    for (auto &kv : m.overlap[j]) {
      if (obj) obj[pos] = (int32_t)kv.first;
      if (count) count[pos] = kv.second;
      pos++;
    }
  }
  offsets[m.M] = pos;
}

// ---- map export
int oracle_n_objects(void *h) { return (int)((Map *)h)->objs.size(); }
long long oracle_n_voxels(void *h) { return (long long)((Map *)h)->owner.size(); }
void oracle_read(void *h, oracle_object *objs, float *desc, uint64_t *keys, uint32_t *owners) {
  Map &m = *(Map *)h;
  for (size_t o = 0; o < m.objs.size(); ++o) {
    const Object &ob = m.objs[o];
    if (objs) {
      oracle_object &q = objs[o];
      q.id = (int32_t)o;
      q.n_voxels = ob.n_voxels;
      q.n_obs = ob.n_obs;
      for (int k = 0; k < 3; ++k) {
        q.aabb_min[k] = ob.amin[k];
        q.aabb_max[k] = ob.amax[k];
        q.best_cam_pos[k] = ob.best.cam[k];
      }
      q.best_frame = ob.best.frame;
      q.best_det = ob.best.det;
      q.best_pixels = ob.best.n_px;
      q.n_points = ob.n_points;
    }
    if (desc) std::memcpy(desc + o * (size_t)m.D, ob.f.data(), sizeof(float) * m.D);
  }
  if (keys || owners) {
    size_t i = 0;
    for (auto &kv : m.owner) {  // ascending key order
      if (keys) keys[i] = kv.first;
      if (owners) owners[i] = kv.second;
      ++i;
    }
  }
}

// R26: bulk load into an empty map.  Ownership must be exclusive (duplicate key -> -1).  Descriptors are
// renormalised and shadowed as in R21.
int oracle_import(void *h, const oracle_object *objs, int n_objects, const float *desc, const uint64_t *keys,
                  const uint32_t *owners, long long n_voxels) {
  Map &m = *(Map *)h;
  if (!m.objs.empty() || !m.owner.empty()) return -4;
  m.objs.resize(n_objects);
  for (int o = 0; o < n_objects; ++o) {
    Object &ob = m.objs[o];
    const oracle_object &q = objs[o];
    ob.n_voxels = q.n_voxels;
    ob.n_obs = q.n_obs;
    ob.n_points = q.n_points;
    for (int k = 0; k < 3; ++k) {
      ob.amin[k] = q.aabb_min[k];
      ob.amax[k] = q.aabb_max[k];
      ob.best.cam[k] = q.best_cam_pos[k];
    }
    ob.best.frame = q.best_frame;
    ob.best.det = q.best_det;
    ob.best.n_px = q.best_pixels;
    std::vector<double> v(m.D);
    for (int i = 0; i < m.D; ++i) v[i] = (double)desc[(size_t)o * m.D + i];
    normalise(v);
    ob.f.resize(m.D);
    for (int i = 0; i < m.D; ++i) ob.f[i] = (float)v[i];
    refresh_shadow(m, ob);
  }
  for (long long i = 0; i < n_voxels; ++i) {
    if (owners[i] >= (uint32_t)n_objects) return -1;
    if (!m.owner.emplace(keys[i], owners[i]).second) return -1;
  }
  return 0;
}

// storage-dtype conversions exposed so the tests can pin them against torch
// G1: Gaussians of the last call's detections (mu [M,3], cov [M,6]; zeros for skipped ones) and G4 distances [M]
void oracle_last_gaussians(void *h, float *mu, float *cov, float *hell) {
  Map &m = *(Map *)h;
  for (int j = 0; j < m.M; ++j) {
    double mu_d[3] = {0, 0, 0}, c_d[6] = {0, 0, 0, 0, 0, 0};
    if (m.n_px[j]) gaussian_from_moments((double)m.n_px[j], &m.gS1[(size_t)j * 3], &m.gS2[(size_t)j * 6], mu_d, c_d);
    for (int k = 0; k < 3; ++k) mu[(size_t)j * 3 + k] = (float)mu_d[k];
    for (int k = 0; k < 6; ++k) cov[(size_t)j * 6 + k] = (float)c_d[k];
    hell[j] = m.hell[j];
  }
}
// G2: entity Gaussians (weight [N] = merged points, 0 = none; mu [N,3]; cov [N,6])
void oracle_read_gaussians(void *h, double *weight, float *mu, float *cov) {
  Map &m = *(Map *)h;
  for (size_t o = 0; o < m.objs.size(); ++o) {
    double mu_o[3] = {0, 0, 0}, c_o[6] = {0, 0, 0, 0, 0, 0};
    if (m.objs[o].gW > 0.0) gaussian_from_moments(m.objs[o].gW, m.objs[o].gM1, m.objs[o].gM2, mu_o, c_o);
    weight[o] = m.objs[o].gW;
    for (int k = 0; k < 3; ++k) mu[o * 3 + k] = (float)mu_o[k];
    for (int k = 0; k < 6; ++k) cov[o * 6 + k] = (float)c_o[k];
  }
}
// C1: rows [N, ceil(N/64)] of the covisibility bitset
int oracle_covis_words(void *h) { return (int)((((Map *)h)->objs.size() + 63) / 64); }
void oracle_read_covis(void *h, uint64_t *rows) {
  Map &m = *(Map *)h;
  const size_t N = m.objs.size(), words = (N + 63) / 64;
  for (size_t a = 0; a < N; ++a)
    for (size_t w = 0; w < words; ++w) rows[a * words + w] = a < m.covis.size() && w < m.covis[a].size() ? m.covis[a][w] : 0;
}
// tests only: per detection the smallest |score - tau| over every pair that was scored (entities, and detection pairs of U2)
void oracle_last_tau_gap(void *h, float *gap) {
  Map &m = *(Map *)h;
  for (int j = 0; j < m.M; ++j) gap[j] = m.tau_gap[j];
}
// W: the weighted edges, weights decayed to the current call count; a < b; ascending (a, b).  Returns their number.
long long oracle_read_edges(void *h, int32_t *a, int32_t *b, double *w) {
  Map &m = *(Map *)h;
  long long n = 0;
  for (auto &kv : m.edges) {
    if (a) a[n] = kv.first.first;
    if (b) b[n] = kv.first.second;
    if (w) w[n] = kv.second.first * std::pow((double)m.edge_decay, (double)(m.call_index - kv.second.second));
    ++n;
  }
  return n;
}
// U4: alias[o] = o for a live entity, else the live entity that (transitively) absorbed it
void oracle_read_alias(void *h, int32_t *alias) {
  Map &m = *(Map *)h;
  for (size_t o = 0; o < m.objs.size(); ++o) {
    size_t r = o;
    while (!m.objs[r].alive) r = (size_t)m.objs[r].alias;
    alias[o] = (int32_t)r;
  }
}
// U4: (loser, winner) pairs of the last call; returns their number
int oracle_last_merges(void *h, int32_t *from, int32_t *into) {
  Map &m = *(Map *)h;
  for (size_t i = 0; i < m.merged_from.size(); ++i) {
    if (from) from[i] = m.merged_from[i];
    if (into) into[i] = m.merged_into[i];
  }
  return (int)m.merged_from.size();
}
// V: retained views, [N, k] records of 12 floats/ints each: frame, det, n_px, cam[3], dir[3], dist; counts [N]
typedef struct {
  int32_t frame, det;
  uint32_t n_px;
  float cam[3], dir[3], dist;
} oracle_view;
void oracle_read_views(void *h, oracle_view *views, int32_t *counts, int k) {
  Map &m = *(Map *)h;
  for (size_t o = 0; o < m.objs.size(); ++o) {
    counts[o] = (int32_t)m.objs[o].views.size();
    for (int i = 0; i < k; ++i) {
      oracle_view &q = views[o * (size_t)k + i];
      std::memset(&q, 0, sizeof q);
      q.frame = q.det = -1;
      if (i < (int)m.objs[o].views.size()) {
        const View &v = m.objs[o].views[i];
        q.frame = v.frame, q.det = v.det, q.n_px = v.n_px, q.dist = v.dist;
        for (int c = 0; c < 3; ++c) q.cam[c] = v.cam[c], q.dir[c] = v.dir[c];
      }
    }
  }
}

// ---- Q1-Q5: retrieval-side scoring, a second workload over the finished memory.
// Inputs (the three retrieval embedding spaces of PAPER.md:356 are INPUTS here, as descriptors are for the mapper):
//   emb[s]  [N, dim[s]] fp32 values of the storage dtype, s = 0 caption text, 1 image (SigLIP2-like), 2 image (VL-like)
//   cls     [N] class id per entity (int), centroid [N,3] entity centroids (Gaussian mean where the entity has one)
//   alive   [N] 0/1
//   channels of ONE query variable: q[0] target description in space 0 (w = 1.0), q[1] raw utterance in space 0
//   (w = 0.5), q[2] prompt (ensemble mean) in space 1 (w = 0.75), q[3] target description in space 2 (w = 1.0).
// Q1 per channel: cos of the query with every live entity (R15 arithmetic), rank 1 = largest, ties -> lower id.
// Q2 s_sem(o) = sum_c w_c / (mu + rank_c(o)), mu = 5  ("each channel contributes w/(mu+rank) with offset mu = 5").
// Q3 class factor: s_sem *= 0.3 when target_class >= 0 and cls[o] != target_class.
// Q4 predicates, each with its own landmark variable (4 channels); the landmark is bound greedily to its top-scoring
//    live entity (largest fused rank score, ties -> lowest id).  Near: exp(-d^2 / (2 sigma^2)), sigma = 0.5 m; NextTo:
//    sigma = 1.0 m, d = inter-centroid distance.  Closest / Farthest: 1 / (|rank - r*| + 1) with rank = position of the
//    entity among the live entities ordered by d (1 = nearest, ties -> lower id), r* = 1 / n_live.
// Q5 gbar = geometric mean of the predicate scores (1 with no predicate); s = s_sem * ((1 - w) + w * gbar), w = 0.5.
// Output: s_sem [N], gbar [N], s [N] (0 for dead entities), landmark ids [P], and the top-K ids by s (ties -> lower id).
namespace {
struct RankItem {
  float c;
  int o;
};
void rrf_scores(int N, const uint8_t *alive, const float *const *emb, const int *dim, const float *const *q,
                std::vector<double> &out, std::vector<float> *cos_out) {
  static const int space_of[4] = {0, 0, 1, 2};
  static const double wch[4] = {1.0, 0.5, 0.75, 1.0};
  out.assign(N, 0.0);
  for (int ch = 0; ch < 4; ++ch) {
    const int sp = space_of[ch], Dn = dim[sp];
    std::vector<RankItem> items;
    for (int o = 0; o < N; ++o) {
      if (!alive[o]) continue;
      const float c = cosine(q[ch], emb[sp] + (size_t)o * Dn, Dn);
      items.push_back({c, o});
      if (cos_out) cos_out[ch][o] = c;
    }
    std::stable_sort(items.begin(), items.end(), [](const RankItem &x, const RankItem &y) { return x.c > y.c; });
    for (size_t r = 0; r < items.size(); ++r) out[items[r].o] += wch[ch] / (5.0 + (double)(r + 1));
  }
}
}  // namespace

int oracle_query(int N, const uint8_t *alive, const float *emb0, const float *emb1, const float *emb2, int d0, int d1, int d2,
                 const int32_t *cls, const float *centroid, const float *q_target /*concat of 4 channel vectors*/,
                 int target_class, int P, const int32_t *pred_type, const float *q_landmarks /*P x concat of 4*/,
                 int topk, float *s_sem_out, float *gbar_out, float *s_out, int32_t *landmark_out, int32_t *top_out,
                 float *cos_out /*[4,N] target channels, may be NULL*/) {
  const float *emb[3] = {emb0, emb1, emb2};
  const int dim[3] = {d0, d1, d2};
  const int qlen = d0 + d0 + d1 + d2;
  auto split = [&](const float *base, const float *q[4]) {
    q[0] = base, q[1] = base + d0, q[2] = base + 2 * d0, q[3] = base + 2 * d0 + d1;
  };
  const float *qt[4];
  split(q_target, qt);
  std::vector<double> ssem;
  std::vector<float> cosbuf[4];
  if (cos_out)
    for (int c = 0; c < 4; ++c) cosbuf[c].assign(N, 0.0f);
  rrf_scores(N, alive, emb, dim, qt, ssem, cos_out ? cosbuf : nullptr);
  if (cos_out)
    for (int c = 0; c < 4; ++c) std::memcpy(cos_out + (size_t)c * N, cosbuf[c].data(), sizeof(float) * N);
  int n_live = 0;
  for (int o = 0; o < N; ++o) n_live += alive[o] ? 1 : 0;
  std::vector<double> logsum(N, 0.0);
  std::vector<char> zero(N, 0);
  for (int p = 0; p < P; ++p) {
    const float *ql[4];
    split(q_landmarks + (size_t)p * qlen, ql);
    std::vector<double> ls;
    rrf_scores(N, alive, emb, dim, ql, ls, nullptr);
    int lm = -1;
    for (int o = 0; o < N; ++o)
      if (alive[o] && (lm < 0 || ls[o] > ls[lm])) lm = o;
    landmark_out[p] = lm;
    if (lm < 0) continue;
    std::vector<double> dist(N, 0.0);
    for (int o = 0; o < N; ++o) {
      double d2s = 0;
      for (int k = 0; k < 3; ++k) {
        const double d = (double)centroid[3 * o + k] - (double)centroid[3 * lm + k];
        d2s += d * d;
      }
      dist[o] = std::sqrt(d2s);
    }
    std::vector<int> order;
    for (int o = 0; o < N; ++o)
      if (alive[o]) order.push_back(o);
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) { return dist[x] < dist[y]; });
    std::vector<int> rank(N, 0);
    for (size_t r = 0; r < order.size(); ++r) rank[order[r]] = (int)r + 1;
    for (int o = 0; o < N; ++o) {
      if (!alive[o]) continue;
      double g = 0;
      switch (pred_type[p]) {
        case 0: g = std::exp(-dist[o] * dist[o] / (2.0 * 0.5 * 0.5)); break;           // Near, sigma = 0.5 m
        case 1: g = std::exp(-dist[o] * dist[o] / (2.0 * 1.0 * 1.0)); break;           // NextTo, sigma = 1.0 m
        case 2: g = 1.0 / (std::abs(rank[o] - 1) + 1.0); break;                         // Closest: r* = 1
        case 3: g = 1.0 / (std::abs(rank[o] - n_live) + 1.0); break;                    // Farthest: r* = n_live
        default: return -1;
      }
      if (g > 0) logsum[o] += std::log(g); else zero[o] = 1;
    }
  }
  std::vector<RankItem> fin;
  for (int o = 0; o < N; ++o) {
    double ss = alive[o] ? ssem[o] : 0.0;
    if (alive[o] && target_class >= 0 && cls[o] != target_class) ss *= 0.3;         // Q3 soft class factor
    const double gb = !alive[o] ? 0.0 : (P == 0 ? 1.0 : (zero[o] ? 0.0 : std::exp(logsum[o] / P)));
    const double sc = ss * ((1.0 - 0.5) + 0.5 * gb);                                  // Q5, w = 0.5
    s_sem_out[o] = (float)ss;
    gbar_out[o] = (float)gb;
    s_out[o] = (float)sc;
    if (alive[o]) fin.push_back({(float)sc, o});
  }
  std::stable_sort(fin.begin(), fin.end(), [](const RankItem &x, const RankItem &y) { return x.c > y.c; });
  for (int k = 0; k < topk; ++k) top_out[k] = k < (int)fin.size() ? fin[k].o : -1;
  return 0;
}

double oracle_bhattacharyya(const double *mu1, const double *cov1, const double *mu2, const double *cov2, double eps2) {
  return bhattacharyya(mu1, cov1, mu2, cov2, eps2);
}
double oracle_hellinger(const double *mu1, const double *cov1, const double *mu2, const double *cov2, double eps2) {
  return hellinger(mu1, cov1, mu2, cov2, eps2);
}
float oracle_round_to_storage(float f, int dtype) { return round_to_storage(f, dtype); }
float oracle_cosine(const float *a, const float *b, int D) { return cosine(a, b, D); }

}  // extern "C"
