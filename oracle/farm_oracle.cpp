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

struct Object {  // R1
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
  std::map<uint64_t, uint32_t> owner;  // R11: one owner per key
  std::vector<Object> objs;
  int64_t frame_seq = 0;
  // results of the last call
  int M = 0;
  std::vector<int32_t> assoc;
  std::vector<uint8_t> is_new;
  std::vector<float> best_score, second_score;
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
  int next_id = N;
  for (int j = 0; j < M; ++j) {
    if (m.n_px[j] == 0) {  // R8: empty detection is skipped
      m.stats.skipped++;
      continue;
    }
    for (int i = 0; i < D; ++i) a[i] = load_storage(desc, m.dtype, (size_t)j * D + i);  // R14
    float best = 0.0f, second = -std::numeric_limits<float>::infinity();
    int best_o = -1;
    for (int o = 0; o < N; ++o) {                                // R16: every pair
      const float c = cosine(a.data(), m.objs[o].shadow.data(), D);  // R15
      if (m.dense_arg[j] < 0 || c > m.dense_max[j]) {            // R16 dense row max, ties -> lowest id
        if (m.dense_arg[j] >= 0) m.dense_second[j] = std::fmax(m.dense_second[j], m.dense_max[j]);
        m.dense_max[j] = c;
        m.dense_arg[j] = o;
      } else {
        m.dense_second[j] = std::fmax(m.dense_second[j], c);
      }
      float g = 0.0f;                                            // R10
      auto it = m.overlap[j].find((uint32_t)o);
      const uint32_t cnt = it == m.overlap[j].end() ? 0u : it->second;
      const uint32_t mn = std::min<uint32_t>((uint32_t)m.V[j].size(), m.objs[o].n_voxels);
      if (mn > 0) g = (float)cnt / (float)mn;
      const float score = m.w_geo * g + m.w_sem * c;             // R17 (fp32: two mul, one add)
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
    if (best_o >= 0 && best > m.tau) {  // R18: strict
      target[j] = best_o;
      m.assoc[j] = best_o;
      m.stats.matches++;
      if (m.objs[best_o].gW > 0.0) {  // G4: distance to the matched entity's Gaussian as it was at entry (R2)
        double mu_d[3], c_d[6], mu_o[3], c_o[6];
        gaussian_from_moments((double)m.n_px[j], &m.gS1[(size_t)j * 3], &m.gS2[(size_t)j * 6], mu_d, c_d);
        gaussian_from_moments(m.objs[best_o].gW, m.objs[best_o].gM1, m.objs[best_o].gM2, mu_o, c_o);
        m.hell[j] = (float)hellinger(mu_d, c_d, mu_o, c_o, (double)m.voxel_size * (double)m.voxel_size);
      }
    } else {  // R20: new ids in order of j
      target[j] = next_id++;
      m.assoc[j] = target[j];
      m.is_new[j] = 1;
      m.stats.spawns++;
    }
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
      if (m.n_px[j] > ob.best.n_px) {  // R23: strict > keeps the earliest (frame_seq, det) on ties
        ob.best.n_px = m.n_px[j];
        ob.best.frame = (int32_t)(m.frame_seq + det_frame[j]);
        ob.best.det = det_local[j];
        const float *Tf = T + 16 * det_frame[j];
        ob.best.cam[0] = Tf[3];
        ob.best.cam[1] = Tf[7];
        ob.best.cam[2] = Tf[11];
      }
    }
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
double oracle_hellinger(const double *mu1, const double *cov1, const double *mu2, const double *cov2, double eps2) {
  return hellinger(mu1, cov1, mu2, cov2, eps2);
}
float oracle_round_to_storage(float f, int dtype) { return round_to_storage(f, dtype); }
float oracle_cosine(const float *a, const float *b, int D) { return cosine(a, b, D); }

}  // extern "C"
