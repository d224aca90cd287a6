// ORACLE — TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, obviously-correct CPU statement of what the BVH search of arXiv 2507.23700
// (ArborX 2.0) returns.  A BVH is an exact index (§2.1.1: "indices (the indices
// of the bounding boxes that satisfy the queries) and offsets"; §2.1.2: nearest
// search uses distances to the user data), so the result has a plain definition and the
// oracle IS that definition written out:
//   mode 0  brute force: the definition verbatim, double loop.
//   mode 1  hashed uniform grid: the same per-pair predicate, evaluated only on the
//           primitives of the grid cells that can hold a match (SURVEY.md §8(c-2) Mode B).
// All arithmetic is fp64 on the caller's fp32 inputs.  Shares no code, header, table or
// helper with the CUDA path; only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may call it.  Never tuned for speed.
//
// Pins (tests/test_oracle_pins.py): integer-lattice closed forms, box-lattice closed forms,
// 1-D numpy.searchsorted, grid == brute force, symmetry, monotonicity.  No function here is
// "parity unpinned".
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum Kind { POINT = 0, BOX = 1, SPHERE = 2 };

inline int row_width(int kind, int D) { return kind == POINT ? D : kind == BOX ? 2 * D : D + 1; }

// ---- helper distances, SURVEY.md §8(c-1) "Helper distances" --------------------------------
// squared Euclidean distance between two points
inline double dist2_pp(const float* x, const float* y, int D) {
  double s = 0.0;
  for (int a = 0; a < D; ++a) { double d = (double)x[a] - (double)y[a]; s += d * d; }
  return s;
}
// squared distance from point x to closed box [lo,hi]:  sum_a max(0, lo_a-x_a, x_a-hi_a)^2
inline double dist2_pb(const float* x, const float* lo, const float* hi, int D) {
  double s = 0.0;
  for (int a = 0; a < D; ++a) {
    double d = std::max(0.0, std::max((double)lo[a] - (double)x[a], (double)x[a] - (double)hi[a]));
    s += d * d;
  }
  return s;
}

// Result of one predicate evaluation: 0 = no match, 1 = sure match, 2 = match inside the
// tolerance band |t - T| <= eps*T; exact predicates never return 2.
inline int classify(double t, double T, double eps) {
  if (T == 0.0) return t <= 0.0 ? 1 : 0;          // r = 0: exact comparison, no band
  if (std::fabs(t - T) <= eps * T) return 2;
  return t < T ? 1 : 0;
}

// The table of SURVEY.md §8(c-1): query kind x primitive kind, all sets closed (reading A1),
// Euclidean norm (A2), no self-exclusion (A3).  PAPER.md:L69 (radius), L60/L149 (intersects).
inline int predicate(const float* q, int qkind, const float* p, int pkind, int D, double eps) {
  if (qkind == SPHERE) {
    double r = q[D];
    if (r < 0.0) return 0;                        // reading A21: negative radius matches nothing
    if (pkind == POINT) return classify(dist2_pp(p, q, D), r * r, eps);
    if (pkind == BOX) return classify(dist2_pb(q, p, p + D, D), r * r, eps);
    double R = p[D];
    return classify(dist2_pp(p, q, D), (r + R) * (r + R), eps);
  }
  if (qkind == BOX) {
    const float *qlo = q, *qhi = q + D;
    if (pkind == POINT) {
      for (int a = 0; a < D; ++a) if (!(qlo[a] <= p[a] && p[a] <= qhi[a])) return 0;
      return 1;
    }
    if (pkind == BOX) {
      for (int a = 0; a < D; ++a) if (!(p[a] <= qhi[a] && qlo[a] <= p[D + a])) return 0;
      return 1;
    }
    double R = p[D];
    return classify(dist2_pb(p, qlo, qhi, D), R * R, eps);
  }
  // POINT query
  if (pkind == POINT) {
    for (int a = 0; a < D; ++a) if (!(p[a] == q[a])) return 0;
    return 1;
  }
  if (pkind == BOX) {
    for (int a = 0; a < D; ++a) if (!(p[a] <= q[a] && q[a] <= p[D + a])) return 0;
    return 1;
  }
  double R = p[D];
  return classify(dist2_pp(q, p, D), R * R, eps);
}

// kNN distance from query point y to the stored geometry ("fine" search, PAPER.md:L79;
// SURVEY.md §8(c-1) last table row).
inline double knn_distance(const float* y, const float* p, int pkind, int D) {
  if (pkind == POINT) return std::sqrt(dist2_pp(p, y, D));
  if (pkind == BOX) return std::sqrt(dist2_pb(y, p, p + D, D));
  return std::max(0.0, std::sqrt(dist2_pp(p, y, D)) - (double)p[D]);
}

struct SpatialResult {
  std::vector<int64_t> offsets;   // nq+1
  std::vector<int32_t> indices;   // rows ascending by primitive index
  std::vector<uint8_t> band;      // 1 where the pair is inside the tolerance band
};

struct Hit { int32_t i; uint8_t band; };

// ---- hashed uniform grid (Mode B) -----------------------------------------------------------
struct Grid {
  int D = 0, pkind = 0;
  int64_t n = 0;
  const float* prims = nullptr;
  double cell = 1.0;
  double L[10];             // lower corner of the box of primitive centres
  int64_t ncell[10];        // cells per axis
  int64_t stride[10];
  double H[10];             // max half extent of any primitive along each axis
  double Hinf = 0.0;
  std::vector<int64_t> keys;     // sorted unique cell keys
  std::vector<int64_t> start;    // start[c]..start[c+1] into order
  std::vector<int32_t> order;    // primitive ids grouped by cell

  void centre(int64_t i, double* c) const {
    const float* p = prims + i * row_width(pkind, D);
    for (int a = 0; a < D; ++a)
      c[a] = pkind == BOX ? 0.5 * ((double)p[a] + (double)p[D + a]) : (double)p[a];
  }
  int64_t coord(double x, int a) const {      // cell coordinate, clamped into the grid
    double z = std::floor((x - L[a]) / cell);
    if (!(z >= 0.0)) return 0;
    if (z >= (double)ncell[a]) return ncell[a] - 1;
    return (int64_t)z;
  }
  void build(const float* p, int64_t n_, int D_, int pkind_, double cell_) {
    prims = p; n = n_; D = D_; pkind = pkind_;
    double U[10];
    for (int a = 0; a < D; ++a) { L[a] = 1e300; U[a] = -1e300; H[a] = 0.0; }
    int w = row_width(pkind, D);
    for (int64_t i = 0; i < n; ++i) {
      double c[10]; centre(i, c);
      const float* pi = prims + i * w;
      for (int a = 0; a < D; ++a) {
        L[a] = std::min(L[a], c[a]); U[a] = std::max(U[a], c[a]);
        // half extent measured from the centre used for binning
        double h = pkind == BOX ? std::max((double)pi[D + a] - c[a], c[a] - (double)pi[a])
                 : pkind == SPHERE ? (double)pi[D] : 0.0;
        H[a] = std::max(H[a], h);
      }
    }
    Hinf = 0.0;
    for (int a = 0; a < D; ++a) Hinf = std::max(Hinf, H[a]);
    // cell size: caller's choice, enlarged until the linear key fits in 62 bits
    cell = cell_ > 0.0 ? cell_ : 1.0;
    for (;;) {
      double bits = 0.0;
      for (int a = 0; a < D; ++a) {
        double m = std::floor((U[a] - L[a]) / cell) + 1.0;
        ncell[a] = (int64_t)std::max(1.0, std::min(m, 4.0e18));
        bits += std::log2((double)ncell[a]);
      }
      if (bits <= 62.0) break;
      cell *= 2.0;
    }
    int64_t s = 1;
    for (int a = 0; a < D; ++a) { stride[a] = s; s *= ncell[a]; }
    std::vector<std::pair<int64_t, int32_t>> kv((size_t)n);
    for (int64_t i = 0; i < n; ++i) {
      double c[10]; centre(i, c);
      int64_t key = 0;
      for (int a = 0; a < D; ++a) key += coord(c[a], a) * stride[a];
      kv[(size_t)i] = {key, (int32_t)i};
    }
    std::sort(kv.begin(), kv.end());
    order.resize((size_t)n);
    keys.clear(); start.clear();
    for (int64_t j = 0; j < n; ++j) {
      if (j == 0 || kv[(size_t)j].first != kv[(size_t)j - 1].first) {
        keys.push_back(kv[(size_t)j].first); start.push_back(j);
      }
      order[(size_t)j] = kv[(size_t)j].second;
    }
    start.push_back(n);
  }
  // primitives of the cell with integer coordinates z (already inside the grid)
  inline void cell_range(const int64_t* z, int64_t& b, int64_t& e) const {
    int64_t key = 0;
    for (int a = 0; a < D; ++a) key += z[a] * stride[a];
    auto it = std::lower_bound(keys.begin(), keys.end(), key);
    if (it == keys.end() || *it != key) { b = e = 0; return; }
    size_t c = (size_t)(it - keys.begin());
    b = start[c]; e = start[c + 1];
  }
};

// Visit every cell z with zlo <= z <= zhi (per axis); f(z) is called with the coordinates.
template <class F>
inline void for_cells(int D, const int64_t* zlo, const int64_t* zhi, F&& f) {
  int64_t z[10];
  for (int a = 0; a < D; ++a) { if (zlo[a] > zhi[a]) return; z[a] = zlo[a]; }
  for (;;) {
    f(z);
    int a = 0;
    for (; a < D; ++a) { if (++z[a] <= zhi[a]) break; z[a] = zlo[a]; }
    if (a == D) return;
  }
}

void spatial_query_one(const Grid* g, const float* prims, int64_t n, int D, int pkind,
                       const float* q, int qkind, double eps, std::vector<Hit>& out) {
  out.clear();
  int w = row_width(pkind, D);
  if (!g) {   // Mode A: the definition, verbatim
    for (int64_t i = 0; i < n; ++i) {
      int c = predicate(q, qkind, prims + i * w, pkind, D, eps);
      if (c) out.push_back({(int32_t)i, (uint8_t)(c == 2)});
    }
    return;
  }
  // Mode B step 4: query AABB [a,b], widened by the band (r*(1+eps)) and by H_a.
  int64_t zlo[10], zhi[10];
  for (int a = 0; a < D; ++a) {
    double lo, hi;
    if (qkind == SPHERE) {
      double r = (double)q[D];
      if (r < 0.0) return;
      r *= (1.0 + eps);
      lo = (double)q[a] - r; hi = (double)q[a] + r;
    } else if (qkind == BOX) { lo = q[a]; hi = q[D + a]; if (lo > hi) return; }
    else { lo = hi = q[a]; }
    double pad = g->H[a] * (1.0 + eps) + 1e-12 * (std::fabs(lo) + std::fabs(hi));
    lo -= pad; hi += pad;
    double gmax = g->L[a] + g->cell * (double)g->ncell[a];
    if (hi < g->L[a] - g->cell || lo > gmax + g->cell) return;   // far outside: no centre there
    zlo[a] = g->coord(lo, a); zhi[a] = g->coord(hi, a);
  }
  for_cells(D, zlo, zhi, [&](const int64_t* z) {
    int64_t b, e; g->cell_range(z, b, e);
    for (int64_t j = b; j < e; ++j) {
      int32_t i = g->order[(size_t)j];
      int c = predicate(q, qkind, prims + (int64_t)i * w, pkind, D, eps);
      if (c) out.push_back({i, (uint8_t)(c == 2)});
    }
  });
  std::sort(out.begin(), out.end(), [](const Hit& x, const Hit& y) { return x.i < y.i; });
}

struct Cand { double d; int32_t i; };
inline bool cand_less(const Cand& x, const Cand& y) { return x.d < y.d || (x.d == y.d && x.i < y.i); }

// bounded max-heap of the k best (distance, index) pairs; lower index wins exact ties
struct KHeap {
  std::vector<Cand> h; size_t k;
  explicit KHeap(size_t k_) : k(k_) { h.reserve(k_ + 1); }
  void clear() { h.clear(); }
  bool full() const { return h.size() == k; }
  double worst() const { return h.front().d; }
  void push(double d, int32_t i) {
    Cand c{d, i};
    if (h.size() < k) { h.push_back(c); std::push_heap(h.begin(), h.end(), cand_less); }
    else if (cand_less(c, h.front())) {
      std::pop_heap(h.begin(), h.end(), cand_less); h.back() = c; std::push_heap(h.begin(), h.end(), cand_less);
    }
  }
};

void knn_query_one(const Grid* g, const float* prims, int64_t n, int D, int pkind,
                   const float* y, KHeap& heap) {
  heap.clear();
  int w = row_width(pkind, D);
  if (!g) {
    for (int64_t i = 0; i < n; ++i) heap.push(knn_distance(y, prims + i * w, pkind, D), (int32_t)i);
    return;
  }
  // Mode B step 5: rings of cells of growing Chebyshev radius rho around the query's cell.
  int64_t z0[10];
  for (int a = 0; a < D; ++a) z0[a] = g->coord((double)y[a], a);
  for (int64_t rho = 0;; ++rho) {
    int64_t zlo[10], zhi[10];
    bool covers = true;
    for (int a = 0; a < D; ++a) {
      zlo[a] = std::max<int64_t>(0, z0[a] - rho);
      zhi[a] = std::min<int64_t>(g->ncell[a] - 1, z0[a] + rho);
      if (zlo[a] > 0 || zhi[a] < g->ncell[a] - 1) covers = false;
    }
    for_cells(D, zlo, zhi, [&](const int64_t* z) {
      int64_t cheb = 0;
      for (int a = 0; a < D; ++a) cheb = std::max<int64_t>(cheb, std::llabs(z[a] - z0[a]));
      if (cheb != rho) return;                 // inner cells were visited by earlier rings
      int64_t b, e; g->cell_range(z, b, e);
      for (int64_t j = b; j < e; ++j) {
        int32_t i = g->order[(size_t)j];
        heap.push(knn_distance(y, prims + (int64_t)i * w, pkind, D), i);
      }
    });
    if (covers) return;
    if (!heap.full()) continue;
    // every unvisited primitive has its centre outside the visited block on some axis, hence
    // lies at distance >= beta from y (faces that coincide with the grid boundary hide nothing)
    double beta = std::numeric_limits<double>::infinity();
    for (int a = 0; a < D; ++a) {
      if (z0[a] - rho > 0) beta = std::min(beta, (double)y[a] - (g->L[a] + (double)(z0[a] - rho) * g->cell));
      if (z0[a] + rho < g->ncell[a] - 1) beta = std::min(beta, (g->L[a] + (double)(z0[a] + rho + 1) * g->cell) - (double)y[a]);
    }
    beta -= g->Hinf;
    beta -= 1e-9 * (std::fabs(beta) + g->cell);   // floor() rounding slack of the cell assignment
    if (heap.worst() < beta) return;
  }
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// Grid handle (Mode B).  cell <= 0 picks 1.0; the size is doubled until keys fit 62 bits.
void* orc_grid_build(const float* prims, int64_t n, int dim, int pkind, double cell) {
  Grid* g = new Grid();
  g->build(prims, n, dim, pkind, cell);
  return g;
}
void orc_grid_free(void* g) { delete (Grid*)g; }
double orc_grid_cell(void* g) { return ((Grid*)g)->cell; }

// Spatial search.  grid == NULL -> brute force.  Returns a result object; rows hold every
// primitive with predicate class 1 (sure) or 2 (band), ascending by index.
void* orc_spatial(void* grid, const float* prims, int64_t n, int dim, int pkind,
                  const float* queries, int64_t nq, int qkind, double eps) {
  SpatialResult* R = new SpatialResult();
  R->offsets.assign((size_t)nq + 1, 0);
  std::vector<std::vector<Hit>> rows((size_t)nq);
  int qw = row_width(qkind, dim);
#pragma omp parallel
  {
    std::vector<Hit> tmp;
#pragma omp for schedule(dynamic, 64)
    for (int64_t q = 0; q < nq; ++q) {
      spatial_query_one((const Grid*)grid, prims, n, dim, pkind, queries + q * qw, qkind, eps, tmp);
      rows[(size_t)q] = tmp;
    }
  }
  for (int64_t q = 0; q < nq; ++q) R->offsets[(size_t)q + 1] = R->offsets[(size_t)q] + (int64_t)rows[(size_t)q].size();
  R->indices.resize((size_t)R->offsets[(size_t)nq]);
  R->band.resize((size_t)R->offsets[(size_t)nq]);
#pragma omp parallel for schedule(static)
  for (int64_t q = 0; q < nq; ++q) {
    int64_t o = R->offsets[(size_t)q];
    for (size_t j = 0; j < rows[(size_t)q].size(); ++j) {
      R->indices[(size_t)o + j] = rows[(size_t)q][j].i;
      R->band[(size_t)o + j] = rows[(size_t)q][j].band;
    }
  }
  return R;
}
int64_t orc_spatial_total(void* r) { return (int64_t)((SpatialResult*)r)->indices.size(); }
void orc_spatial_copy(void* r, int64_t* offsets, int32_t* indices, uint8_t* band) {
  SpatialResult* R = (SpatialResult*)r;
  std::memcpy(offsets, R->offsets.data(), R->offsets.size() * sizeof(int64_t));
  if (!R->indices.empty()) {
    std::memcpy(indices, R->indices.data(), R->indices.size() * sizeof(int32_t));
    std::memcpy(band, R->band.data(), R->band.size());
  }
}
void orc_spatial_free(void* r) { delete (SpatialResult*)r; }

// k nearest neighbours.  Rows of k: ascending distance (fp64), ties by lower index; rows are
// padded with index -1 / distance +inf when n < k (reading A8).
void orc_knn(void* grid, const float* prims, int64_t n, int dim, int pkind,
             const float* qpoints, int64_t nq, int k, int32_t* out_idx, double* out_dist) {
#pragma omp parallel
  {
    KHeap heap((size_t)k);
#pragma omp for schedule(dynamic, 64)
    for (int64_t q = 0; q < nq; ++q) {
      knn_query_one((const Grid*)grid, prims, n, dim, pkind, qpoints + q * dim, heap);
      std::vector<Cand> s = heap.h;
      std::sort(s.begin(), s.end(), cand_less);
      for (int j = 0; j < k; ++j) {
        bool ok = (size_t)j < s.size();
        out_idx[q * k + j] = ok ? s[(size_t)j].i : -1;
        out_dist[q * k + j] = ok ? s[(size_t)j].d : std::numeric_limits<double>::infinity();
      }
    }
  }
}

// fp64 kNN distance of explicitly named (query, primitive) pairs -- used by the comparator
// to check that a reported distance belongs to the reported index (SURVEY.md §8(c-3) rule 4).
void orc_knn_distance_pairs(const float* prims, int dim, int pkind, const float* qpoints,
                            const int64_t* qids, const int32_t* pids, int64_t m, double* out) {
  int w = row_width(pkind, dim);
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < m; ++j)
    out[j] = pids[j] < 0 ? std::numeric_limits<double>::infinity()
                         : knn_distance(qpoints + qids[j] * dim, prims + (int64_t)pids[j] * w, pkind, dim);
}

}  // extern "C"
