// tomogen — seeded synthetic tomography systems (the five BASELINE.json configs).
//
// INPUT GENERATOR ONLY.  This module serves both the CPU oracle (oracle/) and the CUDA library
// (paper_2604_11920_b200/); it holds none of the LSQR method's arithmetic and is imported by
// neither of their sources.  It builds, deterministically from a seed:
//   * the CSR matrix A = [G; S]: G = traveltime-sensitivity rows, one per (station pair, period),
//     whose nonzeros are (bilinear lateral weight of node k on the ray, Eq. 1)
//     x (depth kernel of the period over layers, Eq. 2/5), with the unknowns
//     ordered depth-fastest, column l = k*nz + j (Eq. 7);  S = 7-point 3-D Laplacian
//     smoothing rows (BASELINE.json north_star / configs; not in the paper);
//   * x_true and the right-hand side(s) b = [G x_true + noise; 0].
// The recipe (readings G1-G12 of SURVEY.md §8d) is stated there; the
// paper's own data set is not reproduced, these systems only take its shape.
//
// Determinism: every row is a pure function of the station coordinates (and, for bent rays, one
// per-pair offset) drawn up front from a self-contained xoshiro256** stream, so the arrays do not
// depend on the number of OpenMP threads.  libm (exp, sqrt, log, cos, sin) is the only library.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

struct Rng {  // splitmix64-seeded xoshiro256**
  uint64_t s[4];
  bool have_spare = false;
  double spare = 0.0;
  static uint64_t splitmix(uint64_t& z) {
    z += 0x9E3779B97F4A7C15ull;
    uint64_t r = z;
    r = (r ^ (r >> 30)) * 0xBF58476D1CE4E5B9ull;
    r = (r ^ (r >> 27)) * 0x94D049BB133111EBull;
    return r ^ (r >> 31);
  }
  explicit Rng(uint64_t seed) {
    uint64_t z = seed;
    for (int i = 0; i < 4; ++i) s[i] = splitmix(z);
  }
  static uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
  uint64_t next() {
    uint64_t r = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
    return r;
  }
  double uniform() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }  // [0,1)
  double normal() {  // Box-Muller, both branches used
    if (have_spare) { have_spare = false; return spare; }
    double u1;
    do { u1 = uniform(); } while (u1 <= 0.0);
    double u2 = uniform();
    double r = std::sqrt(-2.0 * std::log(u1)), a = 6.283185307179586476925286766559 * u2;
    spare = r * std::sin(a); have_spare = true;
    return r * std::cos(a);
  }
};

struct Config {
  int id;
  int nx, ny, nz, nst, nper, keep;
  double sigma, wsm, damp;
  int bent;          // 1: quadratic Bezier rays (config 4)
  int clustered;     // 1: 60 % of the stations in a 6x6 patch (config 4)
  int64_t npairs_req;  // 0 = all pairs; else random subset (config 2)
  double paircap;    // pair-distance cap for the subset (config 2)
  int nrhs;
  int xkind;         // 0 checkerboard(4,2), 1 smooth random field, 2 checkerboards 2..9 (config 3)
  uint64_t geom_seed, rhs_seed;
};

bool make_config(int id, Config& c) {
  const uint64_t base = 119200;
  switch (id) {
    case 0: c = {0, 16, 16, 8, 20, 5, 8, 1.5, 2.0, 0.10, 0, 0, 0, 0.0, 1, 0, base + 0, base + 0}; return true;
    case 1: c = {1, 48, 48, 20, 229, 10, 12, 2.5, 2.0, 0.05, 0, 0, 0, 0.0, 1, 1, base + 1, base + 1}; return true;
    case 2: c = {2, 128, 128, 40, 1000, 16, 12, 2.5, 1.5, 0.02, 0, 0, 200000, 64.0, 1, 1, base + 2, base + 2}; return true;
    case 3: c = {3, 48, 48, 20, 229, 10, 12, 2.5, 2.0, 0.05, 0, 0, 0, 0.0, 8, 2, base + 1, base + 3}; return true;  // config-1 matrix
    case 4: c = {4, 48, 48, 20, 229, 10, 12, 2.5, 2.0, 0.05, 1, 1, 0, 0.0, 1, 1, base + 4, base + 4}; return true;
    default: return false;
  }
}

struct Gen {
  Config c;
  int64_t n, m_data, m, nnz, npairs;
  std::vector<double> sx, sy;          // station coordinates
  std::vector<int32_t> pa, pb;         // pair -> stations
  std::vector<double> bez;             // per-pair Bezier offset factor (bent rays)
  std::vector<int32_t> pair_nodes;     // lateral nodes touched by each pair (count)
  std::vector<int64_t> pair_off;       // nnz offset of the pair's first row
  std::vector<double> kern;            // nper x keep depth-kernel values (window only)
  std::vector<int32_t> kern_j0;        // first layer of each period's window
  std::vector<double> raylen;
};

// Depth kernel of period p: Gaussian over layers centred at c_p, sigma; the `keep` largest layers
// (a contiguous window, ties -> smaller j), renormalised to sum 1 (readings G5).
void build_kernels(Gen& g) {
  const Config& c = g.c;
  g.kern.assign((size_t)c.nper * c.keep, 0.0);
  g.kern_j0.assign(c.nper, 0);
  for (int p = 0; p < c.nper; ++p) {
    double cp = 1.0 + (c.nper > 1 ? p * (c.nz - 2.4) / (c.nper - 1) : 0.0);
    std::vector<double> v(c.nz);
    for (int j = 0; j < c.nz; ++j) { double t = (j - cp) / c.sigma; v[j] = std::exp(-0.5 * t * t); }
    std::vector<int> idx(c.nz);
    for (int j = 0; j < c.nz; ++j) idx[j] = j;
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return v[a] > v[b]; });
    int j0 = c.nz, j1 = -1;
    for (int t = 0; t < c.keep; ++t) { j0 = std::min(j0, idx[t]); j1 = std::max(j1, idx[t]); }
    // unimodal => contiguous; guard anyway
    if (j1 - j0 + 1 != c.keep) { j0 = std::max(0, std::min(c.nz - c.keep, j0)); }
    double s = 0.0;
    for (int t = 0; t < c.keep; ++t) s += v[j0 + t];
    for (int t = 0; t < c.keep; ++t) g.kern[(size_t)p * c.keep + t] = v[j0 + t] / s;
    g.kern_j0[p] = j0;
  }
}

struct Scratch {
  std::vector<double> W;        // dense nx*ny accumulator
  std::vector<int32_t> touched;
  std::vector<char> mark;
  explicit Scratch(int nlat) : W(nlat, 0.0), mark(nlat, 0) { touched.reserve(1024); }
};

inline void add_sample(const Config& c, Scratch& s, double px, double py, double ds) {
  double gx = std::min(std::max(px - 0.5, 0.0), (double)(c.nx - 1));
  double gy = std::min(std::max(py - 0.5, 0.0), (double)(c.ny - 1));
  int ix = std::min((int)std::floor(gx), c.nx - 2), iy = std::min((int)std::floor(gy), c.ny - 2);
  double fx = gx - ix, fy = gy - iy;
  const int node[4] = {iy * c.nx + ix, iy * c.nx + ix + 1, (iy + 1) * c.nx + ix, (iy + 1) * c.nx + ix + 1};
  const double w[4] = {(1 - fx) * (1 - fy), fx * (1 - fy), (1 - fx) * fy, fx * fy};
  for (int q = 0; q < 4; ++q) {
    if (!s.mark[node[q]]) { s.mark[node[q]] = 1; s.touched.push_back(node[q]); }
    s.W[node[q]] += ds * w[q];
  }
}

// Lateral footprint of one pair: sorted node list (weights > 0 only) in s.touched / s.W.
// Returns the ray length (sum of segment lengths).  Readings G3 (straight) and G4 (bent).
double lateral(const Gen& g, int64_t pair, Scratch& s) {
  const Config& c = g.c;
  for (int32_t k : s.touched) { s.W[k] = 0.0; s.mark[k] = 0; }
  s.touched.clear();
  double ax = g.sx[g.pa[pair]], ay = g.sy[g.pa[pair]], bx = g.sx[g.pb[pair]], by = g.sy[g.pb[pair]];
  double dx = bx - ax, dy = by - ay, L = std::sqrt(dx * dx + dy * dy);
  int nseg = std::max(1, (int)std::ceil(L / 0.5));
  double total = 0.0;
  if (!c.bent) {
    double ds = L / nseg;
    for (int q = 0; q < nseg; ++q) {
      double t = (q + 0.5) / nseg;
      add_sample(c, s, ax + t * dx, ay + t * dy, ds);
    }
    total = L;
  } else {
    double inv = L > 0 ? 1.0 / L : 0.0;
    double cx = 0.5 * (ax + bx) + (-dy * inv) * g.bez[pair] * L, cy = 0.5 * (ay + by) + (dx * inv) * g.bez[pair] * L;
    auto B = [&](double t, double& x, double& y) {
      double a = (1 - t) * (1 - t), b = 2 * (1 - t) * t, d = t * t;
      x = a * ax + b * cx + d * bx; y = a * ay + b * cy + d * by;
    };
    for (int q = 0; q < nseg; ++q) {
      double t0 = (double)q / nseg, t1 = (double)(q + 1) / nseg, x0, y0, x1, y1, xm, ym;
      B(t0, x0, y0); B(t1, x1, y1); B(0.5 * (t0 + t1), xm, ym);
      double ds = std::sqrt((x1 - x0) * (x1 - x0) + (y1 - y0) * (y1 - y0));
      add_sample(c, s, xm, ym, ds);
      total += ds;
    }
  }
  // drop exact zeros, sort ascending
  size_t w = 0;
  for (size_t i = 0; i < s.touched.size(); ++i) {
    int32_t k = s.touched[i];
    if (s.W[k] != 0.0) s.touched[w++] = k; else { s.mark[k] = 0; }
  }
  s.touched.resize(w);
  std::sort(s.touched.begin(), s.touched.end());
  return total;
}

void draw_geometry(Gen& g) {
  const Config& c = g.c;
  Rng r(c.geom_seed);
  g.sx.resize(c.nst); g.sy.resize(c.nst);
  int ncl = 0; double cx0 = 0, cy0 = 0;
  if (c.clustered) {
    ncl = (int)std::floor(0.6 * c.nst + 0.5);
    cx0 = r.uniform() * (c.nx - 6); cy0 = r.uniform() * (c.ny - 6);
  }
  for (int i = 0; i < c.nst; ++i) {
    double ux = r.uniform(), uy = r.uniform();
    if (i < ncl) { g.sx[i] = cx0 + 6.0 * ux; g.sy[i] = cy0 + 6.0 * uy; }
    else { g.sx[i] = ux * c.nx; g.sy[i] = uy * c.ny; }
  }
  if (c.npairs_req == 0) {
    for (int a = 0; a < c.nst; ++a) for (int b = a + 1; b < c.nst; ++b) { g.pa.push_back(a); g.pb.push_back(b); }
  } else {
    // selection sampling (order-preserving) among pairs within the distance cap (reading G7)
    double cap = c.paircap;
    int64_t qual = 0;
    for (;;) {
      qual = 0;
      for (int a = 0; a < c.nst; ++a) for (int b = a + 1; b < c.nst; ++b) {
        double dx = g.sx[a] - g.sx[b], dy = g.sy[a] - g.sy[b];
        if (dx * dx + dy * dy <= cap * cap) ++qual;
      }
      if (qual >= c.npairs_req) break;
      cap += 1.0;
    }
    int64_t need = c.npairs_req, left = qual;
    for (int a = 0; a < c.nst; ++a) for (int b = a + 1; b < c.nst; ++b) {
      double dx = g.sx[a] - g.sx[b], dy = g.sy[a] - g.sy[b];
      if (dx * dx + dy * dy > cap * cap) continue;
      double u = r.uniform();
      if (u * (double)left < (double)need) { g.pa.push_back(a); g.pb.push_back(b); --need; }
      --left;
    }
  }
  g.npairs = (int64_t)g.pa.size();
  g.bez.assign(g.npairs, 0.0);
  if (c.bent) for (int64_t i = 0; i < g.npairs; ++i) g.bez[i] = -0.3 + 0.6 * r.uniform();
}

void count_rows(Gen& g) {
  const Config& c = g.c;
  g.pair_nodes.assign(g.npairs, 0);
  g.raylen.assign(g.npairs, 0.0);
#pragma omp parallel
  {
    Scratch s(c.nx * c.ny);
#pragma omp for schedule(dynamic, 64)
    for (int64_t p = 0; p < g.npairs; ++p) {
      g.raylen[p] = lateral(g, p, s);
      g.pair_nodes[p] = (int32_t)s.touched.size();
    }
  }
  g.pair_off.assign(g.npairs + 1, 0);
  for (int64_t p = 0; p < g.npairs; ++p)
    g.pair_off[p + 1] = g.pair_off[p] + (int64_t)g.pair_nodes[p] * c.keep * c.nper;
  g.n = (int64_t)c.nx * c.ny * c.nz;
  g.m_data = g.npairs * c.nper;
  g.m = g.m_data + g.n;
}

inline int smooth_row(const Config& c, int64_t l, int32_t* col, double* val) {
  int j = (int)(l % c.nz);
  int64_t k = l / c.nz;
  int ix = (int)(k % c.nx), iy = (int)(k / c.nx);
  const int64_t sy = (int64_t)c.nx * c.nz, sx = c.nz;
  int deg = (iy > 0) + (iy < c.ny - 1) + (ix > 0) + (ix < c.nx - 1) + (j > 0) + (j < c.nz - 1);
  int q = 0;
  if (iy > 0) { col[q] = (int32_t)(l - sy); val[q++] = -c.wsm; }
  if (ix > 0) { col[q] = (int32_t)(l - sx); val[q++] = -c.wsm; }
  if (j > 0) { col[q] = (int32_t)(l - 1); val[q++] = -c.wsm; }
  col[q] = (int32_t)l; val[q++] = c.wsm * deg;
  if (j < c.nz - 1) { col[q] = (int32_t)(l + 1); val[q++] = -c.wsm; }
  if (ix < c.nx - 1) { col[q] = (int32_t)(l + sx); val[q++] = -c.wsm; }
  if (iy < c.ny - 1) { col[q] = (int32_t)(l + sy); val[q++] = -c.wsm; }
  return q;
}

inline int smooth_len(const Config& c, int64_t l) {
  int j = (int)(l % c.nz);
  int64_t k = l / c.nz;
  int ix = (int)(k % c.nx), iy = (int)(k / c.nx);
  return 1 + (iy > 0) + (iy < c.ny - 1) + (ix > 0) + (ix < c.nx - 1) + (j > 0) + (j < c.nz - 1);
}

int64_t smooth_nnz(const Config& c) {
  // total = n (diagonals) + 2*(number of in-grid neighbour links)
  int64_t nx = c.nx, ny = c.ny, nz = c.nz;
  return nx * ny * nz + 2 * ((nx - 1) * ny * nz + nx * (ny - 1) * nz + nx * ny * (nz - 1));
}

void xtrue(const Gen& g, int rhs, double* x) {
  const Config& c = g.c;
  auto checker = [&](int blk, int vblk) {
    for (int iy = 0; iy < c.ny; ++iy) for (int ix = 0; ix < c.nx; ++ix) for (int j = 0; j < c.nz; ++j) {
      int par = (ix / blk + iy / blk + j / vblk) & 1;
      x[((int64_t)iy * c.nx + ix) * c.nz + j] = par ? -0.05 : 0.05;
    }
  };
  if (c.xkind == 0) { checker(4, 2); return; }
  if (c.xkind == 2) { checker(2 + rhs, 2); return; }
  // smooth random field: N(0,1), separable Gaussian sigma = 3 index units, taps +-12, edge-renormalised
  Rng r(c.rhs_seed * 1000003ull + 17);
  std::vector<double> f(g.n), t(g.n);
  for (int64_t l = 0; l < g.n; ++l) f[l] = r.normal();
  double tap[25];
  for (int d = -12; d <= 12; ++d) tap[d + 12] = std::exp(-0.5 * (d / 3.0) * (d / 3.0));
  const int dims[3] = {c.nz, c.nx, c.ny};
  const int64_t strides[3] = {1, c.nz, (int64_t)c.nz * c.nx};
  for (int ax = 0; ax < 3; ++ax) {
    int len = dims[ax]; int64_t st = strides[ax];
    for (int64_t l = 0; l < g.n; ++l) {
      int pos = (int)((l / st) % len);
      double s = 0.0, w = 0.0;
      for (int d = -12; d <= 12; ++d) {
        int q = pos + d;
        if (q < 0 || q >= len) continue;
        s += tap[d + 12] * f[l + (int64_t)d * st]; w += tap[d + 12];
      }
      t[l] = s / w;
    }
    f.swap(t);
  }
  double mx = 0.0;
  for (int64_t l = 0; l < g.n; ++l) mx = std::max(mx, std::fabs(f[l]));
  double sc = mx > 0 ? 0.05 / mx : 0.0;
  for (int64_t l = 0; l < g.n; ++l) x[l] = f[l] * sc;
}

}  // namespace

extern "C" {

void* tomogen_open(int cfg) {
  Config c;
  if (!make_config(cfg, c)) return nullptr;
  Gen* g = new (std::nothrow) Gen();
  if (!g) return nullptr;
  g->c = c;
  build_kernels(*g);
  draw_geometry(*g);
  count_rows(*g);
  g->nnz = g->pair_off[g->npairs] + smooth_nnz(c);
  return g;
}

void tomogen_close(void* h) { delete (Gen*)h; }

// out[0..11] = m, n, nnz, m_data, nx, ny, nz, nper, npairs, keep, nrhs, nst
void tomogen_dims(void* h, int64_t* out) {
  Gen* g = (Gen*)h;
  out[0] = g->m; out[1] = g->n; out[2] = g->nnz; out[3] = g->m_data; out[4] = g->c.nx; out[5] = g->c.ny;
  out[6] = g->c.nz; out[7] = g->c.nper; out[8] = g->npairs; out[9] = g->c.keep; out[10] = g->c.nrhs; out[11] = g->c.nst;
}

// out[0..2] = damp, smoothing weight, kernel sigma
void tomogen_params(void* h, double* out) {
  Gen* g = (Gen*)h;
  out[0] = g->c.damp; out[1] = g->c.wsm; out[2] = g->c.sigma;
}

void tomogen_rowptr(void* h, int64_t* rowptr) {
  Gen* g = (Gen*)h;
  const Config& c = g->c;
#pragma omp parallel for schedule(static)
  for (int64_t p = 0; p < g->npairs; ++p) {
    int64_t len = (int64_t)g->pair_nodes[p] * c.keep;
    for (int q = 0; q < c.nper; ++q) rowptr[p * c.nper + q] = g->pair_off[p] + q * len;
  }
  int64_t off = g->pair_off[g->npairs];
  for (int64_t l = 0; l < g->n; ++l) { rowptr[g->m_data + l] = off; off += smooth_len(c, l); }
  rowptr[g->m] = off;
}

// Fill colind/vals of rows [r0, r1); entry e of the matrix is written at index e - base, where
// base = rowptr[r0] (so a row block can be generated into a small buffer and uploaded piecewise).
void tomogen_fill(void* h, int64_t r0, int64_t r1, int32_t* colind, double* vals) {
  Gen* g = (Gen*)h;
  const Config& c = g->c;
  if (r0 < 0) r0 = 0;
  if (r1 > g->m) r1 = g->m;
  if (r0 >= r1) return;
  auto row_start = [&](int64_t r) -> int64_t {
    if (r >= g->m_data) return -1;
    int64_t p = r / c.nper; int q = (int)(r % c.nper);
    return g->pair_off[p] + (int64_t)q * g->pair_nodes[p] * c.keep;
  };
  // base offset
  int64_t base;
  if (r0 < g->m_data) base = row_start(r0);
  else { base = g->pair_off[g->npairs]; for (int64_t l = 0; l < r0 - g->m_data; ++l) base += smooth_len(c, l); }
  int64_t d1 = std::min(r1, g->m_data);
  if (r0 < d1) {
    int64_t p0 = r0 / c.nper, p1 = (d1 - 1) / c.nper + 1;
#pragma omp parallel
    {
      Scratch s(c.nx * c.ny);
#pragma omp for schedule(dynamic, 64)
      for (int64_t p = p0; p < p1; ++p) {
        lateral(*g, p, s);
        int64_t len = (int64_t)s.touched.size() * c.keep;
        for (int q = 0; q < c.nper; ++q) {
          int64_t r = p * c.nper + q;
          if (r < r0 || r >= d1) continue;
          int64_t e = g->pair_off[p] + q * len - base;
          const double* kq = &g->kern[(size_t)q * c.keep];
          int j0 = g->kern_j0[q];
          for (int32_t k : s.touched) {
            double w = s.W[k];
            int32_t cbase = k * c.nz + j0;
            for (int t = 0; t < c.keep; ++t) { colind[e] = cbase + t; vals[e] = w * kq[t]; ++e; }
          }
        }
      }
    }
  }
  if (r1 > g->m_data) {
    int64_t l0 = std::max(r0, g->m_data) - g->m_data, l1 = r1 - g->m_data;
    int64_t e = (r0 < g->m_data) ? g->pair_off[g->npairs] - base : 0;
    if (r0 < g->m_data) { /* e already at first smoothing row */ }
    for (int64_t l = l0; l < l1; ++l) e += smooth_row(c, l, colind + e, vals + e);
  }
}

// ---- the factored parts of the data block (what tomogen_fill multiplies out): lateral footprints and depth kernels ----
// lptr[npairs + 1]: offsets of the pairs' lateral node lists
void tomogen_lateral_ptr(void* h, int64_t* lptr) {
  Gen* g = (Gen*)h;
  lptr[0] = 0;
  for (int64_t p = 0; p < g->npairs; ++p) lptr[p + 1] = lptr[p] + g->pair_nodes[p];
}

// nodes (ascending inside a pair) and accumulated weights W[k] of pairs [p0, p1), entry e written at e - lptr[p0]
void tomogen_lateral_fill(void* h, int64_t p0, int64_t p1, const int64_t* lptr, int32_t* node, double* w) {
  Gen* g = (Gen*)h;
  const Config& c = g->c;
  if (p0 < 0) p0 = 0;
  if (p1 > g->npairs) p1 = g->npairs;
#pragma omp parallel
  {
    Scratch s(c.nx * c.ny);
#pragma omp for schedule(dynamic, 64)
    for (int64_t p = p0; p < p1; ++p) {
      lateral(*g, p, s);
      int64_t e = lptr[p] - lptr[p0];
      for (int32_t k : s.touched) { node[e] = k; w[e] = s.W[k]; ++e; }
    }
  }
}

// j0[nper]: first layer of each period's window; kern[nper * keep]: the window values
void tomogen_kernels(void* h, int32_t* j0, double* kern) {
  Gen* g = (Gen*)h;
  std::memcpy(j0, g->kern_j0.data(), sizeof(int32_t) * g->c.nper);
  std::memcpy(kern, g->kern.data(), sizeof(double) * (size_t)g->c.nper * g->c.keep);
}

void tomogen_xtrue(void* h, int rhs, double* x) { xtrue(*(Gen*)h, rhs, x); }

void tomogen_raylen(void* h, double* L) { Gen* g = (Gen*)h; std::memcpy(L, g->raylen.data(), sizeof(double) * g->npairs); }

void tomogen_stations(void* h, double* xy) {
  Gen* g = (Gen*)h;
  for (int i = 0; i < g->c.nst; ++i) { xy[2 * i] = g->sx[i]; xy[2 * i + 1] = g->sy[i]; }
}

void tomogen_pairs(void* h, int32_t* ab) {
  Gen* g = (Gen*)h;
  for (int64_t i = 0; i < g->npairs; ++i) { ab[2 * i] = g->pa[i]; ab[2 * i + 1] = g->pb[i]; }
}

// b[0..m) for right-hand side `rhs`: data part d = G x_true (each row's entries in storage order)
// plus N(0, (0.01 rms(d))^2) noise drawn in row order; smoothing part 0  (readings G9, G10).
void tomogen_rhs(void* h, int rhs, double* b) {
  Gen* g = (Gen*)h;
  const Config& c = g->c;
  std::vector<double> x(g->n);
  xtrue(*g, rhs, x.data());
#pragma omp parallel
  {
    Scratch s(c.nx * c.ny);
#pragma omp for schedule(dynamic, 64)
    for (int64_t p = 0; p < g->npairs; ++p) {
      lateral(*g, p, s);
      for (int q = 0; q < c.nper; ++q) {
        const double* kq = &g->kern[(size_t)q * c.keep];
        int j0 = g->kern_j0[q];
        double d = 0.0;
        for (int32_t k : s.touched) {
          double w = s.W[k];
          const double* xk = &x[(int64_t)k * c.nz + j0];
          for (int t = 0; t < c.keep; ++t) d += (w * kq[t]) * xk[t];
        }
        b[p * c.nper + q] = d;
      }
    }
  }
  double ss = 0.0;
  for (int64_t i = 0; i < g->m_data; ++i) ss += b[i] * b[i];
  double sd = 0.01 * std::sqrt(ss / (double)std::max<int64_t>(g->m_data, 1));
  Rng r(c.rhs_seed * 1000003ull + 101 + (uint64_t)rhs);
  for (int64_t i = 0; i < g->m_data; ++i) b[i] += sd * r.normal();
  for (int64_t i = g->m_data; i < g->m; ++i) b[i] = 0.0;
}

}  // extern "C"
