// Host-side geometry of BiP-PRISM: beam sets, probe coefficients, hex-ring parents, Sibson weights.
// (readings SURVEY.md 8(c) c5-c8.)  Plain C++17, no CUDA.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>

#include "bip_internal.h"

namespace {

inline int64_t flat_index(int hy, int hx, int ny, int nx) {
  int ky = ((hy % ny) + ny) % ny, kx = ((hx % nx) + nx) % nx;
  return (int64_t)ky * nx + kx;
}

bool grid_ok(const bip_grid* g) {
  return g && g->ny >= 2 && g->nx >= 2 && g->ly > 0 && g->lx > 0 && g->nz >= 0;
}

// ---------------------------------------------------------------------------------------------------
// Convex polygons for the Voronoi-cell intersections of Sibson's construction.
// ---------------------------------------------------------------------------------------------------
struct Pt { double y, x; };

struct Poly {
  std::vector<Pt> v;
  double area() const {
    double a = 0;
    size_t n = v.size();
    for (size_t i = 0, j = n - 1; i < n; j = i++) a += v[j].x * v[i].y - v[i].x * v[j].y;
    return 0.5 * std::fabs(a);
  }
  double max_dist2(Pt c) const {
    double m = 0;
    for (auto& p : v) m = std::max(m, (p.y - c.y) * (p.y - c.y) + (p.x - c.x) * (p.x - c.x));
    return m;
  }
};

// keep {y : |y - a| <= |y - b|}; returns true if something was cut away
bool clip_closer_to(Poly& P, Pt a, Pt b, double tol, std::vector<Pt>& scratch) {
  const double ny = 2.0 * (b.y - a.y), nx = 2.0 * (b.x - a.x);
  const double c = (b.y * b.y + b.x * b.x) - (a.y * a.y + a.x * a.x);
  const size_t n = P.v.size();
  bool any = false;
  for (size_t i = 0; i < n; ++i)
    if (ny * P.v[i].y + nx * P.v[i].x - c > tol) { any = true; break; }
  if (!any) return false;
  scratch.clear();
  for (size_t i = 0; i < n; ++i) {
    const Pt &p = P.v[i], &q = P.v[(i + 1) % n];
    const double sp = ny * p.y + nx * p.x - c, sq = ny * q.y + nx * q.x - c;
    if (sp <= 0.0) scratch.push_back(p);
    if ((sp < 0.0 && sq > 0.0) || (sq < 0.0 && sp > 0.0)) {
      const double t = sp / (sp - sq);
      scratch.push_back(Pt{p.y + t * (q.y - p.y), p.x + t * (q.x - p.x)});
    }
  }
  P.v.swap(scratch);
  return true;
}

// Uniform bucket grid over the parents for ring-ordered neighbour enumeration.
struct Buckets {
  double y0, x0, cs;
  int gy, gx;
  std::vector<std::vector<int>> cell;
  void build(const std::vector<Pt>& pts) {
    double ymin = 1e300, ymax = -1e300, xmin = 1e300, xmax = -1e300;
    for (auto& p : pts) { ymin = std::min(ymin, p.y); ymax = std::max(ymax, p.y); xmin = std::min(xmin, p.x); xmax = std::max(xmax, p.x); }
    const double area = std::max((ymax - ymin) * (xmax - xmin), 1e-300);
    cs = std::sqrt(area / std::max<size_t>(pts.size(), 1)) * 1.5;
    if (!(cs > 0)) cs = 1.0;
    y0 = ymin; x0 = xmin;
    gy = std::max(1, (int)std::floor((ymax - ymin) / cs) + 1);
    gx = std::max(1, (int)std::floor((xmax - xmin) / cs) + 1);
    cell.assign((size_t)gy * gx, {});
    for (size_t i = 0; i < pts.size(); ++i) cell[(size_t)cy(pts[i].y) * gx + cx(pts[i].x)].push_back((int)i);
  }
  int cy(double y) const { return std::min(gy - 1, std::max(0, (int)std::floor((y - y0) / cs))); }
  int cx(double x) const { return std::min(gx - 1, std::max(0, (int)std::floor((x - x0) / cs))); }
  // distance from c to the nearest point outside the (2k+1)^2 block of cells centred on c's (clamped) cell
  double ring_clearance(Pt c, int k) const {
    const int iy = cy(c.y), ix = cx(c.x);
    const double lo_y = y0 + (iy - k) * cs, hi_y = y0 + (iy + k + 1) * cs;
    const double lo_x = x0 + (ix - k) * cs, hi_x = x0 + (ix + k + 1) * cs;
    double d = std::min(std::min(c.y - lo_y, hi_y - c.y), std::min(c.x - lo_x, hi_x - c.x));
    return d;   // may be negative when c lies outside the bucket grid: then no pruning for this ring
  }
  template <class F> void for_ring(Pt c, int k, F&& f) const {
    const int iy = cy(c.y), ix = cx(c.x);
    for (int y = iy - k; y <= iy + k; ++y) {
      if (y < 0 || y >= gy) continue;
      const bool edge_row = (y == iy - k) || (y == iy + k);
      for (int x = ix - k; x <= ix + k; ++x) {
        if (x < 0 || x >= gx) continue;
        if (!edge_row && x != ix - k && x != ix + k) continue;
        for (int id : cell[(size_t)y * gx + x]) f(id);
      }
    }
  }
  int max_ring(Pt c) const {
    const int iy = cy(c.y), ix = cx(c.x);
    return std::max(std::max(iy, gy - 1 - iy), std::max(ix, gx - 1 - ix));
  }
};

}  // namespace

extern "C" {

int32_t bip_beams_in_disc(const bip_grid* g, double qmax, int32_t* h_out, int32_t cap, int32_t* n_out) {
  if (!grid_ok(g) || !n_out || qmax < 0) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_beams_in_disc: bad argument");
  int32_t n = 0;
  for (int ky = 0; ky < g->ny; ++ky) {
    const int hy = ky < (g->ny + 1) / 2 ? ky : ky - g->ny;
    if (2 * std::abs(hy) >= g->ny) continue;
    for (int kx = 0; kx < g->nx; ++kx) {
      const int hx = kx < (g->nx + 1) / 2 ? kx : kx - g->nx;
      if (2 * std::abs(hx) >= g->nx) continue;
      const double qy = hy / g->ly, qx = hx / g->lx;
      if (qy * qy + qx * qx <= qmax * qmax) {
        if (h_out && n < cap) { h_out[2 * n] = hy; h_out[2 * n + 1] = hx; }
        ++n;
      }
    }
  }
  *n_out = n;
  if (h_out && n > cap) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_beams_in_disc: capacity %d < %d beams", cap, n);
  return BIP_OK;
}

int32_t bip_aperture_coeffs(const bip_grid* g, int32_t n, const int32_t* h, double defocus, float* c_out) {
  if (!grid_ok(g) || n <= 0 || !h || !c_out) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_aperture_coeffs: bad argument");
  const double norm = 1.0 / std::sqrt((double)g->ny * (double)g->nx * (double)n);
  for (int32_t b = 0; b < n; ++b) {
    const double qy = h[2 * b] / g->ly, qx = h[2 * b + 1] / g->lx;
    const double ph = -M_PI * g->lambda * defocus * (qy * qy + qx * qx);
    c_out[2 * b] = (float)(std::cos(ph) * norm);
    c_out[2 * b + 1] = (float)(std::sin(ph) * norm);
  }
  return BIP_OK;
}

int32_t bip_prism_coeffs(int32_t n_keep, const int32_t* keep, int32_t n_full, const float* c_full, int32_t fy, int32_t fx, float* c_out) {
  if (n_keep < 0 || (n_keep > 0 && (!keep || !c_out)) || !c_full || fy < 1 || fx < 1)
    return bip::fail(nullptr, BIP_ERR_INVALID, "bip_prism_coeffs: bad argument");
  const float f = (float)(fy * fx);                                   // "the DFT decimation factor"
  for (int32_t j = 0; j < n_keep; ++j) {
    if (keep[j] < 0 || keep[j] >= n_full) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_prism_coeffs: position %d outside 0..%d", keep[j], n_full - 1);
    c_out[2 * j] = c_full[2 * keep[j]] * f;
    c_out[2 * j + 1] = c_full[2 * keep[j] + 1] * f;
  }
  return BIP_OK;
}

int32_t bip_partition(const bip_grid* g, int32_t n, const int32_t* h, double qmax, double factor, int32_t max_nn, int32_t* pos_out,
                      int32_t cap, int32_t* n_parent, int32_t* nn_idx_out, float* nn_w_out) {
  if (!grid_ok(g) || n <= 0 || !h || !n_parent || !pos_out || !(factor >= 1.0) || max_nn < 1 || max_nn > BIP_MAX_NN || !nn_idx_out || !nn_w_out)
    return bip::fail(nullptr, BIP_ERR_INVALID, "bip_partition: bad argument");
  if (factor == 1.0) {                                                // the exactness limit: parents = all beams, w = identity (reading c7)
    *n_parent = n;
    if (cap < n) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_partition: capacity %d < %d parents", cap, n);
    for (int32_t b = 0; b < n; ++b) {
      pos_out[b] = b;
      for (int32_t j = 0; j < max_nn; ++j) { nn_idx_out[(size_t)b * max_nn + j] = j == 0 ? b : -1; nn_w_out[(size_t)b * max_nn + j] = j == 0 ? 1.f : 0.f; }
    }
    return BIP_OK;
  }
  int32_t st = bip_hexring(g, n, h, qmax, bip_n_radial_from_factor(n, factor), 6, pos_out, cap, n_parent);
  if (st != BIP_OK) return st;
  std::vector<int32_t> ph(2 * (size_t)*n_parent);
  for (int32_t p = 0; p < *n_parent; ++p) { ph[2 * p] = h[2 * pos_out[p]]; ph[2 * p + 1] = h[2 * pos_out[p] + 1]; }
  return bip_sibson(g, n, h, *n_parent, ph.data(), qmax, max_nn, nn_idx_out, nn_w_out);
}

int32_t bip_n_radial_from_factor(int32_t n_beams, double factor) {
  if (n_beams <= 0 || !(factor > 0)) return 1;
  return std::max(1, (int)std::floor(std::sqrt(n_beams / M_PI) / factor + 0.5));
}

int32_t bip_hexring(const bip_grid* g, int32_t n, const int32_t* h, double qmax, int32_t n_radial,
                    int32_t n_angular, int32_t* pos_out, int32_t cap, int32_t* n_out) {
  if (!grid_ok(g) || n <= 0 || !h || !n_out || n_radial < 0 || n_angular < 1)
    return bip::fail(nullptr, BIP_ERR_INVALID, "bip_hexring: bad argument");
  std::vector<double> qy(n), qx(n);
  for (int i = 0; i < n; ++i) { qy[i] = h[2 * i] / g->ly; qx[i] = h[2 * i + 1] / g->lx; }
  // beams must come in ascending flat index so that "first minimum" is "lowest flat index"
  for (int i = 1; i < n; ++i)
    if (flat_index(h[2 * i], h[2 * i + 1], g->ny, g->nx) <= flat_index(h[2 * i - 2], h[2 * i - 1], g->ny, g->nx))
      return bip::fail(nullptr, BIP_ERR_INVALID, "bip_hexring: beams not in ascending flat index");
  auto snap = [&](double sy, double sx) {
    int best = 0;
    double bd = 1e300;
    for (int i = 0; i < n; ++i) {
      const double d2 = (qy[i] - sy) * (qy[i] - sy) + (qx[i] - sx) * (qx[i] - sx);
      if (d2 < bd) { bd = d2; best = i; }
    }
    return best;
  };
  std::vector<int> chosen;
  chosen.push_back(snap(0.0, 0.0));
  for (int k = 1; k <= n_radial; ++k) {
    const double r = k * qmax / n_radial;
    const int m = n_angular * k;
    for (int j = 0; j < m; ++j) {
      const double ang = 2.0 * M_PI * j / m;
      chosen.push_back(snap(r * std::sin(ang), r * std::cos(ang)));
    }
  }
  std::sort(chosen.begin(), chosen.end());
  chosen.erase(std::unique(chosen.begin(), chosen.end()), chosen.end());
  *n_out = (int32_t)chosen.size();
  if (pos_out) {
    if ((int)chosen.size() > cap) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_hexring: capacity %d < %zu parents", cap, chosen.size());
    std::copy(chosen.begin(), chosen.end(), pos_out);
  }
  return BIP_OK;
}

int32_t bip_sibson(const bip_grid* g, int32_t n, const int32_t* h, int32_t n_parent, const int32_t* parent_h,
                   double qmax, int32_t max_nn, int32_t* nn_idx_out, float* nn_w_out) {
  if (!grid_ok(g) || n <= 0 || !h || n_parent <= 0 || !parent_h || !(qmax > 0) || max_nn < 1 || max_nn > BIP_MAX_NN ||
      !nn_idx_out || !nn_w_out)
    return bip::fail(nullptr, BIP_ERR_INVALID, "bip_sibson: bad argument");
  std::vector<Pt> par(n_parent);
  for (int p = 0; p < n_parent; ++p) par[p] = Pt{parent_h[2 * p] / g->ly, parent_h[2 * p + 1] / g->lx};
  Buckets bk;
  bk.build(par);
  const double half = 1024.0 * qmax;
  const double tol = 1e-13 * half * half;
  std::vector<Pt> scratch;
  std::vector<int> cutters;
  std::vector<std::pair<int, double>> row;

  for (int b = 0; b < n; ++b) {
    int32_t* oi = nn_idx_out + (size_t)b * max_nn;
    float* ow = nn_w_out + (size_t)b * max_nn;
    for (int j = 0; j < max_nn; ++j) { oi[j] = -1; ow[j] = 0.f; }
    const Pt x{h[2 * b] / g->ly, h[2 * b + 1] / g->lx};
    // delta on a coincident parent (lowest parent number)
    int hit = -1;
    bk.for_ring(x, 0, [&](int id) { if (par[id].y == x.y && par[id].x == x.x && (hit < 0 || id < hit)) hit = id; });
    if (hit < 0) bk.for_ring(x, 1, [&](int id) { if (par[id].y == x.y && par[id].x == x.x && (hit < 0 || id < hit)) hit = id; });
    if (hit >= 0) { oi[0] = hit; ow[0] = 1.f; continue; }

    // C(x): cell of x among parents + {x}
    Poly cx;
    cx.v = {Pt{-half, -half}, Pt{-half, half}, Pt{half, half}, Pt{half, -half}};
    cutters.clear();
    const int kmax = bk.max_ring(x);
    for (int k = 0; k <= kmax; ++k) {
      if (k > 0) {
        const double clear = bk.ring_clearance(x, k - 1);
        if (clear > 0 && clear * clear > 4.0 * cx.max_dist2(x)) break;   // nothing farther can cut C(x)
      }
      bk.for_ring(x, k, [&](int id) { if (clip_closer_to(cx, x, par[id], tol, scratch)) cutters.push_back(id); });
    }
    const double total = cx.area();
    row.clear();
    for (int p : cutters) {
      Poly q = cx;                                       // C(x) & V_P(p)
      const int kp = bk.max_ring(par[p]);
      for (int k = 0; k <= kp && q.v.size() >= 3; ++k) {
        if (k > 0) {
          const double clear = bk.ring_clearance(par[p], k - 1);
          if (clear > 0 && clear * clear > 4.0 * q.max_dist2(par[p])) break;
        }
        bk.for_ring(par[p], k, [&](int id) { if (id != p && q.v.size() >= 3) clip_closer_to(q, par[p], par[id], tol, scratch); });
      }
      const double a = q.v.size() >= 3 ? q.area() / total : 0.0;
      if (a >= 1e-12) row.emplace_back(p, a);
    }
    if (row.empty()) return bip::fail(nullptr, BIP_ERR_INVALID, "bip_sibson: beam %d has no natural neighbour", b);
    if ((int)row.size() > max_nn)
      return bip::fail(nullptr, BIP_ERR_INVALID, "bip_sibson: beam %d needs %zu neighbours > max_nn %d", b, row.size(), max_nn);
    std::sort(row.begin(), row.end());
    double s = 0;
    for (auto& e : row) s += e.second;
    for (size_t j = 0; j < row.size(); ++j) { oi[j] = row[j].first; ow[j] = (float)(row[j].second / s); }
  }
  return BIP_OK;
}

}  // extern "C"
