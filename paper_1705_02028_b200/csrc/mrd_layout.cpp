// mrd_layout.cpp -- host-side mesh-layout stage. See mrd_layout.h. No CUDA, no oracle code.
#include "mrd_layout.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <omp.h>

#ifdef MRD_LAYOUT_TIMING
#include <chrono>
#include <cstdio>
namespace {
struct PhaseTimer {
  std::chrono::steady_clock::time_point t0 = std::chrono::steady_clock::now();
  void mark(const char *what) {
    auto t1 = std::chrono::steady_clock::now();
    std::fprintf(stderr, "[layout] %-28s %7.3f s\n", what, std::chrono::duration<double>(t1 - t0).count());
    t0 = t1;
  }
};
}
#define MRD_PHASE(t, what) (t).mark(what)
#else
namespace { struct PhaseTimer {}; }
#define MRD_PHASE(t, what) (void)0
#endif

namespace {

inline double min_image(double d, double period) {
  // PAPER.md L584 ("periodic boundaries are handled by the mesh"), reading C19
  if (period > 0.0) {
    if (d > 0.5 * period) d -= period;
    else if (d < -0.5 * period) d += period;
  }
  return d;
}
inline int image_shift(double d, double period) {
  if (period > 0.0) {
    if (d > 0.5 * period) return -1;
    if (d < -0.5 * period) return 1;
  }
  return 0;
}

// spread the low 21 bits of v so that there is one zero bit between consecutive bits
inline uint64_t spread21(uint64_t v) {
  v &= 0x1FFFFFull;
  v = (v | (v << 16)) & 0x0000FFFF0000FFFFull;
  v = (v | (v << 8)) & 0x00FF00FF00FF00FFull;
  v = (v | (v << 4)) & 0x0F0F0F0F0F0F0F0Full;
  v = (v | (v << 2)) & 0x3333333333333333ull;
  v = (v | (v << 1)) & 0x5555555555555555ull;
  return v;
}
// Morton (Z-order) key of a point, 21 bits per axis (L669-L675)
inline uint64_t morton_key(double x, double y, const double lo[2], const double inv[2]) {
  const double q = 2097151.0;  // 2^21 - 1
  double fx = (x - lo[0]) * inv[0], fy = (y - lo[1]) * inv[1];
  fx = std::min(std::max(fx, 0.0), 1.0);
  fy = std::min(std::max(fy, 0.0), 1.0);
  return spread21((uint64_t)(fx * q)) | (spread21((uint64_t)(fy * q)) << 1);
}

// stable LSD radix sort of `idx` by 48-bit `key`, 8 bits a pass; passes whose digit is the same for every key are
// skipped.  Parallel: every thread counts the digits of its own contiguous chunk, the offsets are a prefix over
// (digit, thread), and every thread scatters its chunk in order -- stable, and the same result for any thread count.
void radix_sort(std::vector<uint64_t> &key, std::vector<int32_t> &idx) {
  const int64_t n = (int64_t)key.size();
  if (n < 2) return;
  uint64_t vary = 0;
  int unsorted = 0;
#pragma omp parallel for schedule(static) reduction(| : vary) reduction(max : unsorted)
  for (int64_t i = 0; i < n; ++i) {
    vary |= key[i] ^ key[0];
    if (i > 0 && key[i] < key[i - 1]) unsorted = 1;
  }
  // Input already in key order (a mesh numbered along the curve): nothing to do.  (It is also the one slow case of the
  // passes below: equal power-of-two bucket sizes put all 256 write streams of a thread into the same cache sets.)
  if (!unsorted) return;
  std::vector<uint64_t> key2(n);
  std::vector<int32_t> idx2(n);
  const int nth = std::max(1, omp_get_max_threads());
  std::vector<int64_t> hist((size_t)nth * 256);
  for (int pass = 0; pass < 6; ++pass) {
    const int sh = 8 * pass;
    if (((vary >> sh) & 0xFF) == 0) continue;  // all digits equal: nothing to do
    std::fill(hist.begin(), hist.end(), 0);
#pragma omp parallel num_threads(nth)
    {
      const int t = omp_get_thread_num();
      const int64_t i0 = n * t / nth, i1 = n * (t + 1) / nth;
      int64_t *h = &hist[(size_t)t * 256];
      for (int64_t i = i0; i < i1; ++i) h[(key[i] >> sh) & 0xFF]++;
#pragma omp barrier
#pragma omp single
      {
        int64_t run = 0;
        for (int d = 0; d < 256; ++d)
          for (int q = 0; q < nth; ++q) {
            const int64_t c = hist[(size_t)q * 256 + d];
            hist[(size_t)q * 256 + d] = run;
            run += c;
          }
      }
      for (int64_t i = i0; i < i1; ++i) {
        const int64_t d = h[(key[i] >> sh) & 0xFF]++;
        key2[d] = key[i];
        idx2[d] = idx[i];
      }
    }
    key.swap(key2);
    idx.swap(idx2);
  }
}

// per-vertex incidence lists from a flat list of references: off[v] .. off[v+1] in `ent`, every list ascending.
// Parallel: counts and fill positions by atomic increments, then every (short) list is sorted.
template <class Ref>  // Ref(e) -> vertex referenced by entry e, or -1 for none
void build_incidence(int64_t nv, int64_t ne, Ref ref, std::vector<int32_t> &off, std::vector<int32_t> &ent) {
  off.assign(nv + 1, 0);
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    const int64_t v = ref(e);
    if (v < 0) continue;
#pragma omp atomic
    off[v + 1]++;
  }
  for (int64_t i = 0; i < nv; ++i) off[i + 1] += off[i];
  ent.resize(off[nv]);
  std::vector<int32_t> cur(off.begin(), off.end() - 1);
#pragma omp parallel for schedule(static)
  for (int64_t e = 0; e < ne; ++e) {
    const int64_t v = ref(e);
    if (v < 0) continue;
    int32_t pos;
#pragma omp atomic capture
    pos = cur[v]++;
    ent[pos] = (int32_t)e;
  }
#pragma omp parallel for schedule(static, 4096)
  for (int64_t i = 0; i < nv; ++i) std::sort(ent.begin() + off[i], ent.begin() + off[i + 1]);
}

}  // namespace

namespace mrd_host {

static void build_tile_plan(mrd_layout &L, const std::vector<double> &xyi);

// frame of the Morton keys: the bounding box (the period where periodic), one common scale for both axes so that the
// curve's cells stay square
static void morton_frame(int64_t nv, const double *xy, const double period[2], double lo[2], double inv[2]) {
  double hi[2] = {xy[0], xy[1]};
  lo[0] = xy[0]; lo[1] = xy[1];
  for (int64_t i = 0; i < nv; ++i)
    for (int d = 0; d < 2; ++d) {
      lo[d] = std::min(lo[d], xy[2 * i + d]);
      hi[d] = std::max(hi[d], xy[2 * i + d]);
    }
  for (int d = 0; d < 2; ++d)
    if (period[d] > 0.0) { lo[d] = 0.0; hi[d] = period[d]; }
  double ext = std::max(hi[0] - lo[0], hi[1] - lo[1]);
  inv[0] = inv[1] = ext > 0 ? 1.0 / ext : 0.0;
}

void morton_order_vertices(int64_t nv, const double *xy, const double period[2], std::vector<int32_t> &perm) {
  double lo[2], inv[2];
  morton_frame(nv, xy, period, lo, inv);
  std::vector<uint64_t> key(nv);
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < nv; ++i) key[i] = morton_key(xy[2 * i], xy[2 * i + 1], lo, inv);
  perm.resize(nv);
  std::iota(perm.begin(), perm.end(), 0);
  radix_sort(key, perm);
}

// geometry of a CCW triangle v[0..2] (internal vertex ids, coordinates xyi), 2nd and 3rd vertex unwrapped relative to the first
// (reading C19): g[0..2] nx, g[3..5] ny of the unit inward normal of the edge opposite node i (eq. 35; reading C4),
// g[6..8] half edge lengths, g[9] |T|/3, g[10] longest edge, g[11] |T|
static inline void triangle_geometry(const int32_t *v, const double *xyi, const double period[2], double g[12]) {
  double x[3][2];
  x[0][0] = xyi[2 * v[0]]; x[0][1] = xyi[2 * v[0] + 1];
  for (int j = 1; j < 3; ++j)
    for (int d = 0; d < 2; ++d) x[j][d] = x[0][d] + min_image(xyi[2 * v[j] + d] - x[0][d], period[d]);
  double lm = 0.0;
  for (int i = 0; i < 3; ++i) {
    // edge opposite node i runs from node i+1 to node i+2 (CCW); inward normal = (-e_y, e_x)
    int a = (i + 1) % 3, b = (i + 2) % 3;
    double ex = x[b][0] - x[a][0], ey = x[b][1] - x[a][1];
    double l = std::sqrt(ex * ex + ey * ey);
    g[i] = -ey / l;
    g[3 + i] = ex / l;
    g[6 + i] = 0.5 * l;
    lm = std::max(lm, l);
  }
  g[10] = lm;
  g[11] = 0.5 * ((x[1][0] - x[0][0]) * (x[2][1] - x[0][1]) - (x[1][1] - x[0][1]) * (x[2][0] - x[0][0]));
  g[9] = g[11] / 3.0;
}

int layout_build(mrd_layout &L, const mrd_params *p, int64_t nv, const double *xy, int64_t nt,
                 const int32_t *tri, const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge,
                 std::string &err) {
  if (!p || !xy || !tri || nv < 3 || nt < 1) { err = "null or empty mesh"; return MRD_EINVAL; }
  if (nv > 0x7FFFFFF0ll || 3 * nt > 0x7FFFFFF0ll) { err = "mesh too large for 32-bit indices"; return MRD_EINVAL; }
  if (!(p->gamma > 1.0) || !(p->cfl > 0.0)) { err = "gamma must be > 1 and cfl > 0"; return MRD_EINVAL; }
  if (p->scheme < 0 || p->scheme > 5 || (p->time_order != 1 && p->time_order != 2)) { err = "bad scheme/time_order"; return MRD_EINVAL; }
  if (p->precision != MRD_FP64 && p->precision != MRD_FP32) { err = "bad precision"; return MRD_EINVAL; }
  if (p->lumping != 0 && p->lumping != 1) { err = "lumping must be 0 (global) or 1 (selective)"; return MRD_EINVAL; }
  if (p->period_x < 0.0 || p->period_y < 0.0) { err = "negative period"; return MRD_EINVAL; }
  if (p->domain_size < 0.0 || !(p->domain_size == p->domain_size)) { err = "negative domain_size"; return MRD_EINVAL; }
  if (ne < 0 || (ne > 0 && !wall_edge)) { err = "bad wall edge list"; return MRD_EINVAL; }
  if (p->tile != -1 && p->tile != 0 && p->tile != 64 && p->tile != 128 && p->tile != 256) { err = "tile must be -1, 0, 64, 128 or 256"; return MRD_EINVAL; }
  L.p = *p;
  L.nv = nv; L.nt = nt; L.ne = ne;
  const double period[2] = {p->period_x, p->period_y};

  {  // domain size L of the Bx sensor (eq. 56, reading C25): larger side of the bounding box, the period where periodic
    double lo[2] = {xy[0], xy[1]}, hi[2] = {xy[0], xy[1]};
    for (int64_t i = 0; i < nv; ++i)
      for (int d = 0; d < 2; ++d) {
        lo[d] = std::min(lo[d], xy[2 * i + d]);
        hi[d] = std::max(hi[d], xy[2 * i + d]);
      }
    const double sx = period[0] > 0.0 ? period[0] : hi[0] - lo[0], sy = period[1] > 0.0 ? period[1] : hi[1] - lo[1];
    L.domain_size = std::max(sx, sy);
    if (p->domain_size > 0.0) L.domain_size = p->domain_size;  // given by the caller: a part of a decomposition passes the WHOLE mesh's L
  }
  PhaseTimer pt;
  // ---- validation + orientation fix in USER numbering ------------------------------------------
  std::vector<int32_t> utri(tri, tri + 3 * nt);
  std::vector<uint8_t> uswap(nt, 0);
  int bad = 0;  // first kind of error met (any thread): 1 index, 2 degenerate, 3 zero area
#pragma omp parallel for schedule(static) reduction(max : bad)
  for (int64_t t = 0; t < nt; ++t) {
    int32_t *v = &utri[3 * t];
    if (v[0] < 0 || v[0] >= nv || v[1] < 0 || v[1] >= nv || v[2] < 0 || v[2] >= nv) { bad = std::max(bad, 3); continue; }
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) { bad = std::max(bad, 2); continue; }
    double x0 = xy[2 * v[0]], y0 = xy[2 * v[0] + 1];
    double ax = min_image(xy[2 * v[1]] - x0, period[0]), ay = min_image(xy[2 * v[1] + 1] - y0, period[1]);
    double bx = min_image(xy[2 * v[2]] - x0, period[0]), by = min_image(xy[2 * v[2] + 1] - y0, period[1]);
    double cross = ax * by - ay * bx;
    if (cross == 0.0 || !(cross == cross)) { bad = std::max(bad, 1); continue; }
    if (cross < 0.0) { std::swap(v[1], v[2]); uswap[t] = 1; }
  }
  if (bad == 3) { err = "triangle index out of range"; return MRD_EINVAL; }
  if (bad == 2) { err = "degenerate triangle"; return MRD_EINVAL; }
  if (bad == 1) { err = "zero-area triangle"; return MRD_EINVAL; }

  MRD_PHASE(pt, "validate");
  // ---- Morton renumbering (L669-L675) ------------------------------------------------------------
  L.vperm.resize(nv); L.vrank.resize(nv); L.tperm.resize(nt); L.trank.resize(nt);
  std::iota(L.vperm.begin(), L.vperm.end(), 0);
  std::iota(L.tperm.begin(), L.tperm.end(), 0);
  if (p->reorder) {
    double lo[2], inv[2];
    morton_frame(nv, xy, period, lo, inv);
    std::vector<uint64_t> key(nv);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < nv; ++i) key[i] = morton_key(xy[2 * i], xy[2 * i + 1], lo, inv);
    MRD_PHASE(pt, "  vertex keys");
    radix_sort(key, L.vperm);
    MRD_PHASE(pt, "  vertex sort");
    key.assign(nt, 0);
#pragma omp parallel for schedule(static)
    for (int64_t t = 0; t < nt; ++t) {
      const int32_t *v = &utri[3 * t];
      double x0 = xy[2 * v[0]], y0 = xy[2 * v[0] + 1];
      double cx = x0 + (min_image(xy[2 * v[1]] - x0, period[0]) + min_image(xy[2 * v[2]] - x0, period[0])) / 3.0;
      double cy = y0 + (min_image(xy[2 * v[1] + 1] - y0, period[1]) + min_image(xy[2 * v[2] + 1] - y0, period[1])) / 3.0;
      if (period[0] > 0.0) cx -= period[0] * std::floor(cx / period[0]);
      if (period[1] > 0.0) cy -= period[1] * std::floor(cy / period[1]);
      key[t] = morton_key(cx, cy, lo, inv);
    }
    MRD_PHASE(pt, "  triangle keys");
    radix_sort(key, L.tperm);
    MRD_PHASE(pt, "  triangle sort");
  }
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < nv; ++k) L.vrank[L.vperm[k]] = (int32_t)k;
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < nt; ++k) L.trank[L.tperm[k]] = (int32_t)k;

  MRD_PHASE(pt, "morton sort");
  // ---- internal connectivity, geometry (eq. 35), volumes (L441, C5) -------------------
  L.tri.resize(3 * nt); L.tswap.resize(nt);
  // per-triangle geometry arrays are only kept for the unfused kernels: the tile kernels take theirs from the geometry table
  // or from the slot coordinates, both built per tile from triangle_geometry() below (2.4 GB less at 4096^2)
  const bool keep_geom = p->tile < 0;
  if (keep_geom)
    for (int i = 0; i < 3; ++i) { L.nx[i].resize(nt); L.ny[i].resize(nt); L.hl[i].resize(nt); }
  L.area.resize(nt);
  if (keep_geom) L.lmax.resize(nt);
  std::vector<double> xyi(2 * nv);
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < nv; ++k) {
    xyi[2 * k] = xy[2 * (int64_t)L.vperm[k]];
    xyi[2 * k + 1] = xy[2 * (int64_t)L.vperm[k] + 1];
  }
#pragma omp parallel for schedule(static)
  for (int64_t k = 0; k < nt; ++k) {
    const int32_t *uv = &utri[3 * (int64_t)L.tperm[k]];
    int32_t *v = &L.tri[3 * k];
    for (int j = 0; j < 3; ++j) v[j] = L.vrank[uv[j]];
    L.tswap[k] = uswap[L.tperm[k]];
    double g[12];
    triangle_geometry(v, xyi.data(), period, g);
    L.area[k] = g[11];
    if (keep_geom) {
      for (int i = 0; i < 3; ++i) { L.nx[i][k] = g[i]; L.ny[i][k] = g[3 + i]; L.hl[i][k] = g[6 + i]; }
      L.lmax[k] = g[10];
    }
  }
  MRD_PHASE(pt, "geometry");
  // ---- vertex -> (triangle, node) incidence, ascending (replaces the paper's atomics, L734) -------
  build_incidence(nv, 3 * nt, [&](int64_t e) { return (int64_t)L.tri[e]; }, L.csr_off, L.csr_ent);
  // V_i = sum |T|/3 over the fan, in ascending triangle order (L441, reading C5)
  L.vol.assign(nv, 0.0);
  int orphan = 0;
#pragma omp parallel for schedule(static) reduction(max : orphan)
  for (int64_t i = 0; i < nv; ++i) {
    double a = 0.0;
    for (int32_t q = L.csr_off[i]; q < L.csr_off[i + 1]; ++q) a += L.area[L.csr_ent[q] / 3] / 3.0;
    L.vol[i] = a;
    if (L.csr_off[i + 1] == L.csr_off[i]) orphan = 1;
  }
  if (orphan) { err = "vertex without triangle"; return MRD_EINVAL; }

  MRD_PHASE(pt, "csr");
  // ---- frozen vertices (L582) ---------------------------------------------------------------------
  L.frozen.assign(nv, 0);
  L.nf = 0;
  if (vertex_flag)
    for (int64_t k = 0; k < nv; ++k) {
      L.frozen[k] = vertex_flag[L.vperm[k]];  // 1 = frozen (L582), 2 = halo vertex of a partition
      if (L.frozen[k] > 2) { err = "vertex_flag must be 0, 1 or 2"; return MRD_EINVAL; }
      L.nf += L.frozen[k] != 0;
    }

  // ---- reflecting-wall edges (L586-L602; outward normal, reading C15) ------------------------------
  L.wall_a.resize(ne); L.wall_b.resize(ne); L.wall_nx.resize(ne); L.wall_ny.resize(ne); L.wall_len.resize(ne);
  for (int64_t e = 0; e < ne; ++e) {
    int32_t ua = wall_edge[2 * e], ub = wall_edge[2 * e + 1];
    if (ua < 0 || ua >= nv || ub < 0 || ub >= nv || ua == ub) { err = "bad wall edge"; return MRD_EINVAL; }
    int32_t a = L.vrank[ua], b = L.vrank[ub];
    int found = 0;
    int64_t ft = -1;
    int fa = 0, fb = 0;
    for (int32_t q = L.csr_off[a]; q < L.csr_off[a + 1]; ++q) {
      int64_t t = L.csr_ent[q] / 3;
      for (int j = 0; j < 3; ++j)
        if (L.tri[3 * t + j] == b) { ++found; ft = t; fa = L.csr_ent[q] % 3; fb = j; }
    }
    if (found != 1) { err = "wall edge must belong to exactly one triangle"; return MRD_EINVAL; }
    int fc = 3 - fa - fb;
    const int32_t *v = &L.tri[3 * ft];
    double x[3][2];
    x[0][0] = xyi[2 * v[0]]; x[0][1] = xyi[2 * v[0] + 1];
    for (int j = 1; j < 3; ++j)
      for (int d = 0; d < 2; ++d) x[j][d] = x[0][d] + min_image(xyi[2 * v[j] + d] - x[0][d], period[d]);
    double ex = x[fb][0] - x[fa][0], ey = x[fb][1] - x[fa][1];
    double len = std::sqrt(ex * ex + ey * ey);
    double nx = ey / len, ny = -ex / len;
    double mx = 0.5 * (x[fa][0] + x[fb][0]), my = 0.5 * (x[fa][1] + x[fb][1]);
    if (nx * (x[fc][0] - mx) + ny * (x[fc][1] - my) > 0.0) { nx = -nx; ny = -ny; }  // point away from the third vertex
    L.wall_a[e] = a; L.wall_b[e] = b; L.wall_nx[e] = nx; L.wall_ny[e] = ny; L.wall_len[e] = len;
  }
  {
    // wall vertex -> (edge, side) lists, ascending
    std::vector<std::pair<int32_t, int32_t>> inc;
    inc.reserve(2 * ne);
    for (int64_t e = 0; e < ne; ++e) {
      inc.emplace_back(L.wall_a[e], (int32_t)(2 * e));
      inc.emplace_back(L.wall_b[e], (int32_t)(2 * e + 1));
    }
    std::sort(inc.begin(), inc.end());
    {  // the same edge given twice, in either orientation
      std::vector<std::pair<int32_t, int32_t>> keys(ne);
      for (int64_t e = 0; e < ne; ++e) keys[e] = {std::min(L.wall_a[e], L.wall_b[e]), std::max(L.wall_a[e], L.wall_b[e])};
      std::sort(keys.begin(), keys.end());
      for (int64_t e = 1; e < ne; ++e)
        if (keys[e] == keys[e - 1]) { err = "duplicate wall edge"; return MRD_EINVAL; }
    }
    L.wv_vertex.clear(); L.wv_off.assign(1, 0); L.wv_ent.clear();
    for (size_t q = 0; q < inc.size(); ++q) {
      if (q == 0 || inc[q].first != inc[q - 1].first) {
        if (q) L.wv_off.push_back((int32_t)L.wv_ent.size());
        L.wv_vertex.push_back(inc[q].first);
      }
      L.wv_ent.push_back(inc[q].second);
    }
    if (!inc.empty()) L.wv_off.push_back((int32_t)L.wv_ent.size());
  }

  MRD_PHASE(pt, "walls");
  L.tile = p->tile == 0 ? 256 : (p->tile < 0 ? 0 : p->tile);  // 0 = default tile, -1 = unfused kernels
  if (L.tile > 0) build_tile_plan(L, xyi);
  MRD_PHASE(pt, "tile plan total");
  return MRD_OK;
}

// ---------------------------------------------------------------------------------------------------
// Tile plan: tile b = internal triangles [b*tile, (b+1)*tile).  A "slot" is one (vertex, periodic image)
// pair used by the tile; every slot carries the vertex coordinates unwrapped into the tile's frame, so the
// fused kernel needs no minimum-image arithmetic, and receives one partial sum per stage.  See mrd_layout.h for the
// plan record.
// ---------------------------------------------------------------------------------------------------
namespace {
struct Hash128 {
  uint64_t a, b;
  bool operator<(const Hash128 &o) const { return a != o.a ? a < o.a : b < o.b; }
  bool operator==(const Hash128 &o) const { return a == o.a && b == o.b; }
};
inline Hash128 hash_bytes(const void *p, size_t n) {
  const unsigned char *c = static_cast<const unsigned char *>(p);
  uint64_t a = 1469598103934665603ull, b = 0x9E3779B97F4A7C15ull;
  for (size_t i = 0; i < n; ++i) {
    a = (a ^ c[i]) * 1099511628211ull;                                  // FNV-1a
    b = (b + c[i] + 1) * 0xD6E8FEB86659FD93ull; b ^= b >> 29;           // an independent multiplicative mix
  }
  return {a, b};
}
}  // namespace

static void build_tile_plan(mrd_layout &L, const std::vector<double> &xyi) {
  PhaseTimer pt;
  const int64_t nt = L.nt, nv = L.nv;
  const int T = L.tile;
  const double period[2] = {L.p.period_x, L.p.period_y};
  const int64_t ntile = (nt + T - 1) / T;
  L.ntile = ntile;
  // (vertex, periodic image) key of node j of triangle t in the frame of the tile whose anchor vertex sits at (ax, ay)
  auto node_key = [&](int64_t t, int j, double ax, double ay) -> int64_t {
    const int32_t *v = &L.tri[3 * t];
    const double x0 = xyi[2 * v[0]], y0 = xyi[2 * v[0] + 1];
    int sx = image_shift(x0 - ax, period[0]), sy = image_shift(y0 - ay, period[1]);
    if (j) {
      sx += image_shift(xyi[2 * v[j]] - x0, period[0]);
      sy += image_shift(xyi[2 * v[j] + 1] - y0, period[1]);
    }
    return (int64_t)v[j] * 25 + (sx + 2) * 5 + (sy + 2);
  };
  // the node keys of tile b (nk[3 (t - t0) + j]) and its sorted unique keys uk[0 .. return value); recomputed by every
  // pass instead of being kept: 3 T keys per tile are cheaper to rebuild than to hold for 10^5 tiles
  auto tile_keys = [&](int64_t b, int64_t *nk, int64_t *uk) -> int {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int32_t anchor = L.tri[3 * t0];
    const double ax = xyi[2 * anchor], ay = xyi[2 * anchor + 1];
    int n = 0;
    for (int64_t t = t0; t < t1; ++t)
      for (int j = 0; j < 3; ++j) nk[n++] = node_key(t, j, ax, ay);
    std::copy(nk, nk + n, uk);
    std::sort(uk, uk + n);
    return (int)(std::unique(uk, uk + n) - uk);
  };
  // pass 1 (parallel): slots per tile
  std::vector<int32_t> nslot_of(ntile + 1, 0);
#pragma omp parallel
  {
    std::vector<int64_t> nk(3 * T), uk(3 * T);
#pragma omp for schedule(dynamic, 256)
    for (int64_t b = 0; b < ntile; ++b) nslot_of[b + 1] = (tile_keys(b, nk.data(), uk.data()) + 3) / 4 * 4;  // padded: 16-byte granularity of the bulk copies
  }
  L.tile_slot_off.assign(ntile + 1, 0);
  for (int64_t b = 0; b < ntile; ++b) L.tile_slot_off[b + 1] = L.tile_slot_off[b] + nslot_of[b + 1];
  const int64_t nslot = L.tile_slot_off[ntile];
  L.nslot = nslot;
  L.slot_vertex.assign(nslot, -1);  // -1 = padding slot
  L.slot_xy.assign(2 * nslot, 0.0);
  int32_t maxs = 0;
  for (int64_t b = 0; b < ntile; ++b) maxs = std::max(maxs, nslot_of[b + 1]);
  L.maxslots = maxs;
  L.offn = (maxs + 1 + 7) / 8 * 8;
  MRD_PHASE(pt, "plan pass1");
  // pass 2 (parallel): slot records, and per tile the number of incidence batches
  // (a slot's incidences are stored 4 to a batch, the last batch padded with the sentinel entry 3 T)
  std::vector<int32_t> nbatch_of(ntile, 0);
#pragma omp parallel
  {
    std::vector<int64_t> nk(3 * T), uk(3 * T);
    std::vector<int> deg(3 * T);
#pragma omp for schedule(dynamic, 256)
    for (int64_t b = 0; b < ntile; ++b) {
      const int64_t t0 = b * T;
      const int32_t s0 = L.tile_slot_off[b];
      const int32_t anchor = L.tri[3 * t0];
      const double ax = xyi[2 * anchor], ay = xyi[2 * anchor + 1];
      const int nsl = tile_keys(b, nk.data(), uk.data());
      const int nn = 3 * (int)(std::min(nt, t0 + T) - t0);
      for (int q = 0; q < nsl; ++q) {
        const int32_t v = (int32_t)(uk[q] / 25);
        const int r = (int)(uk[q] % 25);
        const int sx = r / 5 - 2, sy = r % 5 - 2;
        L.slot_vertex[s0 + q] = v;
        // relative to the tile's anchor vertex: keeps fp32 coordinates accurate to ulp(tile size), not ulp(domain)
        L.slot_xy[2 * (s0 + q)] = (xyi[2 * v] + sx * period[0]) - ax;
        L.slot_xy[2 * (s0 + q) + 1] = (xyi[2 * v + 1] + sy * period[1]) - ay;
        deg[q] = 0;
      }
      for (int k = 0; k < nn; ++k) deg[std::lower_bound(uk.data(), uk.data() + nsl, nk[k]) - uk.data()]++;
      int nb = 0;
      for (int q = 0; q < nsl; ++q) nb += (deg[q] + 3) / 4;
      nbatch_of[b] = nb;
    }
  }
  int32_t maxb = 0;
  for (int64_t b = 0; b < ntile; ++b) maxb = std::max(maxb, nbatch_of[b]);
  L.maxbatch = (maxb + 1) / 2 * 2;  // 16-byte granularity
  L.plan_stride = 4 * T + L.offn + 4 * L.maxbatch;

  MRD_PHASE(pt, "plan pass2");
  // geometry table: per tile the DISTINCT (bitwise) geometry records of its triangles; the record index goes into the
  // 4th entry of the triangle's plan entry
  std::vector<std::vector<double>> recs(ntile);
  std::vector<int32_t> nshape_of(ntile + 1, 0);
  std::vector<uint16_t> shape_id((size_t)ntile * T, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < ntile; ++b) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int n = (int)(t1 - t0);
    double g[256][12];
    int order[256];
    for (int q = 0; q < n; ++q) {
      triangle_geometry(&L.tri[3 * (t0 + q)], xyi.data(), period, g[q]);
      g[q][11] = 0.0;
      order[q] = q;
    }
    std::sort(order, order + n, [&](int a, int c) { return std::memcmp(g[a], g[c], sizeof g[0]) < 0; });
    std::vector<double> &out = recs[b];
    int ns = 0;
    for (int q = 0; q < n; ++q) {
      if (q == 0 || std::memcmp(g[order[q]], g[order[q - 1]], sizeof g[0]) != 0) {
        out.insert(out.end(), g[order[q]], g[order[q]] + 12);
        ++ns;
      }
      shape_id[(size_t)b * T + order[q]] = (uint16_t)(ns - 1);
    }
    nshape_of[b + 1] = ns;
  }
  L.tile_shape_off.assign(ntile + 1, 0);
  int32_t maxsh = 0;
  for (int64_t b = 0; b < ntile; ++b) {
    L.tile_shape_off[b + 1] = L.tile_shape_off[b] + nshape_of[b + 1];
    maxsh = std::max(maxsh, nshape_of[b + 1]);
  }
  const int64_t nshape = L.tile_shape_off[ntile];
  // it pays when the table is much smaller than per-triangle geometry: 96 B per record against ~60 fp64
  // instructions per triangle and stage
  L.geom_table = nshape * 8 <= nt;
  L.maxshapes = maxsh;
  if (L.geom_table) {
    L.shape_geom.resize((size_t)nshape * 12);
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < ntile; ++b)
      std::memcpy(&L.shape_geom[(size_t)L.tile_shape_off[b] * 12], recs[b].data(), sizeof(double) * recs[b].size());
  }
  recs.clear();
  recs.shrink_to_fit();

  MRD_PHASE(pt, "plan geomtable");
  // per-tile plan record (one bulk copy): [T x 4] local slots of the three nodes + geometry record, [offn] first
  // incidence batch of each slot, [4 maxbatch] incidence entries node * T + local triangle, 4 to a batch, ascending.
  // Tiles with the same record share it (uniform meshes: a handful of distinct records): pass A hashes every tile's
  // record, pass B writes one copy per distinct hash.
  auto make_record = [&](int64_t b, uint16_t *rec, int64_t *nk, int64_t *uk, int *loc, int *off) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int nsl = tile_keys(b, nk, uk), nn = 3 * (int)(t1 - t0);
    std::fill(rec, rec + L.plan_stride, (uint16_t)0);
    uint16_t *boff = rec + 4 * T, *ent = rec + 4 * T + L.offn;
    for (int q = 0; q <= nsl; ++q) off[q] = 0;
    for (int k = 0; k < nn; ++k) {
      loc[k] = (int)(std::lower_bound(uk, uk + nsl, nk[k]) - uk);
      rec[4 * (k / 3) + (k % 3)] = (uint16_t)loc[k];
      off[loc[k] + 1]++;
    }
    for (int64_t t = t0; t < t1; ++t) rec[4 * (t - t0) + 3] = L.geom_table ? shape_id[(size_t)b * T + (t - t0)] : (uint16_t)0;
    int nb = 0;
    for (int q = 0; q < nsl; ++q) {  // off[q]: first ENTRY of slot q (batches of 4), boff[q]: its first batch
      const int d = off[q + 1];
      off[q + 1] = 4 * nb;             // (becomes the running fill position of slot q below)
      boff[q] = (uint16_t)nb;
      nb += (d + 3) / 4;
    }
    for (int q = nsl; q < L.offn; ++q) boff[q] = (uint16_t)nb;
    for (int k = 0; k < 4 * nb; ++k) ent[k] = (uint16_t)(3 * T);  // sentinel: reads a zero residual
    // (k runs over (triangle, node) in ascending order, so every slot's entries come out in the fixed summation order)
    for (int k = 0; k < nn; ++k) ent[off[loc[k] + 1]++] = (uint16_t)((k % 3) * T + k / 3);
  };
  std::vector<Hash128> hashes(ntile);
#pragma omp parallel
  {
    std::vector<uint16_t> rec(L.plan_stride);
    std::vector<int64_t> nk(3 * T), uk(3 * T);
    std::vector<int> loc(3 * T), off(3 * T + 2);
#pragma omp for schedule(dynamic, 256)
    for (int64_t b = 0; b < ntile; ++b) {
      make_record(b, rec.data(), nk.data(), uk.data(), loc.data(), off.data());
      hashes[b] = hash_bytes(rec.data(), sizeof(uint16_t) * L.plan_stride);
    }
  }
  std::vector<int64_t> order(ntile);
  std::iota(order.begin(), order.end(), 0);
  std::sort(order.begin(), order.end(), [&](int64_t a, int64_t c) { return hashes[a] < hashes[c] || (hashes[a] == hashes[c] && a < c); });
  L.tile_plan_idx.assign(ntile, 0);
  std::vector<int64_t> reps;
  for (int64_t q = 0; q < ntile; ++q) {
    if (q == 0 || !(hashes[order[q]] == hashes[order[q - 1]])) reps.push_back(order[q]);
    L.tile_plan_idx[order[q]] = (int32_t)(reps.size() - 1);
  }
  L.nplan = (int64_t)reps.size();
  L.tile_plan.assign((size_t)L.nplan * L.plan_stride, 0);
#pragma omp parallel
  {
    std::vector<int64_t> nk(3 * T), uk(3 * T);
    std::vector<int> loc(3 * T), off(3 * T + 2);
#pragma omp for schedule(dynamic, 64)
    for (int64_t q = 0; q < L.nplan; ++q) make_record(reps[q], &L.tile_plan[(size_t)q * L.plan_stride], nk.data(), uk.data(), loc.data(), off.data());
  }

  MRD_PHASE(pt, "plan records");
  // vertex -> slots, ascending (slots are tile-major, so this is ascending triangle order)
  build_incidence(nv, nslot, [&](int64_t sl) { return (int64_t)L.slot_vertex[sl]; }, L.vslot_off, L.vslot_ent);
  MRD_PHASE(pt, "plan vslot");
}

}  // namespace mrd_host
