// mrd_layout.cpp -- host-side mesh-layout stage. See mrd_layout.h. No CUDA, no oracle code.
#include "mrd_layout.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>

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

// stable LSD radix sort of `idx` by 48-bit `key`
void radix_sort(std::vector<uint64_t> &key, std::vector<int32_t> &idx) {
  const size_t n = key.size();
  std::vector<uint64_t> key2(n);
  std::vector<int32_t> idx2(n);
  for (int pass = 0; pass < 6; ++pass) {
    const int sh = 8 * pass;
    size_t cnt[257] = {0};
    for (size_t i = 0; i < n; ++i) cnt[((key[i] >> sh) & 0xFF) + 1]++;
    if (cnt[((key[0] >> sh) & 0xFF) + 1] == n) continue;  // all digits equal: nothing to do
    for (int b = 0; b < 256; ++b) cnt[b + 1] += cnt[b];
    for (size_t i = 0; i < n; ++i) {
      size_t d = cnt[(key[i] >> sh) & 0xFF]++;
      key2[d] = key[i];
      idx2[d] = idx[i];
    }
    key.swap(key2);
    idx.swap(idx2);
  }
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
  if (p->tile != -1 && p->tile != 0 && p->tile != 64 && p->tile != 128) { err = "tile must be -1, 0, 64 or 128"; return MRD_EINVAL; }
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
  // ---- validation + orientation fix in USER numbering ------------------------------------------
  std::vector<int32_t> utri(tri, tri + 3 * nt);
  std::vector<uint8_t> uswap(nt, 0);
  std::vector<int32_t> deg(nv, 0);
  for (int64_t t = 0; t < nt; ++t) {
    int32_t *v = &utri[3 * t];
    for (int j = 0; j < 3; ++j)
      if (v[j] < 0 || v[j] >= nv) { err = "triangle index out of range"; return MRD_EINVAL; }
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) { err = "degenerate triangle"; return MRD_EINVAL; }
    double x0 = xy[2 * v[0]], y0 = xy[2 * v[0] + 1];
    double ax = min_image(xy[2 * v[1]] - x0, period[0]), ay = min_image(xy[2 * v[1] + 1] - y0, period[1]);
    double bx = min_image(xy[2 * v[2]] - x0, period[0]), by = min_image(xy[2 * v[2] + 1] - y0, period[1]);
    double cross = ax * by - ay * bx;
    if (cross == 0.0 || !(cross == cross)) { err = "zero-area triangle"; return MRD_EINVAL; }
    if (cross < 0.0) { std::swap(v[1], v[2]); uswap[t] = 1; }
    for (int j = 0; j < 3; ++j) deg[v[j]]++;
  }
  for (int64_t i = 0; i < nv; ++i)
    if (deg[i] == 0) { err = "vertex without triangle"; return MRD_EINVAL; }

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
    radix_sort(key, L.vperm);
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
    radix_sort(key, L.tperm);
  }
  for (int64_t k = 0; k < nv; ++k) L.vrank[L.vperm[k]] = (int32_t)k;
  for (int64_t k = 0; k < nt; ++k) L.trank[L.tperm[k]] = (int32_t)k;

  // ---- internal connectivity, geometry (eq. 35), volumes (L441, C5) -------------------
  L.tri.resize(3 * nt); L.tswap.resize(nt);
  for (int i = 0; i < 3; ++i) { L.nx[i].resize(nt); L.ny[i].resize(nt); L.hl[i].resize(nt); }
  L.area.resize(nt); L.lmax.resize(nt);
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
      L.nx[i][k] = -ey / l;
      L.ny[i][k] = ex / l;
      L.hl[i][k] = 0.5 * l;
      lm = std::max(lm, l);
    }
    L.lmax[k] = lm;
    L.area[k] = 0.5 * ((x[1][0] - x[0][0]) * (x[2][1] - x[0][1]) - (x[1][1] - x[0][1]) * (x[2][0] - x[0][0]));
  }
  L.vol.assign(nv, 0.0);
  for (int64_t k = 0; k < nt; ++k)
    for (int j = 0; j < 3; ++j) L.vol[L.tri[3 * k + j]] += L.area[k] / 3.0;

  // ---- vertex -> (triangle, node) incidence, ascending (replaces the paper's atomics, L734) -------
  L.csr_off.assign(nv + 1, 0);
  for (int64_t e = 0; e < 3 * nt; ++e) L.csr_off[L.tri[e] + 1]++;
  for (int64_t i = 0; i < nv; ++i) L.csr_off[i + 1] += L.csr_off[i];
  L.csr_ent.resize(3 * nt);
  {
    std::vector<int32_t> cur(L.csr_off.begin(), L.csr_off.end() - 1);
    for (int64_t e = 0; e < 3 * nt; ++e) L.csr_ent[cur[L.tri[e]]++] = (int32_t)e;
  }

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

  L.tile = p->tile == 0 ? 128 : (p->tile < 0 ? 0 : p->tile);  // 0 = default tile, -1 = unfused kernels
  if (L.tile > 0) build_tile_plan(L, xyi);
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
  const int64_t nt = L.nt, nv = L.nv;
  const int T = L.tile;
  const double period[2] = {L.p.period_x, L.p.period_y};
  const int64_t ntile = (nt + T - 1) / T;
  L.ntile = ntile;
  // pass 1 (parallel): per tile the sorted unique (vertex, image) keys
  std::vector<std::vector<int64_t>> keys(ntile);
  std::vector<int32_t> nslot_of(ntile + 1, 0);
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
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < ntile; ++b) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int32_t anchor = L.tri[3 * t0];
    const double ax = xyi[2 * anchor], ay = xyi[2 * anchor + 1];
    std::vector<int64_t> &uk = keys[b];
    uk.reserve(3 * (t1 - t0));
    for (int64_t t = t0; t < t1; ++t)
      for (int j = 0; j < 3; ++j) uk.push_back(node_key(t, j, ax, ay));
    std::sort(uk.begin(), uk.end());
    uk.erase(std::unique(uk.begin(), uk.end()), uk.end());
    nslot_of[b + 1] = (int32_t)((uk.size() + 3) / 4 * 4);  // padded: 16-byte granularity of the bulk copies
  }
  // slots per vertex (a vertex with one slot has its whole fan in that tile)
  std::vector<int32_t> vcount(nv, 0);
  for (int64_t b = 0; b < ntile; ++b)
    for (int64_t key : keys[b]) vcount[key / 25]++;
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
  // pass 2 (parallel): slot records, and per tile the number of incidence batches
  // (a slot's incidences are stored 4 to a batch, the last batch padded with the sentinel entry 3 T)
  std::vector<int32_t> nbatch_of(ntile, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < ntile; ++b) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int32_t s0 = L.tile_slot_off[b];
    const int32_t anchor = L.tri[3 * t0];
    const double ax = xyi[2 * anchor], ay = xyi[2 * anchor + 1];
    const std::vector<int64_t> &uk = keys[b];
    std::vector<int> deg(uk.size(), 0);
    for (size_t q = 0; q < uk.size(); ++q) {
      const int32_t v = (int32_t)(uk[q] / 25);
      const int r = (int)(uk[q] % 25);
      const int sx = r / 5 - 2, sy = r % 5 - 2;
      L.slot_vertex[s0 + q] = v;
      // relative to the tile's anchor vertex: keeps fp32 coordinates accurate to ulp(tile size), not ulp(domain)
      L.slot_xy[2 * (s0 + q)] = (xyi[2 * v] + sx * period[0]) - ax;
      L.slot_xy[2 * (s0 + q) + 1] = (xyi[2 * v + 1] + sy * period[1]) - ay;
    }
    for (int64_t t = t0; t < t1; ++t)
      for (int j = 0; j < 3; ++j) deg[std::lower_bound(uk.begin(), uk.end(), node_key(t, j, ax, ay)) - uk.begin()]++;
    int nb = 0;
    for (int d : deg) nb += (d + 3) / 4;
    nbatch_of[b] = nb;
  }
  int32_t maxb = 0;
  for (int64_t b = 0; b < ntile; ++b) maxb = std::max(maxb, nbatch_of[b]);
  L.maxbatch = (maxb + 1) / 2 * 2;  // 16-byte granularity
  L.plan_stride = 4 * T + L.offn + 4 * L.maxbatch;

  // geometry table: per tile the DISTINCT (bitwise) geometry records of its triangles; the record index goes into the
  // 4th entry of the triangle's plan entry
  std::vector<std::vector<double>> recs(ntile);
  std::vector<int32_t> nshape_of(ntile + 1, 0);
  std::vector<uint16_t> shape_id((size_t)ntile * T, 0);
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t b = 0; b < ntile; ++b) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int n = (int)(t1 - t0);
    double g[128][12];
    int order[128];
    for (int q = 0; q < n; ++q) {
      const int64_t t = t0 + q;
      for (int i = 0; i < 3; ++i) { g[q][i] = L.nx[i][t]; g[q][3 + i] = L.ny[i][t]; g[q][6 + i] = L.hl[i][t]; }
      g[q][9] = L.area[t] / 3.0;
      g[q][10] = L.lmax[t];
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

  // per-tile plan record (one bulk copy): [T x 4] local slots of the three nodes + geometry record, [offn] first
  // incidence batch of each slot, [4 maxbatch] incidence entries node * T + local triangle, 4 to a batch, ascending.
  // Tiles with the same record share it (uniform meshes: a handful of distinct records): pass A hashes every tile's
  // record, pass B writes one copy per distinct hash.
  auto make_record = [&](int64_t b, uint16_t *rec) {
    const int64_t t0 = b * T, t1 = std::min(nt, t0 + T);
    const int32_t s0 = L.tile_slot_off[b];
    const int32_t anchor = L.tri[3 * t0];
    const double ax = xyi[2 * anchor], ay = xyi[2 * anchor + 1];
    const std::vector<int64_t> &uk = keys[b];
    const int nsl = (int)uk.size(), ns_pad = L.tile_slot_off[b + 1] - s0;
    std::fill(rec, rec + L.plan_stride, (uint16_t)0);
    std::vector<std::vector<uint16_t>> inc(nsl);
    for (int64_t t = t0; t < t1; ++t)
      for (int j = 0; j < 3; ++j) {
        const int loc = (int)(std::lower_bound(uk.begin(), uk.end(), node_key(t, j, ax, ay)) - uk.begin());
        rec[4 * (t - t0) + j] = (uint16_t)loc;
        inc[loc].push_back((uint16_t)(j * T + (t - t0)));
      }
    for (int64_t t = t0; t < t1; ++t) rec[4 * (t - t0) + 3] = L.geom_table ? shape_id[(size_t)b * T + (t - t0)] : (uint16_t)0;
    uint16_t *boff = rec + 4 * T, *ent = rec + 4 * T + L.offn;
    int nb = 0;
    for (int q = 0; q < L.offn; ++q) {
      boff[q] = (uint16_t)nb;
      if (q < nsl) {
        std::vector<uint16_t> &e = inc[q];
        std::sort(e.begin(), e.end(), [&](uint16_t a, uint16_t c) {  // ascending (local triangle, node): the fixed summation order
          return (a % T) != (c % T) ? (a % T) < (c % T) : a < c;
        });
        for (size_t k = 0; k < (e.size() + 3) / 4 * 4; ++k) ent[4 * nb + k] = k < e.size() ? e[k] : (uint16_t)(3 * T);
        nb += (int)((e.size() + 3) / 4);
      }
    }
    (void)ns_pad;
  };
  std::vector<Hash128> hashes(ntile);
#pragma omp parallel
  {
    std::vector<uint16_t> rec(L.plan_stride);
#pragma omp for schedule(dynamic, 64)
    for (int64_t b = 0; b < ntile; ++b) {
      make_record(b, rec.data());
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
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t q = 0; q < L.nplan; ++q) make_record(reps[q], &L.tile_plan[(size_t)q * L.plan_stride]);

  // vertex -> slots, ascending (slots are tile-major, so this is ascending triangle order)
  L.vslot_off.assign(nv + 1, 0);
  for (int64_t i = 0; i < nv; ++i) L.vslot_off[i + 1] = L.vslot_off[i] + vcount[i];
  L.vslot_ent.resize(L.vslot_off[nv]);
  {
    std::vector<int32_t> cur(L.vslot_off.begin(), L.vslot_off.end() - 1);
    for (int64_t s = 0; s < nslot; ++s)
      if (L.slot_vertex[s] >= 0) L.vslot_ent[cur[L.slot_vertex[s]]++] = (int32_t)s;
  }
}

}  // namespace mrd_host
