// mrd_partition.cpp -- host-side domain decomposition for several GPUs. See include/mrd.h.
// Owner-computes over contiguous ranges of the vertices' Morton order (PAPER.md L669-L675 gives the curve; the
// decomposition itself is this library's: the paper ran on one device). Plain C++17, no CUDA, no oracle code.
#include <algorithm>
#include <cstring>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "mrd_layout.h"

namespace mrd_host {

int partition_build(mrd_partition &P, int64_t nv, const double *xy, int64_t nt, const int32_t *tri,
                    const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge, double period_x, double period_y,
                    int32_t n_part, int32_t part, const int32_t *owner_in, std::string &err) {
  if (!xy || !tri || nv < 3 || nt < 1) { err = "null or empty mesh"; return MRD_EINVAL; }
  if (nv > 0x7FFFFFF0ll || 3 * nt > 0x7FFFFFF0ll) { err = "mesh too large for 32-bit indices"; return MRD_EINVAL; }
  if (n_part < 1 || part < 0 || part >= n_part) { err = "bad n_part / part"; return MRD_EINVAL; }
  if (n_part > nv) { err = "more parts than vertices"; return MRD_EINVAL; }
  if (period_x < 0.0 || period_y < 0.0) { err = "negative period"; return MRD_EINVAL; }
  if (ne < 0 || (ne > 0 && !wall_edge)) { err = "bad wall edge list"; return MRD_EINVAL; }
  for (int64_t e = 0; e < 3 * nt; ++e)
    if (tri[e] < 0 || tri[e] >= nv) { err = "triangle index out of range"; return MRD_EINVAL; }
  if (vertex_flag)
    for (int64_t i = 0; i < nv; ++i)
      if (vertex_flag[i] > 1) { err = "vertex_flag of the global mesh must be 0 or 1"; return MRD_EINVAL; }
  for (int64_t e = 0; e < 2 * ne; ++e)
    if (wall_edge[e] < 0 || wall_edge[e] >= nv) { err = "bad wall edge"; return MRD_EINVAL; }
  if (owner_in)
    for (int64_t i = 0; i < nv; ++i)
      if (owner_in[i] < 0 || owner_in[i] >= n_part) { err = "owner out of range"; return MRD_EINVAL; }
  P.nv_g = nv; P.nt_g = nt; P.n_part = n_part; P.part = part;
  {  // L of the Bx sensor (eq. 56, reading C25) of the WHOLE mesh: every part must use the same value
    double lo[2] = {xy[0], xy[1]}, hi[2] = {xy[0], xy[1]};
    for (int64_t i = 0; i < nv; ++i)
      for (int d = 0; d < 2; ++d) {
        lo[d] = std::min(lo[d], xy[2 * i + d]);
        hi[d] = std::max(hi[d], xy[2 * i + d]);
      }
    P.domain_size = std::max(period_x > 0.0 ? period_x : hi[0] - lo[0], period_y > 0.0 ? period_y : hi[1] - lo[1]);
  }

  // owners: given by the caller, or part q owns positions [q nv / P, (q+1) nv / P) of the Morton order
  if (owner_in) {
    P.owner.assign(owner_in, owner_in + nv);
  } else {
    const double period[2] = {period_x, period_y};
    std::vector<int32_t> perm;
    morton_order_vertices(nv, xy, period, perm);
    P.owner.resize(nv);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < nv; ++k) P.owner[perm[k]] = (int32_t)((k * (int64_t)n_part) / nv);
  }
  const int32_t *own = P.owner.data();

  // local triangles and vertices
  std::vector<uint8_t> mark(nv, 0);  // 1 owned, 2 halo
  for (int64_t t = 0; t < nt; ++t) {
    const int32_t *v = &tri[3 * t];
    if (own[v[0]] == part || own[v[1]] == part || own[v[2]] == part) {
      P.tri_global.push_back((int32_t)t);
      for (int j = 0; j < 3; ++j) mark[v[j]] = own[v[j]] == part ? 1 : 2;
    }
  }
  for (int64_t i = 0; i < nv; ++i)
    if (own[i] == part && !mark[i]) { err = "vertex without triangle"; return MRD_EINVAL; }
  std::vector<int32_t> lid(nv, -1);
  for (int pass = 1; pass <= 2; ++pass)
    for (int64_t i = 0; i < nv; ++i)
      if (mark[i] == pass) {
        lid[i] = (int32_t)P.vertex_global.size();
        P.vertex_global.push_back((int32_t)i);
      }
  P.n_owned = 0;
  for (int64_t i = 0; i < nv; ++i) P.n_owned += mark[i] == 1;
  if (P.n_owned == 0) { err = "part without vertices"; return MRD_EINVAL; }
  const int64_t nlv = (int64_t)P.vertex_global.size(), nlt = (int64_t)P.tri_global.size();
  P.xy.resize(2 * nlv); P.flag.resize(nlv);
  for (int64_t k = 0; k < nlv; ++k) {
    const int64_t g = P.vertex_global[k];
    P.xy[2 * k] = xy[2 * g];
    P.xy[2 * k + 1] = xy[2 * g + 1];
    P.flag[k] = mark[g] == 2 ? 2 : (vertex_flag ? vertex_flag[g] : 0);
  }
  P.tri.resize(3 * nlt);
  for (int64_t k = 0; k < nlt; ++k)
    for (int j = 0; j < 3; ++j) P.tri[3 * k + j] = lid[tri[3 * (int64_t)P.tri_global[k] + j]];
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t a = wall_edge[2 * e], b = wall_edge[2 * e + 1];
    if (own[a] == part || own[b] == part) {
      // its one triangle holds the owned end, hence is local, hence both ends are
      if (lid[a] < 0 || lid[b] < 0) { err = "wall edge must belong to exactly one triangle"; return MRD_EINVAL; }
      P.wall.push_back(lid[a]);
      P.wall.push_back(lid[b]);
    }
  }

  // exchange lists: (neighbour, global vertex) pairs, sorted and made unique
  std::vector<std::pair<int32_t, int32_t>> snd, rcv;
  for (int64_t k = 0; k < nlt; ++k) {
    const int32_t *v = &tri[3 * (int64_t)P.tri_global[k]];
    for (int a = 0; a < 3; ++a) {
      if (own[v[a]] != part) { rcv.emplace_back(own[v[a]], v[a]); continue; }
      for (int b = 0; b < 3; ++b)
        if (own[v[b]] != part) snd.emplace_back(own[v[b]], v[a]);
    }
  }
  auto uniq = [](std::vector<std::pair<int32_t, int32_t>> &x) {
    std::sort(x.begin(), x.end());
    x.erase(std::unique(x.begin(), x.end()), x.end());
  };
  uniq(snd); uniq(rcv);
  for (auto &pr : snd) P.nbr.push_back(pr.first);
  for (auto &pr : rcv) P.nbr.push_back(pr.first);
  std::sort(P.nbr.begin(), P.nbr.end());
  P.nbr.erase(std::unique(P.nbr.begin(), P.nbr.end()), P.nbr.end());
  auto fill = [&](const std::vector<std::pair<int32_t, int32_t>> &x, std::vector<int32_t> &off, std::vector<int32_t> &idx) {
    off.assign(P.nbr.size() + 1, 0);
    idx.resize(x.size());
    size_t q = 0;
    for (size_t k = 0; k < P.nbr.size(); ++k) {
      while (q < x.size() && x[q].first == P.nbr[k]) { idx[q] = lid[x[q].second]; ++q; }
      off[k + 1] = (int32_t)q;
    }
  };
  fill(snd, P.send_off, P.send_idx);
  fill(rcv, P.recv_off, P.recv_idx);
  return MRD_OK;
}

// The same part assembled from LOCAL pieces only (no array of the whole mesh on any rank): the caller gives the vertices and
// triangles it knows -- at least every triangle incident to a vertex it owns, with all their vertices -- each with its global
// id and, per vertex, the owning part.  Output as partition_build, except `owner` (a whole-mesh array), which stays empty.
int partition_build_local(mrd_partition &P, int64_t nv_global, double domain_size, int64_t nlv, const int32_t *vertex_global,
                          const int32_t *owner, const double *xy, const uint8_t *vertex_flag, int64_t nlt, const int32_t *tri,
                          const int32_t *tri_global, int64_t ne, const int32_t *wall_edge, int32_t n_part, int32_t part,
                          std::string &err) {
  if (!vertex_global || !owner || !xy || !tri || !tri_global || nlv < 3 || nlt < 1) { err = "null or empty mesh"; return MRD_EINVAL; }
  if (nlv > 0x7FFFFFF0ll || 3 * nlt > 0x7FFFFFF0ll) { err = "part too large for 32-bit indices"; return MRD_EINVAL; }
  if (n_part < 1 || part < 0 || part >= n_part) { err = "bad n_part / part"; return MRD_EINVAL; }
  if (ne < 0 || (ne > 0 && !wall_edge)) { err = "bad wall edge list"; return MRD_EINVAL; }
  for (int64_t e = 0; e < 3 * nlt; ++e)
    if (tri[e] < 0 || tri[e] >= nlv) { err = "triangle index out of range"; return MRD_EINVAL; }
  for (int64_t i = 0; i < nlv; ++i) {
    if (owner[i] < 0 || owner[i] >= n_part) { err = "owner out of range"; return MRD_EINVAL; }
    if (vertex_global[i] < 0 || vertex_global[i] >= nv_global) { err = "global vertex id out of range"; return MRD_EINVAL; }
    if (vertex_flag && vertex_flag[i] > 1) { err = "vertex_flag of the global mesh must be 0 or 1"; return MRD_EINVAL; }
  }
  for (int64_t e = 0; e < 2 * ne; ++e)
    if (wall_edge[e] < 0 || wall_edge[e] >= nlv) { err = "bad wall edge"; return MRD_EINVAL; }
  P.nv_g = nv_global; P.nt_g = 0; P.n_part = n_part; P.part = part; P.domain_size = domain_size;
  // triangles with an owned vertex, ascending global id; the vertices they use
  std::vector<int64_t> keep;
  std::vector<uint8_t> mark(nlv, 0);  // 1 owned, 2 halo
  for (int64_t t = 0; t < nlt; ++t) {
    const int32_t *v = &tri[3 * t];
    if (owner[v[0]] == part || owner[v[1]] == part || owner[v[2]] == part) {
      keep.push_back(t);
      for (int j = 0; j < 3; ++j) mark[v[j]] = owner[v[j]] == part ? 1 : 2;
    }
  }
  std::sort(keep.begin(), keep.end(), [&](int64_t a, int64_t b) { return tri_global[a] < tri_global[b]; });
  for (size_t k = 1; k < keep.size(); ++k)
    if (tri_global[keep[k]] == tri_global[keep[k - 1]]) { err = "duplicate global triangle id"; return MRD_EINVAL; }
  for (int64_t i = 0; i < nlv; ++i)
    if (owner[i] == part && !mark[i]) { err = "vertex without triangle"; return MRD_EINVAL; }
  // local numbering: owned vertices in ascending global id, then halo vertices in ascending global id
  std::vector<int64_t> ord;
  for (int64_t i = 0; i < nlv; ++i)
    if (mark[i]) ord.push_back(i);
  std::sort(ord.begin(), ord.end(), [&](int64_t a, int64_t b) {
    return mark[a] != mark[b] ? mark[a] < mark[b] : vertex_global[a] < vertex_global[b];
  });
  for (size_t k = 1; k < ord.size(); ++k)
    if (vertex_global[ord[k]] == vertex_global[ord[k - 1]]) { err = "duplicate global vertex id"; return MRD_EINVAL; }
  std::vector<int32_t> lid(nlv, -1);
  P.n_owned = 0;
  const int64_t nv2 = (int64_t)ord.size();
  P.vertex_global.resize(nv2); P.xy.resize(2 * nv2); P.flag.resize(nv2);
  std::vector<int32_t> own2(nv2);
  for (int64_t k = 0; k < nv2; ++k) {
    const int64_t i = ord[k];
    lid[i] = (int32_t)k;
    P.vertex_global[k] = vertex_global[i];
    P.xy[2 * k] = xy[2 * i];
    P.xy[2 * k + 1] = xy[2 * i + 1];
    P.flag[k] = mark[i] == 2 ? 2 : (vertex_flag ? vertex_flag[i] : 0);
    own2[k] = owner[i];
    P.n_owned += mark[i] == 1;
  }
  if (P.n_owned == 0) { err = "part without vertices"; return MRD_EINVAL; }
  const int64_t nt2 = (int64_t)keep.size();
  P.tri.resize(3 * nt2); P.tri_global.resize(nt2);
  for (int64_t k = 0; k < nt2; ++k) {
    P.tri_global[k] = tri_global[keep[k]];
    for (int j = 0; j < 3; ++j) P.tri[3 * k + j] = lid[tri[3 * keep[k] + j]];
  }
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t a = wall_edge[2 * e], b = wall_edge[2 * e + 1];
    if (owner[a] == part || owner[b] == part) {
      if (lid[a] < 0 || lid[b] < 0) { err = "wall edge must belong to exactly one triangle"; return MRD_EINVAL; }
      P.wall.push_back(lid[a]);
      P.wall.push_back(lid[b]);
    }
  }
  // exchange lists: (neighbour, GLOBAL vertex id) pairs, sorted and made unique -- the rule of partition_build
  std::vector<std::pair<int32_t, int32_t>> snd, rcv;
  for (int64_t k = 0; k < nt2; ++k) {
    const int32_t *v = &P.tri[3 * k];
    for (int a = 0; a < 3; ++a) {
      if (own2[v[a]] != part) { rcv.emplace_back(own2[v[a]], P.vertex_global[v[a]]); continue; }
      for (int b = 0; b < 3; ++b)
        if (own2[v[b]] != part) snd.emplace_back(own2[v[b]], P.vertex_global[v[a]]);
    }
  }
  auto uniq = [](std::vector<std::pair<int32_t, int32_t>> &x) {
    std::sort(x.begin(), x.end());
    x.erase(std::unique(x.begin(), x.end()), x.end());
  };
  uniq(snd); uniq(rcv);
  for (auto &pr : snd) P.nbr.push_back(pr.first);
  for (auto &pr : rcv) P.nbr.push_back(pr.first);
  std::sort(P.nbr.begin(), P.nbr.end());
  P.nbr.erase(std::unique(P.nbr.begin(), P.nbr.end()), P.nbr.end());
  // global id -> local id of the (sorted) owned and halo groups by binary search
  auto local_of = [&](int32_t g) -> int32_t {
    auto b0 = P.vertex_global.begin(), b1 = b0 + P.n_owned, b2 = P.vertex_global.end();
    auto it = std::lower_bound(b0, b1, g);
    if (it != b1 && *it == g) return (int32_t)(it - b0);
    it = std::lower_bound(b1, b2, g);
    return (int32_t)(it - b0);
  };
  auto fill = [&](const std::vector<std::pair<int32_t, int32_t>> &x, std::vector<int32_t> &off, std::vector<int32_t> &idx) {
    off.assign(P.nbr.size() + 1, 0);
    idx.resize(x.size());
    size_t q = 0;
    for (size_t k = 0; k < P.nbr.size(); ++k) {
      while (q < x.size() && x[q].first == P.nbr[k]) { idx[q] = local_of(x[q].second); ++q; }
      off[k + 1] = (int32_t)q;
    }
  };
  fill(snd, P.send_off, P.send_idx);
  fill(rcv, P.recv_off, P.recv_idx);
  return MRD_OK;
}

// accessors behind mrd_partition_sizes / mrd_partition_get (the C-ABI wrappers live in mrd_api.cu)

int partition_sizes(const mrd_partition &P, int64_t n[8]) {
  n[0] = (int64_t)P.vertex_global.size();
  n[1] = P.n_owned;
  n[2] = (int64_t)P.tri_global.size();
  n[3] = (int64_t)P.wall.size() / 2;
  n[4] = (int64_t)P.nbr.size();
  n[5] = (int64_t)P.send_idx.size();
  n[6] = (int64_t)P.recv_idx.size();
  n[7] = P.nv_g;
  return MRD_OK;
}

int partition_get(const mrd_partition &P, const char *name, void *dst, int64_t bytes, std::string &err) {
  const void *src = nullptr;
  int64_t have = -1;
  auto pick = [&](const char *nm, const auto &v) {
    if (!std::strcmp(name, nm)) { src = v.data(); have = (int64_t)(v.size() * sizeof(v[0])); }
  };
  if (!name) { err = "null argument"; return MRD_EINVAL; }
  pick("vertex_global", P.vertex_global); pick("xy", P.xy); pick("tri", P.tri); pick("tri_global", P.tri_global);
  pick("vertex_flag", P.flag); pick("wall_edge", P.wall); pick("neighbour", P.nbr); pick("send_off", P.send_off);
  pick("send_idx", P.send_idx); pick("recv_off", P.recv_off); pick("recv_idx", P.recv_idx); pick("owner", P.owner);
  if (have < 0) { err = std::string("unknown partition array: ") + name; return MRD_EINVAL; }
  if (have != bytes) { err = std::string("wrong size for partition array ") + name; return MRD_EINVAL; }
  if (have && !dst) { err = "null argument"; return MRD_EINVAL; }
  if (have) std::memcpy(dst, src, (size_t)have);
  return MRD_OK;
}

}  // namespace mrd_host
