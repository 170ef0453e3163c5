// mrd_layout.h -- host-side mesh-layout stage: orientation fix, minimum-image
// unwrap, Morton renumbering, vertex -> incident-triangle CSR (new: the paper
// had no such map and used atomics, L734), triangle geometry (eq. 35-37), dual volumes
// V_i (L441, reading C5), wall-edge and frozen-vertex lists (L580-L602), and the tile plan of the
// fused kernels.  Plain C++17, no CUDA.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/mrd.h"

struct mrd_layout {
  mrd_params p{};
  int64_t nv = 0, nt = 0, ne = 0, nf = 0;
  double domain_size = 1.0;           // L of eq. 56 (Bx)
  // renumbering: internal k <-> user index
  std::vector<int32_t> vperm, vrank;  // vperm[k] = user vertex of internal k; vrank = inverse
  std::vector<int32_t> tperm, trank;
  std::vector<uint8_t> tswap;         // [nt] internal: 1 = user nodes 2 and 3 were swapped (CCW fix)
  std::vector<int32_t> tri;           // [nt][3] internal vertex ids, CCW
  std::vector<int32_t> csr_off, csr_ent;  // [nv+1], [3 nt]: entries tri*3+node ascending
  // geometry, internal triangle order (double; cast to the sweep precision at upload)
  std::vector<double> nx[3], ny[3], hl[3];  // unit inward normals, half edge lengths
  std::vector<double> area, lmax;           // |T|, longest edge
  std::vector<double> vol;                  // [nv] V_i
  std::vector<uint8_t> frozen;              // [nv] internal
  // reflecting-wall edges (internal vertex ids) with OUTWARD unit normal and length (reading C15)
  std::vector<int32_t> wall_a, wall_b;
  std::vector<double> wall_nx, wall_ny, wall_len;
  // wall vertex -> (edge*2 + side) incidence, ascending; side 0 = vertex is `a`, 1 = `b`
  std::vector<int32_t> wv_vertex, wv_off, wv_ent;
  // ---- tile plan of the fused kernels ----
  int32_t tile = 0;                    // triangles per tile (0: no plan built)
  int64_t ntile = 0, nslot = 0;
  std::vector<int32_t> tile_slot_off;  // [ntile+1]: first slot of each tile (slot counts padded to multiples of 4)
  std::vector<int32_t> slot_vertex;    // [nslot]: internal vertex of each (tile-local vertex) slot, -1 = padding
  std::vector<double> slot_xy;         // [nslot][2]: coordinates unwrapped into the tile's frame
  std::vector<int32_t> vslot_off, vslot_ent;  // vertex -> its slots, ascending: [nv+1], [#real slots]
  // plan record of a tile (uint16 units; one bulk copy): [4 T] per triangle the tile-local slots of its three nodes and
  // its geometry record, [offn] first incidence batch of each slot (slot j: batches boff[j] .. boff[j+1]), [4 maxbatch]
  // incidence entries `node * T + local triangle` in ascending (triangle, node) order, four to a batch, the last batch of a
  // slot padded with the sentinel 3 T (which the kernels map to a zero residual).  Identical records are stored once.
  int32_t maxslots = 0, offn = 0, maxbatch = 0, plan_stride = 0;
  int64_t nplan = 0;                   // distinct plan records
  std::vector<int32_t> tile_plan_idx;  // [ntile]: plan record of each tile
  std::vector<uint16_t> tile_plan;     // [nplan][plan_stride]
  // geometry table: per tile the DISTINCT geometry records of its triangles (bitwise; uniform meshes have 2 per tile).
  // Record = nx[3], ny[3], hl[3], |T|/3, l_max, pad (12 values). Used by the tile kernels when it pays (geom_table).
  bool geom_table = false;
  int32_t maxshapes = 0;
  std::vector<int32_t> tile_shape_off;  // [ntile+1]
  std::vector<double> shape_geom;       // [nshape][12]
};

// one part of a domain decomposition (mrd_partition.cpp; include/mrd.h "Domain decomposition")
struct mrd_partition {
  int64_t nv_g = 0, nt_g = 0, n_owned = 0;
  int32_t n_part = 1, part = 0;
  double domain_size = 0.0;            // L of eq. 56 of the WHOLE mesh (reading C25), for the parts' mrd_params.domain_size
  std::vector<int32_t> owner;          // [nv_g]
  std::vector<int32_t> vertex_global;  // local -> global: owned (ascending), then halo (ascending)
  std::vector<double> xy;
  std::vector<int32_t> tri, tri_global;
  std::vector<uint8_t> flag;
  std::vector<int32_t> wall;
  std::vector<int32_t> nbr, send_off, send_idx, recv_off, recv_idx;
};

namespace mrd_host {
int layout_build(mrd_layout &L, const mrd_params *p, int64_t nv, const double *xy, int64_t nt,
                 const int32_t *tri, const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge,
                 std::string &err);
// vertex ids in ascending Morton key (stable), the order the layout stage and the partitioner share
void morton_order_vertices(int64_t nv, const double *xy, const double period[2], std::vector<int32_t> &perm);
int partition_build(mrd_partition &P, int64_t nv, const double *xy, int64_t nt, const int32_t *tri,
                    const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge, double period_x, double period_y,
                    int32_t n_part, int32_t part, const int32_t *owner /* [nv] or null: Morton ranges */, std::string &err);
int partition_build_local(mrd_partition &P, int64_t nv_global, double domain_size, int64_t nlv, const int32_t *vertex_global,
                          const int32_t *owner, const double *xy, const uint8_t *vertex_flag, int64_t nlt, const int32_t *tri,
                          const int32_t *tri_global, int64_t ne, const int32_t *wall_edge, int32_t n_part, int32_t part,
                          std::string &err);
int partition_sizes(const mrd_partition &P, int64_t n[8]);
int partition_get(const mrd_partition &P, const char *name, void *dst, int64_t bytes, std::string &err);
}
