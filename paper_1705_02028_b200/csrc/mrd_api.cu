// mrd_api.cu -- the C-ABI of include/mrd.h: host orchestration of the sm_100a kernels.
// No torch types, no CPU fallback: every step of the path runs in the kernels of mrd_kernels.cuh.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <map>
#include <string>
#include <vector>

#include "../../include/mrd.h"
#include "mrd_kernels.cuh"
#include "mrd_tile.cuh"
#include "mrd_layout.h"

namespace {

thread_local std::string g_err;
int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}
#define CUDA_TRY(expr)                                                                          \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess)                                                                      \
      return fail(e_ == cudaErrorMemoryAllocation ? MRD_ENOMEM : MRD_ECUDA,                     \
                  std::string(#expr) + ": " + cudaGetErrorString(e_));                          \
  } while (0)

inline unsigned blocks_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

}  // namespace

struct mrd_mesh {
  mrd_layout L;
  int device = 0;
  std::vector<void *> allocs;
  int64_t dev_bytes = 0;
  int64_t launches = 0;
  // device arrays (element type per L.p.precision where it says R)
  int32_t *d_vperm = nullptr, *d_vrank = nullptr, *d_tperm = nullptr;
  int32_t *d_tv[3] = {nullptr, nullptr, nullptr};
  void *d_gnx[3], *d_gny[3], *d_ghl[3], *d_area3 = nullptr, *d_lmax = nullptr;  // R
  int32_t *d_csr_off = nullptr, *d_csr_ent = nullptr;
  void *d_vol = nullptr;          // R
  uint8_t *d_frozen = nullptr;    // or null
  uint8_t *d_tswap = nullptr;
  // walls
  int64_t nwv = 0;
  int32_t *d_wv_vertex = nullptr, *d_wv_off = nullptr, *d_wv_ent = nullptr, *d_wall_a = nullptr, *d_wall_b = nullptr;
  void *d_wall_nx = nullptr, *d_wall_ny = nullptr, *d_wall_len = nullptr;  // R
  // state: pairs (W, Z, spd) x 2; `cur` holds W^n
  void *d_W[2] = {nullptr, nullptr}, *d_Z[2] = {nullptr, nullptr}, *d_spd[2] = {nullptr, nullptr};
  int cur = 0;
  void *d_acc = nullptr, *d_dWdt = nullptr, *d_wall_acc = nullptr;       // Vec4<R> [nv]
  void *d_phi = nullptr, *d_phiN = nullptr, *d_phiT = nullptr, *d_sT = nullptr;  // per triangle
  void *d_user = nullptr;         // R [4][nv] staging for the host variants and dumps
  mrd::Ctl *d_ctl = nullptr;
  int *d_flag = nullptr;          // non-physical flag raised by kernels
  double *d_diag = nullptr;       // [DIAG_BLOCKS][6]
  void *h_pinned = nullptr;       // pinned host staging, R [4][nv]
  // fused tile path (mrd_tile.cuh): tile plan + one partial per slot
  bool fused = false;
  bool dbg = false;               // dump: tile kernels also write per-triangle residuals to d_phi / d_sT
  int4 *d_tile_info = nullptr;    // [ntile+1]: first slot, first geometry record, plan record
  void *d_shape_geom = nullptr;   // R [nshape][12] (geometry-table kernels)
  int32_t *d_vslot_off = nullptr, *d_vslot_ent = nullptr;
  uint16_t *d_plan = nullptr;     // [nplan][plan_stride]: distinct plan records
  void *d_slot_xy = nullptr;      // R [nslot][2]
  void *d_part = nullptr, *d_partS = nullptr;  // Vec4<R> [nslot], R [nslot]
  void *d_slotZ[2] = {nullptr, nullptr}, *d_slotS[2] = {nullptr, nullptr}, *d_slotD = nullptr;  // slot-major Z, |v|+c, dW/dt
  void *d_phi12 = nullptr;        // R [ntile][12 T]: phi_0^N, phi_1^N, phi^T of W^n in the cell layout of mrd_tile.cuh
  int nsm = 0;
  std::map<const void *, unsigned> tile_grid;  // persistent grid of each tile-kernel instantiation (launch_tile)
  int launch_rc = 0;              // first error met while ENQUEUEING kernels (enqueue_step is void); returned and cleared by take_launch_rc
  void note(int rc) { if (rc && !launch_rc) launch_rc = rc; }
  // CUDA graphs for launch-bound (small) meshes: two consecutive steps (buffer parity a, then a^1) captured once per
  // starting parity on an internal stream and replayed; forked from / joined to the caller's stream by events
  cudaStream_t s_int = nullptr;
  cudaEvent_t ev_in = nullptr, ev_out = nullptr;
  cudaGraphExec_t gexec[2] = {nullptr, nullptr};
  bool graph_ok = false;
  bool has_state = false;
  int64_t steps_base = 0;         // completed steps at the last sync (for buffer parity)
  // domain decomposition (include/mrd.h "Domain decomposition"): halo lists in INTERNAL vertex ids, phase stepping
  int64_t n_send = 0, n_recv = 0;
  int32_t *d_send_idx = nullptr, *d_recv_idx = nullptr;
  bool in_phases = false;
  int phase_a = 0;                // buffer pair holding W^n of the step in flight
  int phase_next = 0;             // the phase expected next
  int64_t phase_steps0 = 0;       // device step counter at mrd_phase_begin
};

namespace {

constexpr int DIAG_BLOCKS = 1024;

template <class T> int dev_alloc(mrd_mesh *m, T **out, int64_t count) {
  size_t bytes = (size_t)(count > 0 ? count : 1) * sizeof(T);
  void *p = nullptr;
  CUDA_TRY(cudaMalloc(&p, bytes));
  m->allocs.push_back(p);
  m->dev_bytes += (int64_t)bytes;
  *out = static_cast<T *>(p);
  return MRD_OK;
}
template <class T> int dev_upload(mrd_mesh *m, T **out, const T *src, int64_t count) {
  int rc = dev_alloc(m, out, count);
  if (rc) return rc;
  if (count > 0) CUDA_TRY(cudaMemcpy(*out, src, (size_t)count * sizeof(T), cudaMemcpyHostToDevice));
  return MRD_OK;
}
// upload a double array converted to the sweep precision
template <class R> int dev_upload_real(mrd_mesh *m, void **out, const double *src, int64_t count, double scale = 1.0) {
  std::vector<R> tmp((size_t)count);
  for (int64_t i = 0; i < count; ++i) tmp[i] = (R)(src[i] * scale);
  R *p = nullptr;
  int rc = dev_upload<R>(m, &p, tmp.data(), count);
  *out = p;
  return rc;
}

template <class R> mrd::MeshDev<R> mesh_dev(const mrd_mesh *m) {
  mrd::MeshDev<R> d;
  d.nv = m->L.nv;
  d.nt = m->L.nt;
  for (int i = 0; i < 3; ++i) {
    d.tv[i] = m->d_tv[i];
    d.gnx[i] = (const R *)m->d_gnx[i];
    d.gny[i] = (const R *)m->d_gny[i];
    d.ghl[i] = (const R *)m->d_ghl[i];
  }
  d.area3 = (const R *)m->d_area3;
  d.lmax = (const R *)m->d_lmax;
  d.csr_off = m->d_csr_off;
  d.csr_ent = m->d_csr_ent;
  d.vol = (const R *)m->d_vol;
  d.frozen = m->d_frozen;
  return d;
}
template <class R> mrd::TileDev<R> tile_dev(const mrd_mesh *m) {
  mrd::TileDev<R> t;
  t.tile = m->L.tile;
  t.maxslots = m->L.maxslots;
  t.offn = m->L.offn;
  t.maxbatch = m->L.maxbatch;
  t.plan_stride = m->L.plan_stride;
  t.ntile = m->L.ntile;
  t.nslot = m->L.nslot;
  t.nt = m->L.nt;
  t.nv = m->L.nv;
  t.maxshapes = m->L.geom_table ? m->L.maxshapes : 0;
  t.tile_info = m->d_tile_info;
  t.shape_geom = (const R *)m->d_shape_geom;
  t.plan = m->d_plan;
  t.slot_xy = (const R *)m->d_slot_xy;
  t.vslot_off = m->d_vslot_off;
  t.vslot_ent = m->d_vslot_ent;
  return t;
}
// where the vertex kernels put Z / |v|+c / dW/dt of buffer pair `pair`
template <class R> mrd::VertexSink<R> sink_for(const mrd_mesh *m, int pair, bool want_spd, bool want_d) {
  mrd::VertexSink<R> k;
  if (m->fused) {
    k.Z = (mrd::Vec4<R> *)m->d_slotZ[pair];
    k.spd = want_spd ? (R *)m->d_slotS[pair] : nullptr;
    k.D = want_d ? (mrd::Vec4<R> *)m->d_slotD : nullptr;
    k.vslot_off = m->d_vslot_off;
    k.vslot_ent = m->d_vslot_ent;
  } else {
    k.Z = (mrd::Vec4<R> *)m->d_Z[pair];
    k.spd = want_spd ? (R *)m->d_spd[pair] : nullptr;
    k.D = want_d ? (mrd::Vec4<R> *)m->d_dWdt : nullptr;
    k.vslot_off = nullptr;
    k.vslot_ent = nullptr;
  }
  return k;
}
template <class R> mrd::WallDev<R> wall_dev(const mrd_mesh *m) {
  mrd::WallDev<R> w;
  w.nwv = m->nwv;
  w.wv_vertex = m->d_wv_vertex;
  w.wv_off = m->d_wv_off;
  w.wv_ent = m->d_wv_ent;
  w.wall_a = m->d_wall_a;
  w.wall_b = m->d_wall_b;
  w.nx = (const R *)m->d_wall_nx;
  w.ny = (const R *)m->d_wall_ny;
  w.len = (const R *)m->d_wall_len;
  return w;
}

template <class R> int upload_impl(mrd_mesh *m) {
  using V4 = mrd::Vec4<R>;
  mrd_layout &L = m->L;
  const int64_t nv = L.nv, nt = L.nt;
  int rc;
  if ((rc = dev_upload(m, &m->d_vperm, L.vperm.data(), nv))) return rc;
  if ((rc = dev_upload(m, &m->d_vrank, L.vrank.data(), nv))) return rc;
  if ((rc = dev_upload(m, &m->d_tperm, L.tperm.data(), nt))) return rc;
  if ((rc = dev_upload(m, &m->d_tswap, L.tswap.data(), nt))) return rc;
  m->fused = L.tile > 0;
  if (!m->fused) {
    std::vector<int32_t> col(nt);
    for (int j = 0; j < 3; ++j) {
      for (int64_t t = 0; t < nt; ++t) col[t] = L.tri[3 * t + j];
      if ((rc = dev_upload(m, &m->d_tv[j], col.data(), nt))) return rc;
    }
    for (int i = 0; i < 3; ++i) {
      if ((rc = dev_upload_real<R>(m, &m->d_gnx[i], L.nx[i].data(), nt))) return rc;
      if ((rc = dev_upload_real<R>(m, &m->d_gny[i], L.ny[i].data(), nt))) return rc;
      if ((rc = dev_upload_real<R>(m, &m->d_ghl[i], L.hl[i].data(), nt))) return rc;
    }
    if ((rc = dev_upload_real<R>(m, &m->d_area3, L.area.data(), nt, 1.0 / 3.0))) return rc;
    if ((rc = dev_upload_real<R>(m, &m->d_lmax, L.lmax.data(), nt))) return rc;
    if ((rc = dev_upload(m, &m->d_csr_off, L.csr_off.data(), nv + 1))) return rc;
    if ((rc = dev_upload(m, &m->d_csr_ent, L.csr_ent.data(), 3 * nt))) return rc;
  } else {
    {
      std::vector<int4> info(L.ntile + 1);
      for (int64_t b = 0; b <= L.ntile; ++b)
        info[b] = make_int4(L.tile_slot_off[b], L.geom_table ? L.tile_shape_off[b] : 0, b < L.ntile ? L.tile_plan_idx[b] : 0, 0);
      if ((rc = dev_upload(m, &m->d_tile_info, info.data(), L.ntile + 1))) return rc;
    }
    if (L.geom_table && (rc = dev_upload_real<R>(m, &m->d_shape_geom, L.shape_geom.data(), (int64_t)L.shape_geom.size()))) return rc;
    if ((rc = dev_upload(m, &m->d_plan, L.tile_plan.data(), (int64_t)L.tile_plan.size()))) return rc;
    if (!L.geom_table && (rc = dev_upload_real<R>(m, &m->d_slot_xy, L.slot_xy.data(), 2 * L.nslot))) return rc;
    if ((rc = dev_upload(m, &m->d_vslot_off, L.vslot_off.data(), nv + 1))) return rc;
    if ((rc = dev_upload(m, &m->d_vslot_ent, L.vslot_ent.data(), (int64_t)L.vslot_ent.size()))) return rc;
    V4 *pp = nullptr, *sd = nullptr;
    R *ps = nullptr, *p12 = nullptr;
    if ((rc = dev_alloc(m, &pp, L.nslot)) || (rc = dev_alloc(m, &ps, L.nslot)) || (rc = dev_alloc(m, &sd, L.nslot))) return rc;
    if ((rc = dev_alloc(m, &p12, L.ntile * 12 * L.tile))) return rc;
    CUDA_TRY(cudaMemset(sd, 0, sizeof(V4) * L.nslot));
    m->d_slotD = sd; m->d_phi12 = p12;
    for (int b = 0; b < 2; ++b) {
      V4 *z = nullptr;
      R *sp = nullptr;
      if ((rc = dev_alloc(m, &z, L.nslot)) || (rc = dev_alloc(m, &sp, L.nslot))) return rc;
      CUDA_TRY(cudaMemset(z, 0, sizeof(V4) * L.nslot));   // padding slots are copied (never used): keep them defined
      CUDA_TRY(cudaMemset(sp, 0, sizeof(R) * L.nslot));
      m->d_slotZ[b] = z; m->d_slotS[b] = sp;
    }
    m->d_part = pp; m->d_partS = ps;
  }
  {
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, m->device));
    m->nsm = prop.multiProcessorCount;
  }
  if ((rc = dev_upload_real<R>(m, &m->d_vol, L.vol.data(), nv))) return rc;
  if (L.nf > 0 && (rc = dev_upload(m, &m->d_frozen, L.frozen.data(), nv))) return rc;
  m->nwv = (int64_t)L.wv_vertex.size();
  if (L.ne > 0) {
    if ((rc = dev_upload(m, &m->d_wv_vertex, L.wv_vertex.data(), m->nwv))) return rc;
    if ((rc = dev_upload(m, &m->d_wv_off, L.wv_off.data(), m->nwv + 1))) return rc;
    if ((rc = dev_upload(m, &m->d_wv_ent, L.wv_ent.data(), (int64_t)L.wv_ent.size()))) return rc;
    if ((rc = dev_upload(m, &m->d_wall_a, L.wall_a.data(), L.ne))) return rc;
    if ((rc = dev_upload(m, &m->d_wall_b, L.wall_b.data(), L.ne))) return rc;
    if ((rc = dev_upload_real<R>(m, &m->d_wall_nx, L.wall_nx.data(), L.ne))) return rc;
    if ((rc = dev_upload_real<R>(m, &m->d_wall_ny, L.wall_ny.data(), L.ne))) return rc;
    if ((rc = dev_upload_real<R>(m, &m->d_wall_len, L.wall_len.data(), L.ne))) return rc;
    V4 *wa = nullptr;
    if ((rc = dev_alloc(m, &wa, nv))) return rc;
    CUDA_TRY(cudaMemset(wa, 0, (size_t)nv * sizeof(V4)));
    m->d_wall_acc = wa;
  }
  for (int b = 0; b < 2; ++b) {
    V4 *w = nullptr, *z = nullptr;
    R *s = nullptr;
    if ((rc = dev_alloc(m, &w, nv))) return rc;
    if (!m->fused && ((rc = dev_alloc(m, &z, nv)) || (rc = dev_alloc(m, &s, nv)))) return rc;
    m->d_W[b] = w; m->d_Z[b] = z; m->d_spd[b] = s;
  }
  {
    V4 *a = nullptr, *d = nullptr, *p = nullptr, *pn = nullptr, *pt = nullptr;
    R *st = nullptr, *us = nullptr;
    if (!m->fused && ((rc = dev_alloc(m, &a, nv)) || (rc = dev_alloc(m, &d, nv)) || (rc = dev_alloc(m, &p, 3 * nt)) || (rc = dev_alloc(m, &st, nt)) ||
                      (rc = dev_alloc(m, &pn, 3 * nt)) || (rc = dev_alloc(m, &pt, nt))))
      return rc;
    if ((rc = dev_alloc(m, &us, 4 * nv))) return rc;
    m->d_acc = a; m->d_dWdt = d; m->d_phi = p; m->d_phiN = pn; m->d_phiT = pt; m->d_sT = st; m->d_user = us;
  }
  if ((rc = dev_alloc(m, &m->d_ctl, 1)) || (rc = dev_alloc(m, &m->d_flag, 1)) || (rc = dev_alloc(m, &m->d_diag, DIAG_BLOCKS * 6))) return rc;
  CUDA_TRY(cudaMemset(m->d_ctl, 0, sizeof(mrd::Ctl)));
  CUDA_TRY(cudaMemset(m->d_flag, 0, sizeof(int)));
  CUDA_TRY(cudaDeviceSynchronize());
  return MRD_OK;
}

template <class R> int set_state_impl(mrd_mesh *m, const R *W_dev, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const int64_t nv = m->L.nv;
  m->cur = 0;
  m->has_state = false;
  mrd::Ctl c{};
  c.t = 0.0; c.dt = 0.0; c.t_end = 0.0; c.cfl = m->L.p.cfl;
  c.dmin_bits = 0x7FF0000000000000ull; c.steps = 0; c.status = 0; c.active = 0;
  c.bvar = m->L.p.scheme == MRD_SCHEME_BMAX ? 1 : (m->L.p.scheme == MRD_SCHEME_BMIN ? 2 : 0);
  c.lumping = m->L.p.lumping;
  c.bx_L = m->L.domain_size;
  c.vmax_bits[0] = c.vmax_bits[1] = 0ull;
  c.vmin_bits[0] = c.vmin_bits[1] = 0x7FF0000000000000ull;
  CUDA_TRY(cudaMemcpyAsync(m->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice, s));
  CUDA_TRY(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
  mrd::set_state_kernel<R><<<blocks_for(nv, 256), 256, 0, s>>>(nv, m->d_vperm, W_dev, (R)m->L.p.gamma, (V4 *)m->d_W[0],
                                                               sink_for<R>(m, 0, true, false), m->d_flag);
  m->launches++;
  int flag = 0;
  CUDA_TRY(cudaMemcpyAsync(&flag, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  CUDA_TRY(cudaGetLastError());
  m->steps_base = 0;
  if (flag) {
    CUDA_TRY(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
    return fail(MRD_ENONPHYSICAL, "state has rho <= 0 or p <= 0");
  }
  m->has_state = true;
  return MRD_OK;
}

template <class R> int get_state_impl(mrd_mesh *m, R *W_dev, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const int64_t nv = m->L.nv;
  mrd::get_state_kernel<R><<<blocks_for(nv, 256), 256, 0, s>>>(nv, m->d_vrank, (const V4 *)m->d_W[m->cur], W_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}

// persistent launch of a tile kernel: dynamic shared memory opt-in, grid = SMs x resident blocks (<= ntile).  The opt-in
// and the occupancy query run once per (kernel instantiation, mesh); their result is cached in the mesh.
template <class K, class... Args> int launch_tile(mrd_mesh *m, K kernel, size_t sh, cudaStream_t s, Args... args) {
  const int T = m->L.tile;
  const void *key = (const void *)kernel;
  auto it = m->tile_grid.find(key);
  if (it == m->tile_grid.end()) {
    cudaError_t e = cudaFuncSetAttribute(key, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh);
    if (e != cudaSuccess)
      return fail(MRD_ECUDA, "tile kernel: cannot opt in to " + std::to_string(sh) + " bytes of dynamic shared memory: " + cudaGetErrorString(e));
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, T, sh);
    if (e != cudaSuccess || occ < 1)
      return fail(MRD_ECUDA, std::string("tile kernel: no resident block fits (") + std::to_string(sh) + " bytes of shared memory): " + cudaGetErrorString(e));
    it = m->tile_grid.emplace(key, (unsigned)std::min<int64_t>(m->L.ntile, (int64_t)m->nsm * occ)).first;
  }
  kernel<<<it->second, T, sh, s>>>(args...);
  m->launches++;
  return MRD_OK;
}
// tile sizes the fused kernels are compiled for
#define MRD_TILE_DISPATCH_G(T, CALL)                      \
  switch (T) {                                           \
    case 64: { constexpr int TILE = 64; CALL; } break;   \
    case 256: { constexpr int TILE = 256; CALL; } break; \
    default: { constexpr int TILE = 128; CALL; } break;  \
  }
#define MRD_TILE_DISPATCH(T, CALL)                                      \
  if (m->L.geom_table) { constexpr bool GTAB = true; MRD_TILE_DISPATCH_G(T, CALL) } \
  else { constexpr bool GTAB = false; MRD_TILE_DISPATCH_G(T, CALL) }
// `a`: buffer pair holding W^n.  Fused path: residuals of W^n -> one partial per tile slot; unfused path: per-triangle
// residuals d_phi, s_T.
template <class R, int SCHEME> void launch_stage1(mrd_mesh *m, bool store, int a, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const R gamma = (R)m->L.p.gamma;
  if (m->fused) {
    auto td = tile_dev<R>(m);
#define MRD_SMEM(STAGE) mrd::TileSmem<R, STAGE, GTAB>(td.tile, td.maxslots, td.plan_stride, td.maxshapes)
    mrd::TileIO<R> io{};
    io.slotZ = (const V4 *)m->d_slotZ[a];
    io.slotS = (const R *)m->d_slotS[a];
    io.slotD = (const V4 *)m->d_slotD;
    io.phi12 = (R *)m->d_phi12;
    io.part = (V4 *)m->d_part;
    io.partS = (R *)m->d_partS;
    io.phi_dbg = m->dbg ? (V4 *)m->d_phi : nullptr;
    io.sT_dbg = m->dbg ? (R *)m->d_sT : nullptr;
    if (store) {
      MRD_TILE_DISPATCH(td.tile, m->note(launch_tile(m, mrd::tile_kernel<R, SCHEME, 1, true, TILE, GTAB>, MRD_SMEM(1).total, s, td, MRD_SMEM(1), gamma, (const mrd::Ctl *)m->d_ctl, io, m->d_flag)))
    } else {
      MRD_TILE_DISPATCH(td.tile, m->note(launch_tile(m, mrd::tile_kernel<R, SCHEME, 1, false, TILE, GTAB>, MRD_SMEM(1).total, s, td, MRD_SMEM(1), gamma, (const mrd::Ctl *)m->d_ctl, io, m->d_flag)))
    }
    return;
  }
  auto md = mesh_dev<R>(m);
  const unsigned nb = blocks_for(md.nt, 128);
  if (store)
    mrd::tri_stage1_kernel<R, SCHEME, true><<<nb, 128, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_Z[a], (const R *)m->d_spd[a],
                                                            (V4 *)m->d_phi, (V4 *)m->d_phiN, (V4 *)m->d_phiT, (R *)m->d_sT, m->d_flag);
  else
    mrd::tri_stage1_kernel<R, SCHEME, false><<<nb, 128, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_Z[a], (const R *)m->d_spd[a],
                                                             (V4 *)m->d_phi, (V4 *)m->d_phiN, (V4 *)m->d_phiT, (R *)m->d_sT, m->d_flag);
  m->launches++;
}
// `b`: buffer pair holding W*.  Total residuals of eq. 61-65 -> one partial per tile slot (fused) / d_phi (unfused).
template <class R, int SCHEME> void launch_stage2(mrd_mesh *m, int b, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const R gamma = (R)m->L.p.gamma;
  if (m->fused) {
    auto td = tile_dev<R>(m);
    mrd::TileIO<R> io{};
    io.slotZ = (const V4 *)m->d_slotZ[b];
    io.slotD = (const V4 *)m->d_slotD;
    io.phi12 = (R *)m->d_phi12;
    io.part = (V4 *)m->d_part;
    if (m->L.p.lumping) {
      constexpr bool LUMP = true;
      MRD_TILE_DISPATCH(td.tile, m->note(launch_tile(m, mrd::tile_kernel<R, SCHEME, 2, LUMP, TILE, GTAB>, MRD_SMEM(2).total, s, td, MRD_SMEM(2), gamma, (const mrd::Ctl *)m->d_ctl, io, m->d_flag)))
    } else {
      constexpr bool LUMP = false;
      MRD_TILE_DISPATCH(td.tile, m->note(launch_tile(m, mrd::tile_kernel<R, SCHEME, 2, LUMP, TILE, GTAB>, MRD_SMEM(2).total, s, td, MRD_SMEM(2), gamma, (const mrd::Ctl *)m->d_ctl, io, m->d_flag)))
    }
    return;
  }
  auto md = mesh_dev<R>(m);
  mrd::tri_stage2_kernel<R, SCHEME><<<blocks_for(md.nt, 128), 128, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_Z[b],
                                                                        (const V4 *)m->d_dWdt, (const V4 *)m->d_phiN, (const V4 *)m->d_phiT,
                                                                        (V4 *)m->d_phi, m->d_flag);
  m->launches++;
}

// optional per-kernel timing of one step (mrd_step_profile): an event after every launch
struct Prof {
  cudaEvent_t ev[MRD_PROFILE_SLOTS + 2];
  int slot[MRD_PROFILE_SLOTS + 2];
  int n = 0;
  void mark(int k, cudaStream_t s) {
    slot[n] = k;
    cudaEventRecord(ev[n], s);
    ++n;
  }
};
#define PROF_MARK(k) \
  if (prof) prof->mark((k), s);

// one time step enqueued on s; `a` = buffer pair holding W^n.  `mask` selects phases (bit k = MRD_PHASE_k): the
// whole step by default; mrd_phase enqueues them one at a time so that a caller can exchange in between.
template <class R> void enqueue_step(mrd_mesh *m, int scheme, int a, cudaStream_t s, Prof *prof = nullptr, int mask = 15) {
  using V4 = mrd::Vec4<R>;
  const int b = a ^ 1;
  const bool rk2 = m->L.p.time_order == 2;
  auto md = mesh_dev<R>(m);
  const R gamma = (R)m->L.p.gamma;
  const unsigned vb = blocks_for(md.nv, 256);
  const bool fused = m->fused;
  if (mask & (1 << MRD_PHASE_RESIDUAL1)) {
    if (scheme == MRD_SCHEME_BX && !m->in_phases) {  // eq. 56: |v|_max - |v|_min of W^n (in phases: mrd_range_get / _set)
      mrd::vrange_kernel<R><<<std::min<unsigned>(vb, (unsigned)m->nsm * 8), 256, 0, s>>>(md.nv, (const V4 *)m->d_W[a], m->d_ctl, 0);
      m->launches++;
    }
    switch (scheme) {
      case MRD_SCHEME_N: launch_stage1<R, MRD_SCHEME_N>(m, rk2, a, s); break;
      case MRD_SCHEME_LDA: launch_stage1<R, MRD_SCHEME_LDA>(m, rk2, a, s); break;
      case MRD_SCHEME_BX: launch_stage1<R, MRD_SCHEME_BX>(m, rk2, a, s); break;
      default: launch_stage1<R, MRD_SCHEME_B>(m, rk2, a, s); break;
    }
    PROF_MARK(MRD_PROF_TRI1)
    if (fused) {
      // fused path: dt from the partial s_T sums alone; the update kernels gather the residual partials themselves
      mrd::slot_dt_kernel<R><<<std::min<unsigned>(vb, (unsigned)m->nsm * 8), 256, 0, s>>>(md, tile_dev<R>(m), m->d_ctl, (const R *)m->d_partS);
    } else {
      // unfused comparison path: per-triangle residuals through HBM, CSR gathers, acc round trip
      mrd::gather_dt_kernel<R><<<vb, 256, 0, s>>>(md, m->d_ctl, (const V4 *)m->d_phi, (const R *)m->d_sT, (V4 *)m->d_acc);
    }
    m->launches++;
    PROF_MARK(MRD_PROF_GATHER_DT)
    if (m->nwv > 0) {
      if (fused)
        mrd::wall_kernel<R, 1, true><<<blocks_for(m->nwv, 128), 128, 0, s>>>(wall_dev<R>(m), gamma, m->d_ctl, (const V4 *)m->d_W[a], (const V4 *)m->d_W[a],
                                                                          (V4 *)m->d_wall_acc);
      else
        mrd::wall_kernel<R, 1, false><<<blocks_for(m->nwv, 128), 128, 0, s>>>(wall_dev<R>(m), gamma, m->d_ctl, (const V4 *)m->d_W[a], (const V4 *)m->d_W[a],
                                                                           (V4 *)m->d_acc);
      m->launches++;
      PROF_MARK(MRD_PROF_WALL1)
    }
  }
  if (mask & (1 << MRD_PHASE_UPDATE1)) {
    if (fused) {
      auto td = tile_dev<R>(m);
      if (!rk2)
        mrd::slot_gather_update_kernel<R, 1><<<blocks_for(md.nv, mrd::VtxShape<R>::threads), mrd::VtxShape<R>::threads, 0, s>>>(md, td, gamma, m->d_ctl, (const V4 *)m->d_part, (const V4 *)m->d_wall_acc,
                                                             (const V4 *)m->d_W[a], (V4 *)m->d_W[b], sink_for<R>(m, b, true, false), m->d_flag);
      else
        mrd::slot_gather_update_kernel<R, 0><<<blocks_for(md.nv, mrd::VtxShape<R>::threads), mrd::VtxShape<R>::threads, 0, s>>>(md, td, gamma, m->d_ctl, (const V4 *)m->d_part, (const V4 *)m->d_wall_acc,
                                                             (const V4 *)m->d_W[a], (V4 *)m->d_W[b], sink_for<R>(m, b, false, true), m->d_flag);
    } else {
      if (!rk2)
        mrd::update_kernel<R, true><<<vb, 256, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_W[a], (const V4 *)m->d_acc, (V4 *)m->d_W[b],
                                                    sink_for<R>(m, b, true, false), m->d_flag);
      else
        mrd::update_kernel<R, false><<<vb, 256, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_W[a], (const V4 *)m->d_acc, (V4 *)m->d_W[b],
                                                     sink_for<R>(m, b, false, true), m->d_flag);
    }
    m->launches++;
    PROF_MARK(MRD_PROF_UPDATE)
  }
  if (rk2 && (mask & (1 << MRD_PHASE_STAGE2))) {
    if (scheme == MRD_SCHEME_BX && !m->in_phases) {  // ... and of W*
      mrd::vrange_kernel<R><<<std::min<unsigned>(vb, (unsigned)m->nsm * 8), 256, 0, s>>>(md.nv, (const V4 *)m->d_W[b], m->d_ctl, 1);
      m->launches++;
    }
    switch (scheme) {
      case MRD_SCHEME_N: launch_stage2<R, MRD_SCHEME_N>(m, b, s); break;
      case MRD_SCHEME_LDA: launch_stage2<R, MRD_SCHEME_LDA>(m, b, s); break;
      case MRD_SCHEME_BX: launch_stage2<R, MRD_SCHEME_BX>(m, b, s); break;
      default: launch_stage2<R, MRD_SCHEME_B>(m, b, s); break;
    }
    PROF_MARK(MRD_PROF_TRI2)
    if (m->nwv > 0) {
      mrd::wall_kernel<R, 2><<<blocks_for(m->nwv, 128), 128, 0, s>>>(wall_dev<R>(m), gamma, m->d_ctl, (const V4 *)m->d_W[a], (const V4 *)m->d_W[b],
                                                                  (V4 *)m->d_wall_acc);
      m->launches++;
      PROF_MARK(MRD_PROF_WALL2)
    }
    if (fused)
      mrd::slot_gather_update_kernel<R, 2><<<blocks_for(md.nv, mrd::VtxShape<R>::threads), mrd::VtxShape<R>::threads, 0, s>>>(md, tile_dev<R>(m), gamma, m->d_ctl, (const V4 *)m->d_part, (const V4 *)m->d_wall_acc,
                                                           (const V4 *)m->d_W[b], (V4 *)m->d_W[b], sink_for<R>(m, b, true, false), m->d_flag);
    else
      mrd::gather_update_kernel<R><<<vb, 256, 0, s>>>(md, gamma, m->d_ctl, (const V4 *)m->d_phi, (const V4 *)m->d_wall_acc, (V4 *)m->d_W[b],
                                                   sink_for<R>(m, b, true, false), m->d_flag);
    m->launches++;
    PROF_MARK(MRD_PROF_GATHER_UPDATE)
  }
  if (mask & (1 << MRD_PHASE_END)) {
    mrd::ctl_kernel<<<1, 1, 0, s>>>(m->d_ctl, 1, 0.0, m->d_flag);
    m->launches++;
    PROF_MARK(MRD_PROF_CTL)
  }
  // a launch that could not be enqueued (bad configuration, shared-memory opt-in refused) is reported by the caller
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) m->note(fail(MRD_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(e)));
}
// kernel launches of one step (the CUDA-graph replay counts them without launching)
inline int64_t launches_per_step(const mrd_mesh *m, int scheme) {
  const bool rk2 = m->L.p.time_order == 2;
  int64_t n = rk2 ? 6 : 4;
  if (m->nwv > 0) n += rk2 ? 2 : 1;
  if (scheme == MRD_SCHEME_BX) n += m->L.p.time_order;
  return n;
}
// the first error met while enqueueing since the last call (0 if none)
int take_launch_rc(mrd_mesh *m) {
  const int rc = m->launch_rc;
  m->launch_rc = 0;
  return rc;
}

// n consecutive steps starting from buffer pair `a` (updated).  Small meshes replay a captured two-step graph.
template <class R> int run_steps(mrd_mesh *m, int scheme, int64_t n, int &a, cudaStream_t s) {
  if (!m->graph_ok || n < 2) {
    for (int64_t k = 0; k < n; ++k, a ^= 1) enqueue_step<R>(m, scheme, a, s);
    return take_launch_rc(m);
  }
  CUDA_TRY(cudaEventRecord(m->ev_in, s));
  CUDA_TRY(cudaStreamWaitEvent(m->s_int, m->ev_in, 0));
  if (!m->gexec[0] || !m->gexec[1]) {
    // first multi-step call: one eager step (sets the kernels' shared-memory attributes before any capture), then the
    // graphs of BOTH starting parities, so that no later call -- a timed one, say -- pays for an instantiation
    enqueue_step<R>(m, scheme, a, m->s_int);
    a ^= 1;
    --n;
    for (int p = 0; p < 2; ++p) {
      if (m->gexec[p]) continue;
      const int64_t lc = m->launches;
      cudaGraph_t g = nullptr;
      CUDA_TRY(cudaStreamBeginCapture(m->s_int, cudaStreamCaptureModeThreadLocal));
      enqueue_step<R>(m, scheme, p, m->s_int);
      enqueue_step<R>(m, scheme, p ^ 1, m->s_int);
      CUDA_TRY(cudaStreamEndCapture(m->s_int, &g));
      m->launches = lc;  // captured, not launched
      cudaError_t e = cudaGraphInstantiate(&m->gexec[p], g, 0);
      cudaGraphDestroy(g);
      if (e != cudaSuccess) return fail(MRD_ECUDA, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
    }
  }
  const int64_t per_step = launches_per_step(m, scheme);
  for (int64_t k = 0; k + 1 < n; k += 2) {
    CUDA_TRY(cudaGraphLaunch(m->gexec[a], m->s_int));
    m->launches += 2 * per_step;
  }
  if (n & 1) {
    enqueue_step<R>(m, scheme, a, m->s_int);
    a ^= 1;
  }
  CUDA_TRY(cudaEventRecord(m->ev_out, m->s_int));
  CUDA_TRY(cudaStreamWaitEvent(s, m->ev_out, 0));
  return take_launch_rc(m);
}

// fetch the control block (after a stream sync) and bring the host bookkeeping up to date
int fetch_ctl(mrd_mesh *m, cudaStream_t s, mrd::Ctl *out) {
  CUDA_TRY(cudaMemcpyAsync(out, m->d_ctl, sizeof(mrd::Ctl), cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  CUDA_TRY(cudaGetLastError());
  // every completed step swapped the buffer pairs once
  int64_t done = out->steps - m->steps_base;
  if (done & 1) m->cur ^= 1;
  m->steps_base = out->steps;
  return MRD_OK;
}

// A step that met rho <= 0, p <= 0 or c^2 <= 0 was discarded on the device (the buffer pair holding W^n is never written
// during a step): clear the flag so that the state -- the last good step -- stays usable, and report it.
int discard_failed_step(mrd_mesh *m, const mrd::Ctl &c, cudaStream_t s) {
  mrd::Ctl fix = c;
  fix.status = 0;
  fix.active = 0;
  CUDA_TRY(cudaMemcpyAsync(m->d_ctl, &fix, sizeof fix, cudaMemcpyHostToDevice, s));
  CUDA_TRY(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
  CUDA_TRY(cudaStreamSynchronize(s));
  return fail(MRD_ENONPHYSICAL, "non-physical state (rho <= 0, p <= 0 or c^2 <= 0) met; state left at the last good step");
}

template <class R> int step_impl(mrd_mesh *m, int64_t max_steps, double t_end, cudaStream_t s, bool sync,
                                 int64_t *steps_done, double *t, double *dt_last) {
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  if (max_steps < 0) return fail(MRD_EINVAL, "max_steps < 0");
  if (m->in_phases) return fail(MRD_EINVAL, "mrd_step inside mrd_phase_begin / mrd_phase_end");
  mrd::Ctl c{};
  int rc;
  // steps enqueued by earlier async calls change the parity: settle it first
  if ((rc = fetch_ctl(m, s, &c))) return rc;
  if (c.status) return fail(MRD_ENONPHYSICAL, "state is non-physical (an earlier step failed)");
  const int64_t steps0 = c.steps;
  mrd::ctl_kernel<<<1, 1, 0, s>>>(m->d_ctl, 0, t_end > 0.0 ? t_end : 0.0, m->d_flag);
  m->launches++;
  const int scheme = m->L.p.scheme;
  int64_t enq = 0;
  int a = m->cur;
  if (!(t_end > 0.0)) {
    if ((rc = run_steps<R>(m, scheme, max_steps, a, s))) return rc;
    enq = max_steps;
    if (!sync) { CUDA_TRY(cudaGetLastError()); return MRD_OK; }
    if ((rc = fetch_ctl(m, s, &c))) return rc;
  } else {
    // t_end mode: the device decides when to stop; the host enqueues in chunks and looks at the clock
    const int64_t chunk = 32;
    while (enq < max_steps) {
      int64_t n = std::min<int64_t>(chunk, max_steps - enq);
      if ((rc = run_steps<R>(m, scheme, n, a, s))) return rc;
      enq += n;
      if ((rc = fetch_ctl(m, s, &c))) return rc;
      a = m->cur;
      if (c.status || c.t >= t_end) break;
      if (c.steps - steps0 < enq) break;  // defensive: device stopped for another reason
    }
  }
  if (steps_done) *steps_done = c.steps - steps0;
  if (t) *t = c.t;
  if (dt_last) *dt_last = c.dt;
  if (c.status) return discard_failed_step(m, c, s);
  return MRD_OK;
}

// ---- phase stepping and halo exchange (include/mrd.h "Domain decomposition") --------------------------------
template <class R> int phase_impl(mrd_mesh *m, int phase, cudaStream_t s) {
  enqueue_step<R>(m, m->L.p.scheme, m->phase_a, s, nullptr, 1 << phase);
  return take_launch_rc(m);
}
template <class R> int halo_pack_impl(mrd_mesh *m, void *buf, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  if (m->n_send > 0) {
    mrd::halo_pack_kernel<R><<<blocks_for(m->n_send, 256), 256, 0, s>>>(m->n_send, m->d_send_idx, m->d_ctl, (const V4 *)m->d_W[m->phase_a ^ 1], (V4 *)buf);
    m->launches++;
    CUDA_TRY(cudaGetLastError());
  }
  return MRD_OK;
}
template <class R> int halo_unpack_impl(mrd_mesh *m, const void *buf, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  if (m->n_recv == 0) return MRD_OK;
  const int a = m->phase_a, b = a ^ 1;
  const R gamma = (R)m->L.p.gamma;
  const unsigned nb = blocks_for(m->n_recv, 256);
  // after UPDATE1 of RK2 the buffer holds W*; otherwise W^{n+1}
  const bool first = m->L.p.time_order == 2 && m->phase_next == MRD_PHASE_STAGE2;
  if (first)
    mrd::halo_unpack_kernel<R, true><<<nb, 256, 0, s>>>(m->n_recv, m->d_recv_idx, gamma, m->d_ctl, (const V4 *)buf, (const V4 *)m->d_W[a], (V4 *)m->d_W[b],
                                                      sink_for<R>(m, b, false, true), m->d_flag);
  else
    mrd::halo_unpack_kernel<R, false><<<nb, 256, 0, s>>>(m->n_recv, m->d_recv_idx, gamma, m->d_ctl, (const V4 *)buf, (const V4 *)m->d_W[a], (V4 *)m->d_W[b],
                                                       sink_for<R>(m, b, true, false), m->d_flag);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}

template <class R> int diag_impl(mrd_mesh *m, double totals[4], double *min_rho, double *min_p, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  mrd::diag_kernel<R><<<DIAG_BLOCKS, 256, 0, s>>>(m->L.nv, (R)m->L.p.gamma, (const V4 *)m->d_W[m->cur], (const R *)m->d_vol, m->d_frozen, m->d_diag);
  m->launches++;
  std::vector<double> h(DIAG_BLOCKS * 6);
  CUDA_TRY(cudaMemcpyAsync(h.data(), m->d_diag, h.size() * sizeof(double), cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  CUDA_TRY(cudaGetLastError());
  double tot[4] = {0, 0, 0, 0}, mr = INFINITY, mp = INFINITY;
  for (int b = 0; b < DIAG_BLOCKS; ++b) {
    for (int k = 0; k < 4; ++k) tot[k] += h[6 * b + k];
    mr = std::fmin(mr, h[6 * b + 4]);
    mp = std::fmin(mp, h[6 * b + 5]);
  }
  if (totals) std::memcpy(totals, tot, sizeof tot);
  if (min_rho) *min_rho = mr;
  if (min_p) *min_p = mp;
  return MRD_OK;
}

// stage 1 of the Bx blend for the dumps: the speed range of the current state (eq. 56), then the Bx kernels
template <class R> void launch_bx_stage1(mrd_mesh *m, int a, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const unsigned vb = blocks_for(m->L.nv, 256);
  mrd::vrange_kernel<R><<<std::min<unsigned>(vb, (unsigned)m->nsm * 8), 256, 0, s>>>(m->L.nv, (const V4 *)m->d_W[a], m->d_ctl, 0);
  m->launches++;
  launch_stage1<R, MRD_SCHEME_BX>(m, true, a, s);
}

// per-triangle dump of stage 1 in USER numbering / node order
template <class R> int dump_impl(mrd_mesh *m, double *phiT, double *phiN, double *phiLDA, double *phiB, double *sT, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const int64_t nt = m->L.nt;
  mrd::Ctl c{};
  int rc;
  if ((rc = fetch_ctl(m, s, &c))) return rc;
  // arm the guard without touching the clock
  mrd::Ctl armed = c;
  armed.active = 1;
  CUDA_TRY(cudaMemcpyAsync(m->d_ctl, &armed, sizeof armed, cudaMemcpyHostToDevice, s));
  std::vector<R> h3((size_t)12 * nt), h1((size_t)4 * nt), hs((size_t)nt);
  auto put3 = [&](double *dst) {  // [nt][3][4] internal -> user triangle order, undo the node swap
    for (int64_t k = 0; k < nt; ++k) {
      int64_t u = m->L.tperm[k];
      for (int i = 0; i < 3; ++i) {
        int iu = (m->L.tswap[k] && i > 0) ? 3 - i : i;
        for (int q = 0; q < 4; ++q) dst[12 * u + 4 * iu + q] = (double)h3[12 * k + 4 * i + q];
      }
    }
  };
  const int a = m->cur;
  if (m->fused && !m->d_phi) {
    V4 *p = nullptr;
    R *st = nullptr;
    if ((rc = dev_alloc(m, &p, 3 * nt)) || (rc = dev_alloc(m, &st, nt))) return rc;
    m->d_phi = p;
    m->d_sT = st;
  }
  m->dbg = m->fused;
  for (int pass = 0; pass < 2; ++pass) {
    // pass 0: the LDA residuals (and the stored N residuals); pass 1: the residuals the configured scheme distributes
    if (pass == 0) launch_stage1<R, MRD_SCHEME_LDA>(m, true, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_BX) launch_bx_stage1<R>(m, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_N) launch_stage1<R, MRD_SCHEME_N>(m, true, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_LDA) launch_stage1<R, MRD_SCHEME_LDA>(m, true, a, s);
    else launch_stage1<R, MRD_SCHEME_B>(m, true, a, s);
    CUDA_TRY(cudaMemcpyAsync(h3.data(), m->d_phi, h3.size() * sizeof(R), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    if (pass == 0 && phiLDA) put3(phiLDA);
    if (pass == 1 && phiB) put3(phiB);
  }
  if (m->fused && (phiN || phiT)) {
    // stored stage-1 values of the fused path, phi12[tile][half][N0 | N1 | T][triangle][2] (the cell layout of mrd_tile.cuh),
    // -> the unfused [nt][3][4] / [nt][4] shapes; phi_2^N = (phi^T - phi_0^N) - phi_1^N as both tile kernels form it
    const int T = m->L.tile;
    std::vector<R> h12((size_t)m->L.ntile * 12 * T);
    CUDA_TRY(cudaMemcpy(h12.data(), m->d_phi12, h12.size() * sizeof(R), cudaMemcpyDeviceToHost));
    for (int64_t k = 0; k < nt; ++k) {
      const R *o = &h12[(size_t)(k / T) * 12 * T];
      const int lt = (int)(k % T);
      for (int c = 0; c < 4; ++c) {
        const int h = c >> 1, c2 = c & 1;
        const R n0 = o[((h * 3 + 0) * T + lt) * 2 + c2], n1 = o[((h * 3 + 1) * T + lt) * 2 + c2], pt = o[((h * 3 + 2) * T + lt) * 2 + c2];
        h3[12 * k + c] = n0;
        h3[12 * k + 4 + c] = n1;
        h3[12 * k + 8 + c] = (pt - n0) - n1;
        h1[4 * k + c] = pt;
      }
    }
  }
  if (phiN) {
    if (!m->fused) CUDA_TRY(cudaMemcpy(h3.data(), m->d_phiN, h3.size() * sizeof(R), cudaMemcpyDeviceToHost));
    put3(phiN);
  }
  if (phiT) {
    if (!m->fused) CUDA_TRY(cudaMemcpy(h1.data(), m->d_phiT, h1.size() * sizeof(R), cudaMemcpyDeviceToHost));
    for (int64_t k = 0; k < nt; ++k)
      for (int q = 0; q < 4; ++q) phiT[4 * (int64_t)m->L.tperm[k] + q] = (double)h1[4 * k + q];
  }
  if (sT) {
    CUDA_TRY(cudaMemcpy(hs.data(), m->d_sT, hs.size() * sizeof(R), cudaMemcpyDeviceToHost));
    for (int64_t k = 0; k < nt; ++k) sT[m->L.tperm[k]] = (double)hs[k];
  }
  m->dbg = false;
  int flag = 0;
  CUDA_TRY(cudaMemcpy(&flag, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
  CUDA_TRY(cudaMemcpy(m->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemset(m->d_flag, 0, sizeof(int)));
  if (flag) return fail(MRD_ENONPHYSICAL, "non-physical linearised state");
  return MRD_OK;
}

// sampled variant of dump_impl: only the listed USER triangles are copied back (full-size meshes)
template <class R> int dump_sample_impl(mrd_mesh *m, int64_t ns, const int64_t *ids, double *phiT, double *phiN, double *phiLDA,
                                        double *phiB, double *sT, cudaStream_t s) {
  using V4 = mrd::Vec4<R>;
  const int64_t nt = m->L.nt;
  for (int64_t q = 0; q < ns; ++q)
    if (ids[q] < 0 || ids[q] >= nt) return fail(MRD_EINVAL, "sample triangle id out of range");
  mrd::Ctl c{};
  int rc;
  if ((rc = fetch_ctl(m, s, &c))) return rc;
  mrd::Ctl armed = c;
  armed.active = 1;
  CUDA_TRY(cudaMemcpyAsync(m->d_ctl, &armed, sizeof armed, cudaMemcpyHostToDevice, s));
  if (m->fused && !m->d_phi) {
    V4 *p = nullptr;
    R *st = nullptr;
    if ((rc = dev_alloc(m, &p, 3 * nt)) || (rc = dev_alloc(m, &st, nt))) return rc;
    m->d_phi = p;
    m->d_sT = st;
  }
  m->dbg = m->fused;
  const int a = m->cur;
  R buf[12];
  auto fetch3 = [&](const void *base, int64_t k, int64_t q, double *dst) -> cudaError_t {  // [nt][3][4] layout
    cudaError_t e = cudaMemcpy(buf, (const R *)base + 12 * k, sizeof(R) * 12, cudaMemcpyDeviceToHost);
    for (int i = 0; i < 3; ++i) {
      int iu = (m->L.tswap[k] && i > 0) ? 3 - i : i;
      for (int x = 0; x < 4; ++x) dst[12 * q + 4 * iu + x] = (double)buf[4 * i + x];
    }
    return e;
  };
  for (int pass = 0; pass < 2; ++pass) {
    // pass 0: the LDA residuals (and the stored N residuals); pass 1: the residuals the configured scheme distributes
    if (pass == 0) launch_stage1<R, MRD_SCHEME_LDA>(m, true, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_BX) launch_bx_stage1<R>(m, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_N) launch_stage1<R, MRD_SCHEME_N>(m, true, a, s);
    else if (m->L.p.scheme == MRD_SCHEME_LDA) launch_stage1<R, MRD_SCHEME_LDA>(m, true, a, s);
    else launch_stage1<R, MRD_SCHEME_B>(m, true, a, s);
    CUDA_TRY(cudaStreamSynchronize(s));
    CUDA_TRY(cudaGetLastError());
    double *dst = pass == 0 ? phiLDA : phiB;
    if (dst)
      for (int64_t q = 0; q < ns; ++q) CUDA_TRY(fetch3(m->d_phi, m->L.trank[ids[q]], q, dst));
  }
  m->dbg = false;
  for (int64_t q = 0; q < ns; ++q) {
    const int64_t k = m->L.trank[ids[q]];
    R v16[16];
    if (m->fused) {
      const int T = m->L.tile;
      const int lt = (int)(k % T);
      const R *o = (const R *)m->d_phi12 + (size_t)(k / T) * 12 * T;
      R c6[6][2];   // cells (half, N0 | N1 | T) of this triangle
      for (int hc = 0; hc < 6; ++hc) CUDA_TRY(cudaMemcpy(c6[hc], o + ((size_t)hc * T + lt) * 2, sizeof(R) * 2, cudaMemcpyDeviceToHost));
      for (int c = 0; c < 4; ++c) {
        const int h = c >> 1, c2 = c & 1;
        const R n0 = c6[h * 3 + 0][c2], n1 = c6[h * 3 + 1][c2], pt = c6[h * 3 + 2][c2];
        v16[c] = n0;
        v16[4 + c] = n1;
        v16[8 + c] = (pt - n0) - n1;
        v16[12 + c] = pt;
      }
    } else {
      CUDA_TRY(cudaMemcpy(v16, (const R *)m->d_phiN + 12 * k, sizeof(R) * 12, cudaMemcpyDeviceToHost));
      CUDA_TRY(cudaMemcpy(v16 + 12, (const R *)m->d_phiT + 4 * k, sizeof(R) * 4, cudaMemcpyDeviceToHost));
    }
    if (phiN)
      for (int i = 0; i < 3; ++i) {
        int iu = (m->L.tswap[k] && i > 0) ? 3 - i : i;
        for (int x = 0; x < 4; ++x) phiN[12 * q + 4 * iu + x] = (double)v16[4 * i + x];
      }
    if (phiT)
      for (int x = 0; x < 4; ++x) phiT[4 * q + x] = (double)v16[12 + x];
    if (sT) {
      R v;
      CUDA_TRY(cudaMemcpy(&v, (const R *)m->d_sT + k, sizeof(R), cudaMemcpyDeviceToHost));
      sT[q] = (double)v;
    }
  }
  int flag = 0;
  CUDA_TRY(cudaMemcpy(&flag, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost));
  CUDA_TRY(cudaMemcpy(m->d_ctl, &c, sizeof c, cudaMemcpyHostToDevice));
  CUDA_TRY(cudaMemset(m->d_flag, 0, sizeof(int)));
  if (flag) return fail(MRD_ENONPHYSICAL, "non-physical linearised state");
  return MRD_OK;
}

}  // namespace

extern "C" {

const char *mrd_last_error(void) { return g_err.c_str(); }
// error hook of the other translation units of the library (mrd_meshgen.cu): same thread-local message
int mrd_internal_set_error(int code, const char *msg) { return fail(code, msg ? msg : ""); }
const char *mrd_version(void) { return "mrd 0.1 (sm_100a)"; }

int mrd_layout_create(mrd_layout **out, const mrd_params *p, int64_t nv, const double *xy, int64_t nt,
                      const int32_t *tri, const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge) {
  if (!out) return fail(MRD_EINVAL, "null output pointer");
  mrd_layout *L = new (std::nothrow) mrd_layout();
  if (!L) return fail(MRD_ENOMEM, "out of memory");
  std::string err;
  int rc;
  try {
    rc = mrd_host::layout_build(*L, p, nv, xy, nt, tri, vertex_flag, ne, wall_edge, err);
  } catch (const std::bad_alloc &) {
    rc = MRD_ENOMEM;
    err = "out of host memory in the layout stage";
  }
  if (rc) { delete L; return fail(rc, err); }
  *out = L;
  return MRD_OK;
}
void mrd_layout_destroy(mrd_layout *l) { delete l; }

int mrd_layout_sizes(const mrd_layout *l, int64_t n[6]) {
  if (!l || !n) return fail(MRD_EINVAL, "null argument");
  n[0] = l->nv; n[1] = l->nt; n[2] = l->ne; n[3] = l->nf; n[4] = l->ntile; n[5] = l->nslot;
  return MRD_OK;
}
int mrd_layout_get(const mrd_layout *l, int32_t *vperm, int32_t *tperm, int32_t *tri_int, int32_t *csr_off,
                   int32_t *csr_ent, double *area, double *vol) {
  if (!l) return fail(MRD_EINVAL, "null argument");
  if (vperm) std::memcpy(vperm, l->vperm.data(), sizeof(int32_t) * l->nv);
  if (tperm) std::memcpy(tperm, l->tperm.data(), sizeof(int32_t) * l->nt);
  if (tri_int) std::memcpy(tri_int, l->tri.data(), sizeof(int32_t) * 3 * l->nt);
  if (csr_off) std::memcpy(csr_off, l->csr_off.data(), sizeof(int32_t) * (l->nv + 1));
  if (csr_ent) std::memcpy(csr_ent, l->csr_ent.data(), sizeof(int32_t) * 3 * l->nt);
  if (area) std::memcpy(area, l->area.data(), sizeof(double) * l->nt);
  if (vol) std::memcpy(vol, l->vol.data(), sizeof(double) * l->nv);
  return MRD_OK;
}

int mrd_mesh_create(mrd_mesh **out, const mrd_params *p, int64_t nv, const double *xy, int64_t nt,
                    const int32_t *tri, const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge) {
  if (!out) return fail(MRD_EINVAL, "null output pointer");
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0)
    return fail(MRD_ECUDA, std::string("no CUDA device (there is no CPU fallback): ") + cudaGetErrorString(e));
  mrd_mesh *m = new (std::nothrow) mrd_mesh();
  if (!m) return fail(MRD_ENOMEM, "out of memory");
  std::string err;
  int rc;
  try {
    rc = mrd_host::layout_build(m->L, p, nv, xy, nt, tri, vertex_flag, ne, wall_edge, err);
    if (rc) { delete m; return fail(rc, err); }
    cudaGetDevice(&m->device);
    rc = m->L.p.precision == MRD_FP64 ? upload_impl<double>(m) : upload_impl<float>(m);
  } catch (const std::bad_alloc &) {
    rc = fail(MRD_ENOMEM, "out of host memory");
  }
  if (rc) { mrd_mesh_destroy(m); return rc; }
  // launch-bound regime: below ~4M triangles a step is tens of microseconds, comparable to 6 kernel launches
  if (m->L.nt <= (int64_t(1) << 22)) {
    if (cudaStreamCreateWithFlags(&m->s_int, cudaStreamNonBlocking) == cudaSuccess &&
        cudaEventCreateWithFlags(&m->ev_in, cudaEventDisableTiming) == cudaSuccess &&
        cudaEventCreateWithFlags(&m->ev_out, cudaEventDisableTiming) == cudaSuccess)
      m->graph_ok = true;
  }
  *out = m;
  return MRD_OK;
}

void mrd_mesh_destroy(mrd_mesh *m) {
  if (!m) return;
  for (int k = 0; k < 2; ++k)
    if (m->gexec[k]) cudaGraphExecDestroy(m->gexec[k]);
  if (m->ev_in) cudaEventDestroy(m->ev_in);
  if (m->ev_out) cudaEventDestroy(m->ev_out);
  if (m->s_int) cudaStreamDestroy(m->s_int);
  for (void *p : m->allocs) cudaFree(p);
  if (m->h_pinned) cudaFreeHost(m->h_pinned);
  delete m;
}

int mrd_mesh_device_bytes(const mrd_mesh *m, int64_t *bytes) {
  if (!m || !bytes) return fail(MRD_EINVAL, "null argument");
  *bytes = m->dev_bytes;
  return MRD_OK;
}

int mrd_set_state(mrd_mesh *m, const void *W_dev, void *stream) {
  if (!m || !W_dev) return fail(MRD_EINVAL, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? set_state_impl<double>(m, (const double *)W_dev, s)
                                      : set_state_impl<float>(m, (const float *)W_dev, s);
}

int mrd_set_state_host(mrd_mesh *m, const void *W_host, void *stream) {
  if (!m || !W_host) return fail(MRD_EINVAL, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  size_t bytes = (size_t)4 * m->L.nv * (m->L.p.precision == MRD_FP64 ? 8 : 4);
  CUDA_TRY(cudaMemcpyAsync(m->d_user, W_host, bytes, cudaMemcpyHostToDevice, s));
  return mrd_set_state(m, m->d_user, stream);
}

int mrd_get_state(mrd_mesh *m, void *W_out_dev, void *stream) {
  if (!m || !W_out_dev) return fail(MRD_EINVAL, "null argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  cudaStream_t s = (cudaStream_t)stream;
  mrd::Ctl c{};
  int rc = fetch_ctl(m, s, &c);  // settles the buffer parity after async steps
  if (rc) return rc;
  return m->L.p.precision == MRD_FP64 ? get_state_impl<double>(m, (double *)W_out_dev, s)
                                      : get_state_impl<float>(m, (float *)W_out_dev, s);
}

int mrd_get_state_host(mrd_mesh *m, void *W_out_host, void *stream) {
  if (!m || !W_out_host) return fail(MRD_EINVAL, "null argument");
  int rc = mrd_get_state(m, m->d_user, stream);
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  size_t bytes = (size_t)4 * m->L.nv * (m->L.p.precision == MRD_FP64 ? 8 : 4);
  CUDA_TRY(cudaMemcpyAsync(W_out_host, m->d_user, bytes, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(cudaStreamSynchronize(s));
  return MRD_OK;
}

int mrd_step(mrd_mesh *m, int64_t max_steps, double t_end, void *stream, int64_t *steps_done, double *t, double *dt_last) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? step_impl<double>(m, max_steps, t_end, s, true, steps_done, t, dt_last)
                                      : step_impl<float>(m, max_steps, t_end, s, true, steps_done, t, dt_last);
}

int mrd_step_async(mrd_mesh *m, int64_t n_steps, void *stream) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? step_impl<double>(m, n_steps, 0.0, s, false, nullptr, nullptr, nullptr)
                                      : step_impl<float>(m, n_steps, 0.0, s, false, nullptr, nullptr, nullptr);
}

int mrd_sync(mrd_mesh *m, void *stream, int64_t *steps_total, double *t, double *dt_last) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  mrd::Ctl c{};
  int rc = fetch_ctl(m, (cudaStream_t)stream, &c);
  if (rc) return rc;
  if (steps_total) *steps_total = c.steps;
  if (t) *t = c.t;
  if (dt_last) *dt_last = c.dt;
  if (c.status) return discard_failed_step(m, c, (cudaStream_t)stream);
  return MRD_OK;
}

int mrd_get_diagnostics(mrd_mesh *m, double totals[4], double *min_rho, double *min_p, void *stream) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  cudaStream_t s = (cudaStream_t)stream;
  mrd::Ctl c{};
  int rc = fetch_ctl(m, s, &c);
  if (rc) return rc;
  return m->L.p.precision == MRD_FP64 ? diag_impl<double>(m, totals, min_rho, min_p, s) : diag_impl<float>(m, totals, min_rho, min_p, s);
}

int mrd_dump_stage1(mrd_mesh *m, double *phiT, double *phiN, double *phiLDA, double *phiB, double *sT, void *stream) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? dump_impl<double>(m, phiT, phiN, phiLDA, phiB, sT, s)
                                      : dump_impl<float>(m, phiT, phiN, phiLDA, phiB, sT, s);
}

int mrd_dump_stage1_sample(mrd_mesh *m, int64_t n_sample, const int64_t *tri_user, double *phiT, double *phiN, double *phiLDA,
                           double *phiB, double *sT, void *stream) {
  if (!m || (n_sample > 0 && !tri_user) || n_sample < 0) return fail(MRD_EINVAL, "bad argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? dump_sample_impl<double>(m, n_sample, tri_user, phiT, phiN, phiLDA, phiB, sT, s)
                                      : dump_sample_impl<float>(m, n_sample, tri_user, phiT, phiN, phiLDA, phiB, sT, s);
}

int mrd_step_profile(mrd_mesh *m, void *stream, float ms[MRD_PROFILE_SLOTS]) {
  if (!m || !ms) return fail(MRD_EINVAL, "null argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  cudaStream_t s = (cudaStream_t)stream;
  mrd::Ctl c{};
  int rc = fetch_ctl(m, s, &c);
  if (rc) return rc;
  if (c.status) return fail(MRD_ENONPHYSICAL, "state is non-physical (an earlier step failed)");
  Prof prof;
  const int nev = MRD_PROFILE_SLOTS + 2;
  for (int k = 0; k < nev; ++k) CUDA_TRY(cudaEventCreate(&prof.ev[k]));
  mrd::ctl_kernel<<<1, 1, 0, s>>>(m->d_ctl, 0, 0.0, m->d_flag);
  m->launches++;
  prof.mark(-1, s);
  if (m->L.p.precision == MRD_FP64) enqueue_step<double>(m, m->L.p.scheme, m->cur, s, &prof);
  else enqueue_step<float>(m, m->L.p.scheme, m->cur, s, &prof);
  rc = take_launch_rc(m);
  if (!rc) rc = fetch_ctl(m, s, &c);
  for (int k = 0; k < MRD_PROFILE_SLOTS; ++k) ms[k] = 0.f;
  if (!rc)
    for (int k = 1; k < prof.n; ++k) {
      float t = 0.f;
      cudaEventElapsedTime(&t, prof.ev[k - 1], prof.ev[k]);
      ms[prof.slot[k]] += t;
    }
  for (int k = 0; k < nev; ++k) cudaEventDestroy(prof.ev[k]);
  if (rc) return rc;
  if (c.status) return fail(MRD_ENONPHYSICAL, "non-physical state met in the profiled step");
  return MRD_OK;
}

int mrd_partition_create(mrd_partition **out, int64_t nv, const double *xy, int64_t nt, const int32_t *tri,
                         const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge, double period_x, double period_y,
                         int32_t n_part, int32_t part) {
  if (!out) return fail(MRD_EINVAL, "null output pointer");
  mrd_partition *P = new (std::nothrow) mrd_partition();
  if (!P) return fail(MRD_ENOMEM, "out of memory");
  std::string err;
  int rc;
  try {
    rc = mrd_host::partition_build(*P, nv, xy, nt, tri, vertex_flag, ne, wall_edge, period_x, period_y, n_part, part, nullptr, err);
  } catch (const std::bad_alloc &) {
    rc = MRD_ENOMEM;
    err = "out of host memory in the partitioner";
  }
  if (rc) { delete P; return fail(rc, err); }
  *out = P;
  return MRD_OK;
}
int mrd_partition_create_owned(mrd_partition **out, int64_t nv, const double *xy, int64_t nt, const int32_t *tri,
                               const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge, double period_x, double period_y,
                               int32_t n_part, int32_t part, const int32_t *owner) {
  if (!out || !owner) return fail(MRD_EINVAL, "null argument");
  mrd_partition *P = new (std::nothrow) mrd_partition();
  if (!P) return fail(MRD_ENOMEM, "out of memory");
  std::string err;
  int rc;
  try {
    rc = mrd_host::partition_build(*P, nv, xy, nt, tri, vertex_flag, ne, wall_edge, period_x, period_y, n_part, part, owner, err);
  } catch (const std::bad_alloc &) {
    rc = MRD_ENOMEM;
    err = "out of host memory in the partitioner";
  }
  if (rc) { delete P; return fail(rc, err); }
  *out = P;
  return MRD_OK;
}
int mrd_partition_create_local(mrd_partition **out, int64_t nv_global, double domain_size, int64_t n_local_vertex,
                               const int32_t *vertex_global, const int32_t *owner, const double *xy, const uint8_t *vertex_flag,
                               int64_t n_local_triangle, const int32_t *tri, const int32_t *tri_global, int64_t n_wall_edge,
                               const int32_t *wall_edge, int32_t n_part, int32_t part) {
  if (!out) return fail(MRD_EINVAL, "null output pointer");
  mrd_partition *P = new (std::nothrow) mrd_partition();
  if (!P) return fail(MRD_ENOMEM, "out of memory");
  std::string err;
  int rc;
  try {
    rc = mrd_host::partition_build_local(*P, nv_global, domain_size, n_local_vertex, vertex_global, owner, xy, vertex_flag,
                                         n_local_triangle, tri, tri_global, n_wall_edge, wall_edge, n_part, part, err);
  } catch (const std::bad_alloc &) {
    rc = MRD_ENOMEM;
    err = "out of host memory in the partitioner";
  }
  if (rc) { delete P; return fail(rc, err); }
  *out = P;
  return MRD_OK;
}
void mrd_partition_destroy(mrd_partition *p) { delete p; }
int mrd_partition_domain_size(const mrd_partition *p, double *L) {
  if (!p || !L) return fail(MRD_EINVAL, "null argument");
  *L = p->domain_size;
  return MRD_OK;
}
int mrd_partition_sizes(const mrd_partition *p, int64_t n[8]) {
  if (!p || !n) return fail(MRD_EINVAL, "null argument");
  return mrd_host::partition_sizes(*p, n);
}
int mrd_partition_get(const mrd_partition *p, const char *name, void *dst, int64_t bytes) {
  if (!p) return fail(MRD_EINVAL, "null argument");
  std::string err;
  int rc = mrd_host::partition_get(*p, name, dst, bytes, err);
  return rc ? fail(rc, err) : MRD_OK;
}

int mrd_halo_set(mrd_mesh *m, int64_t n_send, const int32_t *send_idx, int64_t n_recv, const int32_t *recv_idx) {
  if (!m || n_send < 0 || n_recv < 0 || (n_send > 0 && !send_idx) || (n_recv > 0 && !recv_idx)) return fail(MRD_EINVAL, "bad halo lists");
  if (m->in_phases) return fail(MRD_EINVAL, "mrd_halo_set inside mrd_phase_begin / mrd_phase_end");
  const int64_t nv = m->L.nv;
  std::vector<int32_t> si((size_t)n_send), ri((size_t)n_recv);
  for (int64_t k = 0; k < n_send; ++k) {
    if (send_idx[k] < 0 || send_idx[k] >= nv) return fail(MRD_EINVAL, "halo send index out of range");
    si[k] = m->L.vrank[send_idx[k]];
    if (m->L.frozen[si[k]] == 2) return fail(MRD_EINVAL, "halo send list names a halo vertex");
  }
  for (int64_t k = 0; k < n_recv; ++k) {
    if (recv_idx[k] < 0 || recv_idx[k] >= nv) return fail(MRD_EINVAL, "halo receive index out of range");
    ri[k] = m->L.vrank[recv_idx[k]];
    if (m->L.frozen[ri[k]] != 2) return fail(MRD_EINVAL, "halo receive list names a vertex that is not flagged 2 (halo)");
  }
  int rc;
  if ((rc = dev_upload(m, &m->d_send_idx, si.data(), n_send))) return rc;
  if ((rc = dev_upload(m, &m->d_recv_idx, ri.data(), n_recv))) return rc;
  m->n_send = n_send;
  m->n_recv = n_recv;
  return MRD_OK;
}

int mrd_phase_begin(mrd_mesh *m, double t_end, void *stream) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  if (!m->has_state) return fail(MRD_EINVAL, "no state set");
  if (m->in_phases) return fail(MRD_EINVAL, "mrd_phase_begin called twice");
  cudaStream_t s = (cudaStream_t)stream;
  mrd::Ctl c{};
  int rc = fetch_ctl(m, s, &c);
  if (rc) return rc;
  if (c.status) return fail(MRD_ENONPHYSICAL, "state is non-physical (an earlier step failed)");
  mrd::ctl_kernel<<<1, 1, 0, s>>>(m->d_ctl, 0, t_end > 0.0 ? t_end : 0.0, m->d_flag);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  m->in_phases = true;
  m->phase_a = m->cur;
  m->phase_next = MRD_PHASE_RESIDUAL1;
  m->phase_steps0 = c.steps;
  return MRD_OK;
}

int mrd_phase(mrd_mesh *m, int32_t phase, void *stream) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases) return fail(MRD_EINVAL, "mrd_phase outside mrd_phase_begin / mrd_phase_end");
  if (phase != m->phase_next) return fail(MRD_EINVAL, "phases out of order (RESIDUAL1, UPDATE1, [STAGE2], END)");
  cudaStream_t s = (cudaStream_t)stream;
  int rc = m->L.p.precision == MRD_FP64 ? phase_impl<double>(m, phase, s) : phase_impl<float>(m, phase, s);
  if (rc) return rc;
  if (phase == MRD_PHASE_END) {
    m->phase_a ^= 1;
    m->phase_next = MRD_PHASE_RESIDUAL1;
  } else if (phase == MRD_PHASE_UPDATE1 && m->L.p.time_order == 1) {
    m->phase_next = MRD_PHASE_END;
  } else {
    m->phase_next = phase + 1;
  }
  return MRD_OK;
}

int mrd_phase_end(mrd_mesh *m, void *stream, int64_t *steps_done, double *t, double *dt_last) {
  if (!m) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases) return fail(MRD_EINVAL, "mrd_phase_end without mrd_phase_begin");
  if (m->phase_next != MRD_PHASE_RESIDUAL1) return fail(MRD_EINVAL, "mrd_phase_end in the middle of a step");
  m->in_phases = false;
  cudaStream_t s = (cudaStream_t)stream;
  mrd::Ctl c{};
  int rc = fetch_ctl(m, s, &c);
  if (rc) return rc;
  if (steps_done) *steps_done = c.steps - m->phase_steps0;
  if (t) *t = c.t;
  if (dt_last) *dt_last = c.dt;
  if (c.status) return discard_failed_step(m, c, s);
  return MRD_OK;
}

int mrd_dt_get(mrd_mesh *m, double *d_dev, void *stream) {
  if (!m || !d_dev) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || m->phase_next != MRD_PHASE_UPDATE1) return fail(MRD_EINVAL, "mrd_dt_get must follow mrd_phase(RESIDUAL1)");
  mrd::dt_get_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(m->d_ctl, m->d_flag, d_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}
int mrd_dt_set(mrd_mesh *m, const double *d_dev, void *stream) {
  if (!m || !d_dev) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || m->phase_next != MRD_PHASE_UPDATE1) return fail(MRD_EINVAL, "mrd_dt_set must follow mrd_phase(RESIDUAL1)");
  mrd::dt_set_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(m->d_ctl, m->d_flag, d_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}

int mrd_status_get(mrd_mesh *m, double *d_dev, void *stream) {
  if (!m || !d_dev) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || m->phase_next != MRD_PHASE_END) return fail(MRD_EINVAL, "mrd_status_get must precede mrd_phase(END)");
  mrd::status_get_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(m->d_ctl, m->d_flag, d_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}
int mrd_status_set(mrd_mesh *m, const double *d_dev, void *stream) {
  if (!m || !d_dev) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || m->phase_next != MRD_PHASE_END) return fail(MRD_EINVAL, "mrd_status_set must precede mrd_phase(END)");
  mrd::status_set_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(m->d_flag, d_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}

int mrd_range_get(mrd_mesh *m, int32_t stage, double *d_dev, void *stream) {
  if (!m || !d_dev || (stage != 1 && stage != 2)) return fail(MRD_EINVAL, "bad argument");
  if (!m->in_phases) return fail(MRD_EINVAL, "mrd_range_get outside mrd_phase_begin / mrd_phase_end");
  cudaStream_t s = (cudaStream_t)stream;
  // stage 1: the state the next RESIDUAL1 reads (W^n); stage 2: W* written by UPDATE1 (and the halo unpack after it)
  const int pair = stage == 1 ? m->phase_a : (m->phase_a ^ 1);
  const unsigned vb = blocks_for(m->L.nv, 256), nb = std::min<unsigned>(vb, (unsigned)m->nsm * 8);
  mrd::range_reset_kernel<<<1, 1, 0, s>>>(m->d_ctl, stage - 1);
  if (m->L.p.precision == MRD_FP64)
    mrd::vrange_kernel<double><<<nb, 256, 0, s>>>(m->L.nv, (const mrd::Vec4<double> *)m->d_W[pair], m->d_ctl, stage - 1);
  else
    mrd::vrange_kernel<float><<<nb, 256, 0, s>>>(m->L.nv, (const mrd::Vec4<float> *)m->d_W[pair], m->d_ctl, stage - 1);
  mrd::range_get_kernel<<<1, 1, 0, s>>>(m->d_ctl, stage - 1, d_dev);
  m->launches += 3;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}
int mrd_range_set(mrd_mesh *m, int32_t stage, const double *d_dev, void *stream) {
  if (!m || !d_dev || (stage != 1 && stage != 2)) return fail(MRD_EINVAL, "bad argument");
  if (!m->in_phases) return fail(MRD_EINVAL, "mrd_range_set outside mrd_phase_begin / mrd_phase_end");
  mrd::range_set_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(m->d_ctl, stage - 1, d_dev);
  m->launches++;
  CUDA_TRY(cudaGetLastError());
  return MRD_OK;
}

int mrd_halo_pack(mrd_mesh *m, void *buf_dev, void *stream) {
  if (!m || (m->n_send > 0 && !buf_dev)) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || (m->phase_next != MRD_PHASE_STAGE2 && m->phase_next != MRD_PHASE_END))
    return fail(MRD_EINVAL, "mrd_halo_pack must follow mrd_phase(UPDATE1) or mrd_phase(STAGE2)");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? halo_pack_impl<double>(m, buf_dev, s) : halo_pack_impl<float>(m, buf_dev, s);
}
int mrd_halo_unpack(mrd_mesh *m, const void *buf_dev, void *stream) {
  if (!m || (m->n_recv > 0 && !buf_dev)) return fail(MRD_EINVAL, "null argument");
  if (!m->in_phases || (m->phase_next != MRD_PHASE_STAGE2 && m->phase_next != MRD_PHASE_END))
    return fail(MRD_EINVAL, "mrd_halo_unpack must follow mrd_phase(UPDATE1) or mrd_phase(STAGE2)");
  cudaStream_t s = (cudaStream_t)stream;
  return m->L.p.precision == MRD_FP64 ? halo_unpack_impl<double>(m, buf_dev, s) : halo_unpack_impl<float>(m, buf_dev, s);
}

int mrd_launch_count(const mrd_mesh *m, int64_t *launches) {
  if (!m || !launches) return fail(MRD_EINVAL, "null argument");
  *launches = m->launches;
  return MRD_OK;
}

int mrd_measure_peaks(double *fp64_tflops, double *fp32_tflops, double *copy_gbs, void *stream) {
  cudaStream_t s = (cudaStream_t)stream;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(MRD_ECUDA, "no CUDA device");
  cudaDeviceProp prop;
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  cudaEvent_t e0, e1;
  CUDA_TRY(cudaEventCreate(&e0));
  CUDA_TRY(cudaEventCreate(&e1));
  const int blocks = prop.multiProcessorCount * 8, threads = 256;
  double *scratch = nullptr;
  CUDA_TRY(cudaMalloc(&scratch, (size_t)blocks * threads * sizeof(double)));
  float ms = 0.f;
  auto best_of = [&](auto launch, int reps, float &best) -> cudaError_t {
    best = 1e30f;
    for (int r = 0; r < reps; ++r) {
      cudaEventRecord(e0, s);
      launch();
      cudaEventRecord(e1, s);
      cudaError_t e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) return e;
      float t;
      cudaEventElapsedTime(&t, e0, e1);
      if (r > 0 && t < best) best = t;
    }
    return cudaGetLastError();
  };
  if (fp64_tflops) {
    const int iters = 4096;
    CUDA_TRY(best_of([&] { mrd::fma_peak_kernel<double><<<blocks, threads, 0, s>>>(scratch, iters, 0.999999, 1e-7); }, 4, ms));
    *fp64_tflops = 2.0 * 64.0 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-12;
  }
  if (fp32_tflops) {
    const int iters = 8192;
    CUDA_TRY(best_of([&] { mrd::fma_peak_kernel<float><<<blocks, threads, 0, s>>>((float *)scratch, iters, 0.999999f, 1e-7f); }, 4, ms));
    *fp32_tflops = 2.0 * 64.0 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-12;
  }
  cudaFree(scratch);
  if (copy_gbs) {
    const int64_t n = (int64_t)1 << 26;  // 2 x 1 GiB
    double2 *a = nullptr, *b = nullptr;
    CUDA_TRY(cudaMalloc(&a, n * sizeof(double2)));
    CUDA_TRY(cudaMalloc(&b, n * sizeof(double2)));
    CUDA_TRY(cudaMemsetAsync(a, 0, n * sizeof(double2), s));
    CUDA_TRY(best_of([&] { mrd::copy_kernel<<<prop.multiProcessorCount * 16, 256, 0, s>>>(a, b, n); }, 5, ms));
    *copy_gbs = 2.0 * n * sizeof(double2) / (ms * 1e-3) * 1e-9;
    cudaFree(a);
    cudaFree(b);
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return MRD_OK;
}

}  // extern "C"
