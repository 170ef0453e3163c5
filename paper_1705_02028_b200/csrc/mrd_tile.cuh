// mrd_tile.cuh -- the fused tile kernels (the production path): one thread block owns a run of
// `tile` consecutive (Morton-ordered) triangles.
//
//   prologue : the block's tile-local vertices ("slots", mrd_layout.h) are staged in shared memory ONCE:
//              parameter vector Z, signal speed, tile-frame coordinates (stage 2 also dW/dt)
//   body     : one thread per triangle; geometry of eq. 35 (L397-L399) from the staged coordinates,
//              then S2-S5 / S9 of SURVEY 8a exactly as the unfused kernels (same device functions)
//   epilogue : the distributed residuals go to shared memory and every slot sums its incident
//              (triangle, node) entries in ascending order -> ONE partial per slot leaves the SM, instead
//              of three 4-vectors per triangle (no float atomics, deterministic; replaces L734)
// The vertex kernels then add a vertex's few partials (ascending slot = ascending triangle order).
#pragma once
#include "mrd_kernels.cuh"

namespace mrd {

template <class R> struct TileDev {
  int32_t tile;
  int64_t ntile, nslot, nt;
  const int32_t *tile_slot_off;  // [ntile+1]
  const int32_t *slot_vertex;    // [nslot]
  const R *slot_xy;              // [nslot][2], relative to the tile's first slot
  const ushort4 *tile_tri;       // [ntile*tile]: tile-local slot of nodes 0..2
  const int32_t *slot_ent_off;   // [nslot+1]
  const uint16_t *slot_ent;      // [3 nt]: (local triangle)*4 + node, ascending
  const int32_t *vslot_off;      // [nv+1]
  const int32_t *vslot_ent;      // [nslot]
};

// geometry of one CCW triangle from its vertex coordinates (eq. 35; reading C4):
// the edge opposite node i runs from node i+1 to node i+2, inward normal (-e_y, e_x)
template <class R>
__device__ __forceinline__ void tile_geometry(const R x[3], const R y[3], TriGeom<R> &g, R &area3, R &lmax) {
  using F = Fast<R>;
  R hmax = R(0);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const int a = (i + 1) % 3, b = (i + 2) % 3;
    R ex = x[b] - x[a], ey = y[b] - y[a];
    R l2 = ex * ex + ey * ey;
    R rl = F::rsqrt(l2);
    g.nx[i] = -ey * rl;
    g.ny[i] = ex * rl;
    g.hl[i] = R(0.5) * (l2 * rl);
    hmax = F::max(hmax, g.hl[i]);
  }
  lmax = R(2) * hmax;
  area3 = ((x[1] - x[0]) * (y[2] - y[0]) - (y[1] - y[0]) * (x[2] - x[0])) * (R(1) / R(6));
}

// shared-memory carve-up (dynamic): all arrays sized for the worst case of 3*tile slots
template <class R> struct TileSmem {
  Vec4<R> *Z;   // [3T]
  Vec4<R> *D;   // [3T]  (stage 2: dW/dt)
  R *X, *Y;     // [3T]
  R *spd;       // [3T]  (stage 1)
  R *res;       // [12][T]  component-major distributed residuals
  R *sT;        // [T]
  __device__ TileSmem(unsigned char *base, int T, bool stage2) {
    Z = reinterpret_cast<Vec4<R> *>(base);
    unsigned char *p = base + sizeof(Vec4<R>) * 3 * T;
    if (stage2) { D = reinterpret_cast<Vec4<R> *>(p); p += sizeof(Vec4<R>) * 3 * T; } else { D = nullptr; }
    X = reinterpret_cast<R *>(p); p += sizeof(R) * 3 * T;
    Y = reinterpret_cast<R *>(p); p += sizeof(R) * 3 * T;
    spd = reinterpret_cast<R *>(p); p += sizeof(R) * 3 * T;
    res = reinterpret_cast<R *>(p); p += sizeof(R) * 12 * T;
    sT = reinterpret_cast<R *>(p);
  }
  static size_t bytes(int T, bool stage2) {
    return sizeof(Vec4<R>) * 3 * T * (stage2 ? 2 : 1) + sizeof(R) * (9 * T + 12 * T + T);
  }
};

// epilogue shared by both stages: per slot, ascending sum of its tile-local incidences
template <class R, bool WITH_ST>
__device__ __forceinline__ void tile_epilogue(const TileDev<R> &td, const TileSmem<R> &sm, int s0, int ns,
                                              Vec4<R> *__restrict__ part, R *__restrict__ partS) {
  const int T = blockDim.x;
  for (int j = threadIdx.x; j < ns; j += T) {
    const int32_t q0 = __ldg(td.slot_ent_off + s0 + j), q1 = __ldg(td.slot_ent_off + s0 + j + 1);
    R a0 = 0, a1 = 0, a2 = 0, a3 = 0, S = 0;
    for (int32_t q = q0; q < q1; ++q) {
      const int e = __ldg(td.slot_ent + q);
      const int lt = e >> 2, nd = e & 3;
      const R *r = sm.res + (nd * 4) * T + lt;
      a0 += r[0];
      a1 += r[T];
      a2 += r[2 * T];
      a3 += r[3 * T];
      if (WITH_ST) S += sm.sT[lt];
    }
    st4(&part[s0 + j], Vec4<R>{a0, a1, a2, a3});
    if (WITH_ST) partS[s0 + j] = S;
  }
}

template <class R, int SCHEME, bool STORE>
__global__ void __launch_bounds__(256)
tile_stage1_kernel(TileDev<R> td, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Z,
                   const R *__restrict__ spd, Vec4<R> *__restrict__ part, R *__restrict__ partS,
                   Vec4<R> *__restrict__ phiN_n, Vec4<R> *__restrict__ phiT_n, Vec4<R> *__restrict__ phi_dbg,
                   R *__restrict__ sT_dbg, int *status) {
  MRD_CTL_GUARD(ctl)
  extern __shared__ __align__(32) unsigned char smem_raw[];
  const int T = blockDim.x, tid = threadIdx.x;
  TileSmem<R> sm(smem_raw, T, false);
  const int64_t b = blockIdx.x;
  const int s0 = __ldg(td.tile_slot_off + b), ns = __ldg(td.tile_slot_off + b + 1) - s0;
  for (int j = tid; j < ns; j += T) {
    const int32_t v = __ldg(td.slot_vertex + s0 + j);
    sm.Z[j] = ld4(&Z[v]);
    sm.spd[j] = __ldg(spd + v);
    sm.X[j] = __ldg(td.slot_xy + 2 * (int64_t)(s0 + j));
    sm.Y[j] = __ldg(td.slot_xy + 2 * (int64_t)(s0 + j) + 1);
  }
  __syncthreads();
  const int64_t t = b * T + tid;
  R pN[3][4];
  R st = R(0);
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int c = 0; c < 4; ++c) pN[i][c] = R(0);
  if (t < td.nt) {
    const ushort4 lv = __ldg(td.tile_tri + t);
    const int l[3] = {lv.x, lv.y, lv.z};
    Vec4<R> z[3] = {sm.Z[l[0]], sm.Z[l[1]], sm.Z[l[2]]};
    R x[3] = {sm.X[l[0]], sm.X[l[1]], sm.X[l[2]]}, y[3] = {sm.Y[l[0]], sm.Y[l[1]], sm.Y[l[2]]};
    TriGeom<R> g;
    R area3, lmax;
    tile_geometry(x, y, g, area3, lmax);
    st = lmax * Fast<R>::max(sm.spd[l[0]], Fast<R>::max(sm.spd[l[1]], sm.spd[l[2]]));  // eq. 44-45
    TriCore<R> k;
    R pT[4];
    triangle_core(gamma, z, g, k, pT, pN);
    if (!k.ok) atomicOr(status, 1);
    if (STORE) {
      st4(&phiT_n[t], Vec4<R>{pT[0], pT[1], pT[2], pT[3]});
#pragma unroll
      for (int i = 0; i < 3; ++i) st4(&phiN_n[3 * t + i], Vec4<R>{pN[i][0], pN[i][1], pN[i][2], pN[i][3]});
    }
    if (SCHEME != MRD_SCHEME_N) {
      R pL[3][4];
      apply_beta(gamma, k, g, pT, pL);
      if (SCHEME == MRD_SCHEME_B) {
        blend(pT, pN, pL);
      } else {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
          for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c];
      }
    }
    if (phi_dbg) {
#pragma unroll
      for (int i = 0; i < 3; ++i) st4(&phi_dbg[3 * t + i], Vec4<R>{pN[i][0], pN[i][1], pN[i][2], pN[i][3]});
      sT_dbg[t] = st;
    }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int c = 0; c < 4; ++c) sm.res[(i * 4 + c) * T + tid] = pN[i][c];
  sm.sT[tid] = st;
  __syncthreads();
  tile_epilogue<R, true>(td, sm, s0, ns, part, partS);
}

template <class R, int SCHEME>
__global__ void __launch_bounds__(256)
tile_stage2_kernel(TileDev<R> td, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Zs,
                   const Vec4<R> *__restrict__ dWdt, const Vec4<R> *__restrict__ phiN_n,
                   const Vec4<R> *__restrict__ phiT_n, Vec4<R> *__restrict__ part, int *status) {
  MRD_CTL_GUARD(ctl)
  extern __shared__ __align__(32) unsigned char smem_raw[];
  const int T = blockDim.x, tid = threadIdx.x;
  TileSmem<R> sm(smem_raw, T, true);
  const int64_t b = blockIdx.x;
  const int s0 = __ldg(td.tile_slot_off + b), ns = __ldg(td.tile_slot_off + b + 1) - s0;
  for (int j = tid; j < ns; j += T) {
    const int32_t v = __ldg(td.slot_vertex + s0 + j);
    sm.Z[j] = ld4(&Zs[v]);
    sm.D[j] = ld4(&dWdt[v]);
    sm.X[j] = __ldg(td.slot_xy + 2 * (int64_t)(s0 + j));
    sm.Y[j] = __ldg(td.slot_xy + 2 * (int64_t)(s0 + j) + 1);
  }
  __syncthreads();
  const int64_t t = b * T + tid;
  R pN[3][4];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int c = 0; c < 4; ++c) pN[i][c] = R(0);
  if (t < td.nt) {
    const ushort4 lv = __ldg(td.tile_tri + t);
    const int l[3] = {lv.x, lv.y, lv.z};
    Vec4<R> z[3] = {sm.Z[l[0]], sm.Z[l[1]], sm.Z[l[2]]};
    R x[3] = {sm.X[l[0]], sm.X[l[1]], sm.X[l[2]]}, y[3] = {sm.Y[l[0]], sm.Y[l[1]], sm.Y[l[2]]};
    TriGeom<R> g;
    R a3, lmax;
    tile_geometry(x, y, g, a3, lmax);
    TriCore<R> k;
    R pT[4];
    triangle_core(gamma, z, g, k, pT, pN);  // all matrices re-evaluated at W* (reading C12)
    if (!k.ok) atomicOr(status, 1);
    // eq. 57 / 61: Phi^T = |T|/3 sum_j dW_j/dt + (phi^T(W^n) + phi^T(W*))/2;  eq. 62 per node
    R PT[4];
    {
      Vec4<R> o = ld4(&phiT_n[t]);
      PT[0] = R(0.5) * (o.x + pT[0]); PT[1] = R(0.5) * (o.y + pT[1]);
      PT[2] = R(0.5) * (o.z + pT[2]); PT[3] = R(0.5) * (o.w + pT[3]);
    }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      Vec4<R> d = sm.D[l[i]];
      Vec4<R> o = ld4(&phiN_n[3 * t + i]);
      R m0 = a3 * d.x, m1 = a3 * d.y, m2 = a3 * d.z, m3 = a3 * d.w;
      PT[0] += m0; PT[1] += m1; PT[2] += m2; PT[3] += m3;
      pN[i][0] = m0 + R(0.5) * (pN[i][0] + o.x);
      pN[i][1] = m1 + R(0.5) * (pN[i][1] + o.y);
      pN[i][2] = m2 + R(0.5) * (pN[i][2] + o.z);
      pN[i][3] = m3 + R(0.5) * (pN[i][3] + o.w);
    }
    if (SCHEME != MRD_SCHEME_N) {
      R pL[3][4];
      apply_beta(gamma, k, g, PT, pL);  // eq. 63 with eq. 65
      if (SCHEME == MRD_SCHEME_B) {
        blend(PT, pN, pL);
      } else {
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
          for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c];
      }
    }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int c = 0; c < 4; ++c) sm.res[(i * 4 + c) * T + tid] = pN[i][c];
  __syncthreads();
  tile_epilogue<R, false>(td, sm, s0, ns, part, nullptr);
}

// ---------------------------------------------------------------------------------------------
// vertex side of the fused path: add the vertex's partials (ascending slot order)
// ---------------------------------------------------------------------------------------------
template <class R>
__global__ void __launch_bounds__(256)
slot_gather_dt_kernel(MeshDev<R> m, TileDev<R> td, Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ part,
                      const R *__restrict__ partS, Vec4<R> *__restrict__ acc) {
  MRD_CTL_GUARD(ctl)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double d = __longlong_as_double(0x7FF0000000000000ll);
  if (i < m.nv) {
    R a0 = 0, a1 = 0, a2 = 0, a3 = 0, S = 0;
    const int32_t q0 = __ldg(td.vslot_off + i), q1 = __ldg(td.vslot_off + i + 1);
    for (int32_t q = q0; q < q1; ++q) {
      const int32_t s = __ldg(td.vslot_ent + q);
      Vec4<R> f = ld4(&part[s]);
      a0 += f.x; a1 += f.y; a2 += f.z; a3 += f.w;
      S += __ldg(partS + s);
    }
    st4(&acc[i], Vec4<R>{a0, a1, a2, a3});
    d = 2.0 * (double)__ldg(m.vol + i) / (double)S;  // eq. 44
  }
  block_min_to_global(d, &ctl->dmin_bits);
}

template <class R>
__global__ void __launch_bounds__(256)
slot_gather_update_kernel(MeshDev<R> m, TileDev<R> td, R gamma, const Ctl *__restrict__ ctl,
                          const Vec4<R> *__restrict__ part, const Vec4<R> *__restrict__ wall_acc,
                          Vec4<R> *__restrict__ Ws, Vec4<R> *__restrict__ Zs, R *__restrict__ spd, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m.nv) return;
  R a[4] = {0, 0, 0, 0};
  const int32_t q0 = __ldg(td.vslot_off + i), q1 = __ldg(td.vslot_off + i + 1);
  for (int32_t q = q0; q < q1; ++q) {
    Vec4<R> f = ld4(&part[__ldg(td.vslot_ent + q)]);
    a[0] += f.x; a[1] += f.y; a[2] += f.z; a[3] += f.w;
  }
  if (wall_acc) {
    Vec4<R> f = wall_acc[i];
    a[0] += f.x; a[1] += f.y; a[2] += f.z; a[3] += f.w;
  }
  R dt = (R)ctl_dt(ctl);
  Vec4<R> w = Ws[i];
  bool fr = m.frozen ? (m.frozen[i] != 0) : false;
  vertex_finish<R, false>(gamma, dt, __ldg(m.vol + i), fr, w, a, w, &Ws[i], &Zs[i], &spd[i], nullptr, status);
}

}  // namespace mrd
