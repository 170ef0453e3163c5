// mrd_kernels.cuh -- sm_100a kernels of the sweep: triangle residual/distribution (two stages),
// vertex gather + update, CFL reduction, wall terms, state I/O, diagnostics.  R = double | float.
#pragma once
#include <cstdint>

#include "mrd_math.cuh"

namespace mrd {

// Device-resident step control (no host round trip inside a multi-step call).
struct Ctl {
  double t;                      // current time
  double dt;                     // time step of the step in flight / last step
  double t_end;                  // <= 0: none
  double cfl;
  unsigned long long dmin_bits;  // bit pattern of min_i 2 V_i / sum s_T (positive double) of the step in flight
  long long steps;               // completed steps since set_state
  int status;                    // 0, or MRD_ENONPHYSICAL (as positive flag 1)
  int active;                    // 1 while the step in flight has to be done
  int bvar;                      // blend variant of scheme B (L503): 0 = diagonal Theta, 1 = Bmax, 2 = Bmin
  int lumping;                   // 0 = global lumping (L576), 1 = selective lumping (eq. 66-67)
  // Bx (eq. 56): domain size and the bit patterns of max / min vertex speed of the state of stage 1 ([0]) and 2 ([1])
  double bx_L;
  unsigned long long vmax_bits[2], vmin_bits[2];
};
// 1 / (|v|_max - |v|_min) of stage `k`, 0 when the speeds are all equal (reading C24)
__device__ __forceinline__ double bx_inv_range(const Ctl *c, int k) {
  double r = __longlong_as_double((long long)c->vmax_bits[k]) - __longlong_as_double((long long)c->vmin_bits[k]);
  return r > 0.0 ? 1.0 / r : 0.0;
}

template <class R> struct MeshDev {
  int64_t nv, nt;
  const int32_t *tv[3];         // connectivity, SoA
  const R *gnx[3], *gny[3], *ghl[3];  // geometry, SoA
  const R *area3, *lmax;        // |T|/3, longest edge
  const int32_t *csr_off, *csr_ent;
  const R *vol;                 // V_i
  const uint8_t *frozen;        // or nullptr
};

// Where a vertex kernel puts the per-vertex quantities the triangle kernels read: per-vertex arrays (unfused
// path) or one copy per tile slot of the vertex (fused path: the tile kernels then stream contiguous slot
// ranges with bulk copies and never gather by vertex index).
template <class R> struct VertexSink {
  Vec4<R> *Z;                 // parameter vector (S1)
  R *spd;                     // |v| + c (S6), may be null
  Vec4<R> *D;                 // dW/dt of stage 1 (eq. 57), may be null
  const int32_t *vslot_off;   // null: index by vertex; else Z/spd/D are indexed by slot
  const int32_t *vslot_ent;
  __device__ __forceinline__ void put(int64_t i, const Vec4<R> &z, R s, bool has_d, const Vec4<R> &d) const {
    if (vslot_off) {
      const int32_t q0 = __ldg(vslot_off + i), q1 = __ldg(vslot_off + i + 1);
      for (int32_t q = q0; q < q1; ++q) {
        const int32_t sl = __ldg(vslot_ent + q);
        st4(&Z[sl], z);
        if (spd) spd[sl] = s;
        if (has_d) st4(&D[sl], d);
      }
    } else {
      st4(&Z[i], z);
      if (spd) spd[i] = s;
      if (has_d) st4(&D[i], d);
    }
  }
};

#define MRD_CTL_GUARD(ctl) \
  if ((ctl)->status != 0 || (ctl)->active == 0) return;

__device__ __forceinline__ double ctl_dt(const Ctl *c) {
  // eq. 44 (L443): dt = CFL * min_i 2 V_i / sum_T l_max lambda_max; clipped to t_end (reading C13)
  double dt = c->cfl * __longlong_as_double((long long)c->dmin_bits);
  if (c->t_end > 0.0 && c->t + dt > c->t_end) dt = c->t_end - c->t;
  return dt;
}

// ---------------------------------------------------------------------------------------------
// step control: one thread.  mode 0 = start of mrd_step (set t_end, arm), 1 = a step finished
// ---------------------------------------------------------------------------------------------
__global__ void ctl_kernel(Ctl *c, int mode, double t_end, const int *flag) {
  if (mode == 0) {
    c->t_end = t_end;
  } else {
    if (*flag) c->status = 1;  // a kernel of this step met rho <= 0, p <= 0 or c^2 <= 0: discard the step
    if (c->status == 0 && c->active) {
      double dt = ctl_dt(c);
      c->dt = dt;
      c->t = (c->t_end > 0.0 && c->t + dt >= c->t_end) ? c->t_end : c->t + dt;
      c->steps += 1;
    }
  }
  c->dmin_bits = 0x7FF0000000000000ull;  // +inf
  c->vmax_bits[0] = c->vmax_bits[1] = 0ull;
  c->vmin_bits[0] = c->vmin_bits[1] = 0x7FF0000000000000ull;
  c->active = (c->status == 0 && !(c->t_end > 0.0 && c->t >= c->t_end)) ? 1 : 0;
}

// ---------------------------------------------------------------------------------------------
// state I/O: user-numbered SoA <-> internal AoS; prepare Z and the signal speed (S1, S6)
// ---------------------------------------------------------------------------------------------
template <class R>
__global__ void set_state_kernel(int64_t nv, const int32_t *__restrict__ vperm, const R *__restrict__ Wuser,
                                 R gamma, Vec4<R> *__restrict__ W, VertexSink<R> sink, int *bad) {
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  int64_t u = vperm[i];
  Vec4<R> w{Wuser[u], Wuser[nv + u], Wuser[2 * nv + u], Wuser[3 * nv + u]};
  Vec4<R> z;
  R s, p;
  bool ok = vertex_prepare(gamma, w, z, s, p);
  st4(&W[i], w);
  sink.put(i, z, s, false, z);
  if (!ok) atomicOr(bad, 1);
}

template <class R>
__global__ void get_state_kernel(int64_t nv, const int32_t *__restrict__ vrank, const Vec4<R> *__restrict__ W,
                                 R *__restrict__ Wuser) {
  int64_t u = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= nv) return;
  Vec4<R> w = ld4(&W[vrank[u]]);
  Wuser[u] = w.x;
  Wuser[nv + u] = w.y;
  Wuser[2 * nv + u] = w.z;
  Wuser[3 * nv + u] = w.w;
}

// ---------------------------------------------------------------------------------------------
// Triangle kernel, one thread per triangle.
//   STAGE 1: phi (scheme residuals) [nt][3], stored phi^N(W^n) and phi^T(W^n) for stage 2, s_T
//   STAGE 2: total residuals of eq. 57, 61-65 from Z*, dW/dt and the stored stage-1 values
// ---------------------------------------------------------------------------------------------
template <class R> __device__ __forceinline__ void load_geom(const MeshDev<R> &m, int64_t t, TriGeom<R> &g) {
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    g.nx[i] = __ldg(m.gnx[i] + t);
    g.ny[i] = __ldg(m.gny[i] + t);
    g.hl[i] = __ldg(m.ghl[i] + t);
  }
}

template <class R, int SCHEME, bool STORE>
__global__ void __launch_bounds__(128)
tri_stage1_kernel(MeshDev<R> m, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Z,
                  const R *__restrict__ spd, Vec4<R> *__restrict__ phi, Vec4<R> *__restrict__ phiN_n,
                  Vec4<R> *__restrict__ phiT_n, R *__restrict__ sT, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m.nt) return;
  int32_t v[3] = {__ldg(m.tv[0] + t), __ldg(m.tv[1] + t), __ldg(m.tv[2] + t)};
  Vec4<R> z[3] = {ld4(&Z[v[0]]), ld4(&Z[v[1]]), ld4(&Z[v[2]])};
  R sp = Fast<R>::max(__ldg(spd + v[0]), Fast<R>::max(__ldg(spd + v[1]), __ldg(spd + v[2])));
  TriGeom<R> g;
  load_geom(m, t, g);
  TriCore<R> k;
  R pT[4], pN[3][4];
  triangle_core(gamma, z, g, k, pT, pN);
  if (!k.ok) atomicOr(status, 1);
  sT[t] = __ldg(m.lmax + t) * sp;  // eq. 44-45: l_max^T * max_j (|v_j| + c_j)
  if (STORE) {
    st4(&phiT_n[t], Vec4<R>{pT[0], pT[1], pT[2], pT[3]});
#pragma unroll
    for (int i = 0; i < 3; ++i) st4(&phiN_n[3 * t + i], Vec4<R>{pN[i][0], pN[i][1], pN[i][2], pN[i][3]});
  }
  if (SCHEME != MRD_SCHEME_N) {
    R pL[3][4];
    apply_beta(gamma, k, g, pT, pL);
    if (SCHEME == MRD_SCHEME_B) {
      blend(pT, pN, pL, ctl->bvar);
    } else if (SCHEME == MRD_SCHEME_BX) {
      const R th = bx_theta(z, g, __ldg(m.area3 + t), __ldg(m.lmax + t), (R)ctl->bx_L, (R)bx_inv_range(ctl, 0));
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c] + th * (pN[i][c] - pL[i][c]);
    } else {
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c];
    }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) st4(&phi[3 * t + i], Vec4<R>{pN[i][0], pN[i][1], pN[i][2], pN[i][3]});
}

template <class R, int SCHEME>
__global__ void __launch_bounds__(128)
tri_stage2_kernel(MeshDev<R> m, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Zs,
                  const Vec4<R> *__restrict__ dWdt, const Vec4<R> *__restrict__ phiN_n,
                  const Vec4<R> *__restrict__ phiT_n, Vec4<R> *__restrict__ phi, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= m.nt) return;
  int32_t v[3] = {__ldg(m.tv[0] + t), __ldg(m.tv[1] + t), __ldg(m.tv[2] + t)};
  Vec4<R> z[3] = {ld4(&Zs[v[0]]), ld4(&Zs[v[1]]), ld4(&Zs[v[2]])};
  TriGeom<R> g;
  load_geom(m, t, g);
  TriCore<R> k;
  R pT[4], pN[3][4];
  triangle_core(gamma, z, g, k, pT, pN);  // all matrices re-evaluated at W* (reading C12)
  if (!k.ok) atomicOr(status, 1);
  const R a3 = __ldg(m.area3 + t);
  // eq. 57 / 61: Phi^T = |T|/3 sum_j dW_j/dt + (phi^T(W^n) + phi^T(W*))/2;  eq. 62: Phi_i^N likewise per node
  R PT[4];
  {
    Vec4<R> o = ld4(&phiT_n[t]);
    PT[0] = R(0.5) * (o.x + pT[0]); PT[1] = R(0.5) * (o.y + pT[1]);
    PT[2] = R(0.5) * (o.z + pT[2]); PT[3] = R(0.5) * (o.w + pT[3]);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    Vec4<R> d = ld4(&dWdt[v[i]]);
    Vec4<R> o = ld4(&phiN_n[3 * t + i]);
    R m0 = a3 * d.x, m1 = a3 * d.y, m2 = a3 * d.z, m3 = a3 * d.w;
    PT[0] += m0; PT[1] += m1; PT[2] += m2; PT[3] += m3;
    pN[i][0] = m0 + R(0.5) * (pN[i][0] + o.x);
    pN[i][1] = m1 + R(0.5) * (pN[i][1] + o.y);
    pN[i][2] = m2 + R(0.5) * (pN[i][2] + o.z);
    pN[i][3] = m3 + R(0.5) * (pN[i][3] + o.w);
  }
  R E[3][4];
  const bool lump = ctl->lumping != 0;
  if (lump) {  // selective lumping (eq. 66-67): E_i = |T|/12 (3 dW_i/dt - sum_j dW_j/dt), on Phi^N and Phi^LDA alike
    Vec4<R> d0 = ld4(&dWdt[v[0]]), d1 = ld4(&dWdt[v[1]]), d2 = ld4(&dWdt[v[2]]);
    R dv[3][4] = {{d0.x, d0.y, d0.z, d0.w}, {d1.x, d1.y, d1.z, d1.w}, {d2.x, d2.y, d2.z, d2.w}};
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        E[i][c] = (R(0.25) * a3) * (R(3) * dv[i][c] - (dv[0][c] + dv[1][c] + dv[2][c]));
        pN[i][c] += E[i][c];
      }
  }
  if (SCHEME != MRD_SCHEME_N) {
    R pL[3][4];
    apply_beta(gamma, k, g, PT, pL);  // eq. 63 with eq. 65: Phi_i^LDA = beta_i(W*) Phi^T
    if (lump) {
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int c = 0; c < 4; ++c) pL[i][c] += E[i][c];
    }
    if (SCHEME == MRD_SCHEME_B) {
      blend(PT, pN, pL, ctl->bvar);
    } else if (SCHEME == MRD_SCHEME_BX) {  // the sensor of W*, the state the matrices are evaluated at (as C12)
      const R th = bx_theta(z, g, a3, __ldg(m.lmax + t), (R)ctl->bx_L, (R)bx_inv_range(ctl, 1));
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c] + th * (pN[i][c] - pL[i][c]);
    } else {
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int c = 0; c < 4; ++c) pN[i][c] = pL[i][c];
    }
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) st4(&phi[3 * t + i], Vec4<R>{pN[i][0], pN[i][1], pN[i][2], pN[i][3]});
}

// ---------------------------------------------------------------------------------------------
// Vertex kernels.  gather: acc_i = sum_{T ni i} phi_i^T in ascending CSR order (deterministic; replaces
// the paper's atomic scatter, L734); stage 1 also d_i = 2 V_i / sum s_T and its global minimum (S7).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void block_min_to_global(double d, unsigned long long *dmin_bits) {
  // warp shuffle -> shared -> one atomicMin per block; positive doubles order like their bit patterns
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) d = fmin(d, __shfl_xor_sync(0xFFFFFFFFu, d, o));
  __shared__ double wmin[32];
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) wmin[w] = d;
  __syncthreads();
  if (w == 0) {
    int nw = (blockDim.x + 31) >> 5;
    d = lane < nw ? wmin[lane] : __longlong_as_double(0x7FF0000000000000ll);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) d = fmin(d, __shfl_xor_sync(0xFFFFFFFFu, d, o));
    if (lane == 0) atomicMin(dmin_bits, (unsigned long long)__double_as_longlong(d));
  }
}

template <class R>
__global__ void __launch_bounds__(256)
gather_dt_kernel(MeshDev<R> m, Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ phi, const R *__restrict__ sT,
                 Vec4<R> *__restrict__ acc) {
  MRD_CTL_GUARD(ctl)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double d = __longlong_as_double(0x7FF0000000000000ll);
  if (i < m.nv) {
    R a0 = 0, a1 = 0, a2 = 0, a3 = 0, S = 0;
    int32_t q0 = __ldg(m.csr_off + i), q1 = __ldg(m.csr_off + i + 1);
    for (int32_t q = q0; q < q1; ++q) {
      int32_t e = __ldg(m.csr_ent + q);
      Vec4<R> f = ld4(&phi[e]);
      a0 += f.x; a1 += f.y; a2 += f.z; a3 += f.w;
      S += __ldg(sT + e / 3);
    }
    st4(&acc[i], Vec4<R>{a0, a1, a2, a3});
    if (!(m.frozen && m.frozen[i] == 2)) d = 2.0 * (double)__ldg(m.vol + i) / (double)S;  // halo: fan incomplete here
  }
  block_min_to_global(d, &ctl->dmin_bits);
}

// Bx (eq. 56, reading C24): max and min of the vertex speeds |v_i| of the state W, into slot `k` of the control block
template <class R>
__global__ void __launch_bounds__(256) vrange_kernel(int64_t nv, const Vec4<R> *__restrict__ W, Ctl *__restrict__ ctl, int k) {
  MRD_CTL_GUARD(ctl)
  double hi = 0.0, lo = __longlong_as_double(0x7FF0000000000000ll);
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += (int64_t)gridDim.x * blockDim.x) {
    Vec4<R> w = ld4(&W[i]);
    double u = (double)w.y / (double)w.x, v = (double)w.z / (double)w.x;
    double a = sqrt(u * u + v * v);
    hi = fmax(hi, a);
    lo = fmin(lo, a);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    hi = fmax(hi, __shfl_xor_sync(0xFFFFFFFFu, hi, o));
    lo = fmin(lo, __shfl_xor_sync(0xFFFFFFFFu, lo, o));
  }
  __shared__ double shi[8], slo[8];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) { shi[w] = hi; slo[w] = lo; }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int q = 1; q < 8; ++q) { hi = fmax(hi, shi[q]); lo = fmin(lo, slo[q]); }
    atomicMax(&ctl->vmax_bits[k], (unsigned long long)__double_as_longlong(hi));  // non-negative doubles order like their bits
    atomicMin(&ctl->vmin_bits[k], (unsigned long long)__double_as_longlong(lo));
  }
}

// Bx on a partitioned mesh: the local range of stage k as d = (|v|_max, -|v|_min) -- a max-reduction over all parts of both
// numbers gives the global range -- and back
__global__ void range_reset_kernel(Ctl *c, int k) {
  c->vmax_bits[k] = 0ull;
  c->vmin_bits[k] = 0x7FF0000000000000ull;
}
__global__ void range_get_kernel(const Ctl *__restrict__ c, int k, double *__restrict__ d) {
  d[0] = __longlong_as_double((long long)c->vmax_bits[k]);
  d[1] = -__longlong_as_double((long long)c->vmin_bits[k]);
}
__global__ void range_set_kernel(Ctl *__restrict__ c, int k, const double *__restrict__ d) {
  c->vmax_bits[k] = (unsigned long long)__double_as_longlong(d[0]);
  c->vmin_bits[k] = (unsigned long long)__double_as_longlong(-d[1]);
}

// finish a vertex: W_new = W_old - dt/V * acc (eq. 43 / 60 / 61); frozen vertices keep W_old (their
// initial state, L582); then Z and the signal speed of the new state (S1, S6), positivity check.
template <class R, bool WANT_DWDT>
__device__ __forceinline__ void vertex_finish(R gamma, R dt, R vol, bool frozen, const Vec4<R> &Wold, const R a[4],
                                              int64_t i, Vec4<R> *Wout, const VertexSink<R> &sink, int *status) {
  R f = frozen ? R(0) : dt * Fast<R>::rcp(vol);
  Vec4<R> w{Wold.x - f * a[0], Wold.y - f * a[1], Wold.z - f * a[2], Wold.w - f * a[3]};
  Vec4<R> z;
  R s, p;
  bool ok = vertex_prepare(gamma, w, z, s, p);
  if (!ok) atomicOr(status, 1);
  st4(&Wout[i], w);
  Vec4<R> d{0, 0, 0, 0};
  if (WANT_DWDT) {
    R idt = Fast<R>::rcp(dt);
    d = Vec4<R>{(w.x - Wold.x) * idt, (w.y - Wold.y) * idt, (w.z - Wold.z) * idt, (w.w - Wold.w) * idt};
  }
  sink.put(i, z, s, WANT_DWDT, d);
}

// after gather_dt (+ wall terms): FINAL = false: stage 1 of RK2 -> W*, Z*, dW/dt; true: eq. 43 -> W^{n+1}
template <class R, bool FINAL>
__global__ void __launch_bounds__(256)
update_kernel(MeshDev<R> m, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Wn,
              const Vec4<R> *__restrict__ acc, Vec4<R> *__restrict__ Wout, VertexSink<R> sink, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m.nv) return;
  R dt = (R)ctl_dt(ctl);
  Vec4<R> w = ld4(&Wn[i]);
  Vec4<R> a = ld4(&acc[i]);
  R av[4] = {a.x, a.y, a.z, a.w};
  bool fr = m.frozen ? (m.frozen[i] != 0) : false;
  vertex_finish<R, !FINAL>(gamma, dt, __ldg(m.vol + i), fr, w, av, i, Wout, sink, status);
}

// stage 2: gather the total residuals and finish W^{n+1} = W* - dt/V sum Phi_i (eq. 61), in place over W*
template <class R>
__global__ void __launch_bounds__(256)
gather_update_kernel(MeshDev<R> m, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ phi,
                     const Vec4<R> *__restrict__ wall_acc, Vec4<R> *__restrict__ Ws, VertexSink<R> sink, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m.nv) return;
  R a[4] = {0, 0, 0, 0};
  int32_t q0 = __ldg(m.csr_off + i), q1 = __ldg(m.csr_off + i + 1);
  for (int32_t q = q0; q < q1; ++q) {
    Vec4<R> f = ld4(&phi[__ldg(m.csr_ent + q)]);
    a[0] += f.x; a[1] += f.y; a[2] += f.z; a[3] += f.w;
  }
  if (wall_acc) {
    Vec4<R> f = wall_acc[i];
    a[0] += f.x; a[1] += f.y; a[2] += f.z; a[3] += f.w;
  }
  R dt = (R)ctl_dt(ctl);
  Vec4<R> w = Ws[i];
  bool fr = m.frozen ? (m.frozen[i] != 0) : false;
  vertex_finish<R, false>(gamma, dt, __ldg(m.vol + i), fr, w, a, i, Ws, sink, status);
}

// ---------------------------------------------------------------------------------------------
// Reflecting walls (eq. 68-71; alpha = 0.75; outward normal, reading C15): one thread per
// wall VERTEX adds, in ascending edge order, the correction of every wall edge it belongs to.
//   stage 1: dst[v] += Phi^c(W^n)            (dst = acc of gather_dt; SET: dst[v] = ..., dst = wall_acc, fused path)
//   stage 2: dst[v]  = sum (Phi^c(W^n) + Phi^c(W*))/2   (dst = wall_acc, zero elsewhere)
// ---------------------------------------------------------------------------------------------
template <class R> struct WallDev {
  int64_t nwv;
  const int32_t *wv_vertex, *wv_off, *wv_ent, *wall_a, *wall_b;
  const R *nx, *ny, *len;
};

template <class R> __device__ __forceinline__ void wall_flux(R gamma, const Vec4<R> &W, R nx, R ny, R F[4]) {
  R ir = Fast<R>::rcp(W.x);
  R u = W.y * ir, v = W.z * ir;
  R p = (gamma - R(1)) * (W.w - R(0.5) * (W.y * u + W.z * v));
  R vn = u * nx + v * ny;
  F[0] = -(W.x * vn);  // eq. 68: desired (no through-flow) minus computed boundary flux
  F[1] = -(W.y * vn);
  F[2] = -(W.z * vn);
  F[3] = -((W.w + p) * vn);
}

template <class R, int STAGE, bool SET = (STAGE == 2)>
__global__ void wall_kernel(WallDev<R> wd, R gamma, const Ctl *__restrict__ ctl, const Vec4<R> *__restrict__ Wn,
                            const Vec4<R> *__restrict__ Ws, Vec4<R> *__restrict__ dst) {
  MRD_CTL_GUARD(ctl)
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= wd.nwv) return;
  int32_t vtx = wd.wv_vertex[k];
  R s[4] = {0, 0, 0, 0};
  for (int32_t q = wd.wv_off[k]; q < wd.wv_off[k + 1]; ++q) {
    int32_t ent = wd.wv_ent[q];
    int32_t e = ent >> 1, side = ent & 1;
    int32_t a = wd.wall_a[e], b = wd.wall_b[e];
    R nx = wd.nx[e], ny = wd.ny[e], hl = R(0.5) * wd.len[e];
    // eq. 70-71: Phi_a = l/2 (alpha F_a + (1-alpha) F_b), Phi_b = l/2 ((1-alpha) F_a + alpha F_b)
    R ca = side == 0 ? R(0.75) : R(0.25), cb = R(1) - ca;
    R Fa[4], Fb[4];
    wall_flux(gamma, Wn[a], nx, ny, Fa);
    wall_flux(gamma, Wn[b], nx, ny, Fb);
    if (STAGE == 1) {
#pragma unroll
      for (int c = 0; c < 4; ++c) s[c] += hl * (ca * Fa[c] + cb * Fb[c]);
    } else {
      R Ga[4], Gb[4];
      wall_flux(gamma, Ws[a], nx, ny, Ga);
      wall_flux(gamma, Ws[b], nx, ny, Gb);
#pragma unroll
      for (int c = 0; c < 4; ++c) s[c] += R(0.5) * (hl * (ca * Fa[c] + cb * Fb[c]) + hl * (ca * Ga[c] + cb * Gb[c]));
    }
  }
  Vec4<R> d;
  if (SET) {
    d = Vec4<R>{s[0], s[1], s[2], s[3]};
  } else {
    d = dst[vtx];
    d.x += s[0]; d.y += s[1]; d.z += s[2]; d.w += s[3];
  }
  dst[vtx] = d;
}

// ---------------------------------------------------------------------------------------------
// Diagnostics (S13): fixed-shape two-level reduction -> deterministic.  partial[b][6] per block:
// sum V W_k (4), min rho, min p.
// ---------------------------------------------------------------------------------------------
template <class R>
__global__ void __launch_bounds__(256)
diag_kernel(int64_t nv, R gamma, const Vec4<R> *__restrict__ W, const R *__restrict__ vol, const uint8_t *__restrict__ flag,
            double *__restrict__ partial) {
  double s[4] = {0, 0, 0, 0}, mr = __longlong_as_double(0x7FF0000000000000ll), mp = mr;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += (int64_t)gridDim.x * blockDim.x) {
    Vec4<R> w = ld4(&W[i]);
    double V = (flag && flag[i] == 2) ? 0.0 : (double)vol[i];  // a halo vertex is counted by the part that owns it
    s[0] += V * (double)w.x; s[1] += V * (double)w.y; s[2] += V * (double)w.z; s[3] += V * (double)w.w;
    double p = ((double)gamma - 1.0) * ((double)w.w - 0.5 * ((double)w.y * (double)w.y + (double)w.z * (double)w.z) / (double)w.x);
    mr = fmin(mr, (double)w.x);
    mp = fmin(mp, p);
  }
  __shared__ double sh[256][6];
  int tid = threadIdx.x;
  sh[tid][0] = s[0]; sh[tid][1] = s[1]; sh[tid][2] = s[2]; sh[tid][3] = s[3]; sh[tid][4] = mr; sh[tid][5] = mp;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (tid < o) {
#pragma unroll
      for (int c = 0; c < 4; ++c) sh[tid][c] += sh[tid + o][c];
      sh[tid][4] = fmin(sh[tid][4], sh[tid + o][4]);
      sh[tid][5] = fmin(sh[tid][5], sh[tid + o][5]);
    }
    __syncthreads();
  }
  if (tid < 6) partial[blockIdx.x * 6 + tid] = sh[0][tid];
}

// ---------------------------------------------------------------------------------------------
// Domain decomposition (include/mrd.h "Domain decomposition"): halo pack / unpack, dt exchange
// ---------------------------------------------------------------------------------------------
template <class R>
__global__ void halo_pack_kernel(int64_t n, const int32_t *__restrict__ idx, const Ctl *__restrict__ ctl,
                                 const Vec4<R> *__restrict__ W, Vec4<R> *__restrict__ buf) {
  MRD_CTL_GUARD(ctl)
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k < n) st4(&buf[k], ld4(&W[idx[k]]));
}

// FIRST: after stage 1 of RK2 (the owner's W*; Z* and dW/dt = (W* - W^n)/dt to the slots, as vertex_finish<.., true>);
// else the owner's W^{n+1} (Z and |v| + c to the slots)
template <class R, bool FIRST>
__global__ void halo_unpack_kernel(int64_t n, const int32_t *__restrict__ idx, R gamma, const Ctl *__restrict__ ctl,
                                   const Vec4<R> *__restrict__ buf, const Vec4<R> *__restrict__ Wold,
                                   Vec4<R> *__restrict__ Wout, VertexSink<R> sink, int *status) {
  MRD_CTL_GUARD(ctl)
  int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int64_t i = idx[k];
  Vec4<R> w = ld4(&buf[k]);
  Vec4<R> z;
  R s, p;
  bool ok = vertex_prepare(gamma, w, z, s, p);
  if (!ok) atomicOr(status, 1);
  Vec4<R> d{0, 0, 0, 0};
  if (FIRST) {
    Vec4<R> o = ld4(&Wold[i]);
    R idt = Fast<R>::rcp((R)ctl_dt(ctl));
    d = Vec4<R>{(w.x - o.x) * idt, (w.y - o.y) * idt, (w.z - o.z) * idt, (w.w - o.w) * idt};
  }
  st4(&Wout[i], w);
  sink.put(i, z, s, FIRST, d);
}

// d[0] = local min of 2 V_i / sum s_T (eq. 44), d[1] = -1 if a kernel of this part met a non-physical state
__global__ void dt_get_kernel(const Ctl *__restrict__ c, const int *__restrict__ flag, double *__restrict__ d) {
  d[0] = __longlong_as_double((long long)c->dmin_bits);
  d[1] = (*flag || c->status) ? -1.0 : 0.0;
}
__global__ void dt_set_kernel(Ctl *__restrict__ c, int *__restrict__ flag, const double *__restrict__ d) {
  c->dmin_bits = (unsigned long long)__double_as_longlong(d[0]);
  if (d[1] < 0.0) *flag = 1;
}

// d[0] = 1 if a kernel of this part met a non-physical state in the step in flight (or earlier), else 0; after a
// max-reduction over the parts, status_set raises the flag everywhere, so that every part discards the SAME step at END
__global__ void status_get_kernel(const Ctl *__restrict__ c, const int *__restrict__ flag, double *__restrict__ d) {
  d[0] = (*flag || c->status) ? 1.0 : 0.0;
}
__global__ void status_set_kernel(int *__restrict__ flag, const double *__restrict__ d) {
  if (d[0] > 0.0) *flag = 1;
}

// ---------------------------------------------------------------------------------------------
// Peak micro-benchmarks (roofline denominators): FMA throughput and device copy
// ---------------------------------------------------------------------------------------------
template <class R> __global__ void __launch_bounds__(256) fma_peak_kernel(R *out, int iters, R a, R b) {
  R x[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) x[j] = R(threadIdx.x + j) * R(1e-3);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int j = 0; j < 8; ++j) x[j] = Fast<R>::fma_(x[j], a, b);
  }
  R s = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += x[j];
  if (s == R(-12345)) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) copy_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, int64_t n) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

}  // namespace mrd
