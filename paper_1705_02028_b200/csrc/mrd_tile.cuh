// mrd_tile.cuh -- the fused tile kernels (the production path).  A tile is a run of `tile` consecutive
// (Morton-ordered) triangles; a "slot" is one tile-local vertex (mrd_layout.h).  Persistent thread blocks
// walk over tiles with a two-deep software pipeline:
//
//   stage-in : everything a tile needs lives in CONTIGUOUS global ranges (slot-major copies of Z, |v|+c,
//              dW/dt written by the vertex side; tile-frame coordinates or geometry records; the tile's plan
//              record; for stage 2 the stored phi^N(W^n), phi^T(W^n)), so one thread brings the tile AFTER NEXT
//              in with a handful of TMA bulk copies (cp.async.bulk + mbarrier complete_tx) as soon as the last
//              warp has left the buffer it goes into -- no gather by vertex index, no dependent global latency;
//   body     : one thread per triangle; geometry of eq. 35 (L397-L399) from the geometry table or the staged
//              coordinates, then S2-S5 / S9 of SURVEY 8a with the device functions of mrd_math.cuh;
//   epilogue : distributed residuals -> shared memory (16-byte cells); every slot sums its incident (triangle,
//              node) entries in ascending order, four to a batch with all loads issued before the first add; ONE
//              partial per slot leaves the SM (deterministic; replaces the float atomics of L734 and the 3 x 4
//              values per triangle of the unfused design).
// The vertex kernels add a vertex's few partials (ascending slot = ascending triangle order) and scatter the new
// per-vertex quantities back to the vertex's slots.  (Finishing the vertices inside the tile kernels -- directly for
// the 77 % whose fan lies in one tile, by the last tile to arrive for the rest -- was built and measured in round 2:
// the arithmetic of a vertex update costs the fp64-bound tile kernels what it costs, the vertex kernels hide it under
// their HBM time, and the arrival protocol adds a chain of L2 round trips per tile; see profiles/r02_experiments.md.)
// One block barrier per tile (between the residuals and their sums); warps that are done move on to the next tile.
#pragma once
#include "mrd_kernels.cuh"

namespace mrd {

template <class R> struct TileDev {
  int32_t tile, maxslots, offn, maxbatch, plan_stride, maxshapes;
  int64_t ntile, nslot, nt, nv;
  const int4 *tile_info;         // [ntile+1]: .x first slot (padded slot counts: multiples of 4), .y first geometry record, .z plan record
  const R *shape_geom;           // [nshape][12] geometry records (GTAB kernels), else null
  const uint16_t *plan;          // [nplan][plan_stride]: tri[T][4] | boff[offn] | ent[4 maxbatch]  (mrd_layout.h)
  const R *slot_xy;              // [nslot][2], relative to the tile's anchor vertex
  const int32_t *vslot_off;      // [nv+1]
  const int32_t *vslot_ent;      // [#real slots]
};

// ---- PTX wrappers: mbarrier + TMA bulk copy (SASS: UBLKCP) ----------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "MRD_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra MRD_DONE;\n"
      "bra MRD_WAIT;\n"
      "MRD_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// tile_info prefetch: a plain (per-thread register) global load whose result is handed over through an opaque
// move at the point of use.  Without this the compiler turns the block-uniform value into a uniform register
// right after the load (R2UR), stalling every warp on the global latency once per tile (10 % of all stall samples).
__device__ __forceinline__ int4 ld_info(const int4 *p) {
  int4 v;
  asm volatile("ld.global.nc.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ int4 use_info(int4 v) {
  int4 o;
  asm volatile("mov.b32 %0, %4;\n\tmov.b32 %1, %5;\n\tmov.b32 %2, %6;\n\tmov.b32 %3, %7;"
               : "=r"(o.x), "=r"(o.y), "=r"(o.z), "=r"(o.w)
               : "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w));
  return o;
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// shared-memory cells of the residual exchange (two components each: 16 bytes in fp64)
template <class R> struct Cell;
template <> struct __align__(16) Cell<double> { double a, b; };
template <> struct __align__(8) Cell<float> { float a, b; };
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

// ---- shared-memory carve-up (dynamic).  Two stage-in buffers + the residual exchange area ----------------
// Residual cells of one tile (T triangles): cell (half h, node i, triangle t) at index h HOFF + i T + t holds the
// components (2h, 2h + 1) of the residual sent to node i; HOFF = 3T + 1 (fp64; 3T + 2 in fp32, which keeps the second half
// 16-byte aligned for the bulk copies).  The cells 3T and HOFF + 3T stay zero: they are what the sentinel incidence entry
// 3T of the plan reads.
template <class R, int T> struct CellGeom {
  static constexpr int HOFF = 3 * T + 16 / (int)sizeof(Cell<R>);
  static constexpr int NCELL = HOFF + 3 * T + 1;
};
template <class R, int STAGE, bool GTAB> struct TileSmem {
  // computed once on the host and passed to the kernel by value (the device code recomputed it every tile otherwise)
  uint32_t oZ, oD, oS, oXY, oPlan, oPhi, buf_bytes;  // per buffer (oXY holds the geometry records when GTAB)
  uint32_t oRes, oST, oBar, total;                          // shared
  uint32_t res_bytes, st_bytes;
  __host__ __device__ static uint32_t up16(size_t x) { return (uint32_t)((x + 15) & ~size_t(15)); }
  __host__ __device__ TileSmem(int T, int maxslots, int plan_stride, int maxshapes) {
    uint32_t o = 0;
    res_bytes = up16(sizeof(Cell<R>) * (6 * T + 16 / sizeof(Cell<R>) + 1));
    st_bytes = up16(sizeof(R) * (3 * T + 1));
    oZ = o; o += up16(sizeof(Vec4<R>) * maxslots);
    oD = o; if (STAGE == 2) o += up16(sizeof(Vec4<R>) * maxslots);
    oS = o; if (STAGE == 1) o += up16(sizeof(R) * maxslots);
    oXY = o; o += GTAB ? up16(sizeof(R) * 12 * maxshapes) : up16(sizeof(R) * 2 * maxslots);
    oPlan = o; o += up16(sizeof(uint16_t) * plan_stride);
    // stage 2: the stored stage-1 residuals arrive in the cell layout, and the residual exchange area IS that block --
    // thread `tid` only overwrites the six cells it has consumed itself (saves 12 KB: 4 blocks per SM)
    oPhi = o; if (STAGE == 2) o += res_bytes;
    buf_bytes = (o + 31u) & ~31u;
    uint32_t s = 2 * buf_bytes;
    // stage 1: two residual areas (tile k's epilogue may still read one while a faster warp writes tile k+1's)
    oRes = s; if (STAGE == 1) s += 2 * res_bytes;
    oST = s; if (STAGE == 1) s += 2 * st_bytes;
    oBar = s; s += 32;  // two mbarriers, two "warps done with the buffer" counters
    total = s;
  }
};

// bring tile b into buffer `buf` (one thread): expect_tx, then the bulk copies
template <class R, int STAGE, bool GTAB>
__device__ __forceinline__ void tile_stage_in(const TileDev<R> &td, const TileSmem<R, STAGE, GTAB> &L, unsigned char *buf,
                                              uint64_t *bar, int64_t b, int4 i0, int4 i1, const Vec4<R> *slotZ,
                                              const R *slotS, const Vec4<R> *slotD, const R *phi12) {
  const int T = td.tile;
  const int s0 = i0.x, ns = i1.x - i0.x;
  const unsigned bZ = sizeof(Vec4<R>) * ns, bS = sizeof(R) * ns;
  const unsigned bXY = GTAB ? sizeof(R) * 12 * (i1.y - i0.y) : sizeof(R) * 2 * ns;
  const unsigned bPlan = sizeof(uint16_t) * td.plan_stride, bHalf = sizeof(Cell<R>) * 3 * T;
  unsigned total = bZ + bXY + bPlan + (STAGE == 1 ? bS : bZ + 2 * bHalf);
  mbar_expect_tx(bar, total);
  bulk_g2s(buf + L.oZ, slotZ + s0, bZ, bar);
  if (GTAB) bulk_g2s(buf + L.oXY, td.shape_geom + 12 * (int64_t)i0.y, bXY, bar);
  else bulk_g2s(buf + L.oXY, td.slot_xy + 2 * (int64_t)s0, bXY, bar);
  bulk_g2s(buf + L.oPlan, td.plan + (int64_t)i0.z * td.plan_stride, bPlan, bar);
  if (STAGE == 1) {
    bulk_g2s(buf + L.oS, slotS + s0, bS, bar);
  } else {
    bulk_g2s(buf + L.oD, slotD + s0, bZ, bar);
    const R *src = phi12 + b * 12 * T;                       // [half][3 T] cells of two values
    bulk_g2s(buf + L.oPhi, src, bHalf, bar);
    bulk_g2s(buf + L.oPhi + sizeof(Cell<R>) * (3 * T + 16 / sizeof(Cell<R>)), src + 6 * T, bHalf, bar);
  }
}

// sum of the tile-local incidences of one slot, in ascending (triangle, node) order, from the residual cells
template <class R, int T, bool WITH_ST>
__device__ __forceinline__ void slot_sum(const Cell<R> *cell, const R *sTx, const uint16_t *ent, int b0, int b1, R a[4], R &S) {
  a[0] = a[1] = a[2] = a[3] = R(0);
  S = R(0);
  for (int q = b0; q < b1; ++q) {
    const uint2 pk = *reinterpret_cast<const uint2 *>(ent + 4 * q);   // four entries; all loads issued before the first add
    const unsigned e[4] = {pk.x & 0xFFFFu, pk.x >> 16, pk.y & 0xFFFFu, pk.y >> 16};
    Cell<R> lo[4], hi[4];
    R sv[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      lo[u] = cell[e[u]];
      hi[u] = cell[e[u] + CellGeom<R, T>::HOFF];
      if (WITH_ST) sv[u] = sTx[e[u]];
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      a[0] += lo[u].a;
      a[1] += lo[u].b;
      a[2] += hi[u].a;
      a[3] += hi[u].b;
      if (WITH_ST) S += sv[u];
    }
  }
}

// STAGE 1: SCHEME residuals of W^n -> partials, s_T sums, and (STORE) phi^N(W^n), phi^T(W^n) as phi12
// STAGE 2: total residuals (eq. 57, 61-65; reading C12) -> partials
#ifndef MRD_TILE_MINB
#define MRD_TILE_MINB 4
#endif
template <class R> struct TileIO {
  const Vec4<R> *slotZ;    // Z of the state the stage reads (slot-major)
  const R *slotS;          // stage 1: |v| + c
  const Vec4<R> *slotD;    // stage 2: dW/dt of stage 1
  R *phi12;                // [ntile][12 T]: phi_0^N, phi_1^N, phi^T of W^n in the cell layout (written by stage 1, read by stage 2)
  Vec4<R> *part;           // [nslot] out: one partial residual sum per slot
  R *partS;                // [nslot] out, stage 1: partial s_T sums
  Vec4<R> *phi_dbg;        // dumps: per-triangle distributed residuals [nt][3], or null
  R *sT_dbg;
};
// STORE: stage 1 keeps phi^N(W^n), phi^T(W^n) for stage 2; stage 2 reuses the flag for selective lumping (eq. 66-67), a
// compile-time switch because the extra live ranges of a run-time branch cost the headline configuration 8 %.
template <class R, int SCHEME, int STAGE, bool STORE, int TILE, bool GTAB>
__global__ void __launch_bounds__(TILE, (MRD_TILE_MINB * 128) / TILE)
tile_kernel(TileDev<R> td, const TileSmem<R, STAGE, GTAB> L, R gamma, const Ctl *__restrict__ ctl, TileIO<R> io, int *status) {
  MRD_CTL_GUARD(ctl)
  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr int T = TILE;  // compile-time tile size: shared-memory and cell strides become immediates
  constexpr int HOFF = CellGeom<R, TILE>::HOFF;
  const int tid = threadIdx.x;
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + L.oBar);
  unsigned *done = reinterpret_cast<unsigned *>(smem_raw + L.oBar + 16);
  constexpr unsigned NW = TILE / 32;
  int64_t b = blockIdx.x;
  // slot / geometry-record range of the tile in flight (i0, i1); the next tile's range is fetched one iteration ahead
  int4 i0 = __ldg(td.tile_info + b), i1 = __ldg(td.tile_info + b + 1);
  if (tid == 0) {
    mbar_init(&bar[0], 1);
    mbar_init(&bar[1], 1);
    done[0] = done[1] = 0;
    fence_mbar_init();
    // the first two tiles of this block; every later copy is issued by the last warp to leave the buffer it refills
    tile_stage_in<R, STAGE, GTAB>(td, L, smem_raw, &bar[0], b, i0, i1, io.slotZ, io.slotS, io.slotD, io.phi12);
    const int64_t b1 = b + gridDim.x;
    if (b1 < td.ntile)
      tile_stage_in<R, STAGE, GTAB>(td, L, smem_raw + L.buf_bytes, &bar[1], b1, __ldg(td.tile_info + b1), __ldg(td.tile_info + b1 + 1),
                                    io.slotZ, io.slotS, io.slotD, io.phi12);
  }
  // the zero cells (what the sentinel incidence entry reads) of both residual areas; nothing ever writes them again
  if (tid < 2) {
    for (int k = 0; k < 2; ++k) {
      unsigned char *area = STAGE == 1 ? smem_raw + L.oRes + k * L.res_bytes : smem_raw + k * L.buf_bytes + L.oPhi;
      Cell<R> *c = reinterpret_cast<Cell<R> *>(area);
      c[tid == 0 ? 3 * T : CellGeom<R, T>::HOFF + 3 * T] = Cell<R>{R(0), R(0)};
      if (STAGE == 1 && tid == 0) reinterpret_cast<R *>(smem_raw + L.oST + k * L.st_bytes)[3 * T] = R(0);
    }
  }
  __syncthreads();
  int4 n0 = make_int4(0, 0, 0, 0), n1 = n0;
  const int bvar = ctl->bvar;
  const R bxL = (R)ctl->bx_L, bxInv = SCHEME == MRD_SCHEME_BX ? (R)bx_inv_range(ctl, STAGE - 1) : R(0);
  constexpr bool lump = STAGE == 2 && STORE;
  bool bad = false;  // linearised c^2 <= 0 met by this thread (raised once, after the loop)
  for (int k = 0; b < td.ntile; b += gridDim.x, ++k) {
    const int cur = k & 1;
    unsigned char *buf = smem_raw + cur * L.buf_bytes;
    const int64_t nb = b + gridDim.x;
    if (nb < td.ntile) {  // in flight during this iteration, consumed at its end
      n0 = ld_info(td.tile_info + nb);
      n1 = ld_info(td.tile_info + nb + 1);
    }
    const int s0 = i0.x, ns = i1.x - i0.x;
    mbar_wait(&bar[cur], (k >> 1) & 1);
    const Vec4<R> *sZ = reinterpret_cast<const Vec4<R> *>(buf + L.oZ);
    const R *sXY = reinterpret_cast<const R *>(buf + L.oXY);
    const uint16_t *plan = reinterpret_cast<const uint16_t *>(buf + L.oPlan);
    Cell<R> *cell = reinterpret_cast<Cell<R> *>(STAGE == 1 ? smem_raw + L.oRes + cur * L.res_bytes : buf + L.oPhi);
    R *sTx = reinterpret_cast<R *>(smem_raw + L.oST + cur * L.st_bytes);
    const int64_t t = b * T + tid;
    R st = R(0);
    // (no branch around the body: a padding triangle of the last tile computes on triangle 0 and its results are zeroed)
    const bool valid = t < td.nt;
    {
      R pN[3][4];
      const ushort4 lv = reinterpret_cast<const ushort4 *>(plan)[valid ? tid : 0];
      const int l[3] = {lv.x, lv.y, lv.z};
      Vec4<R> z[3] = {sZ[l[0]], sZ[l[1]], sZ[l[2]]};
      TriGeom<R> g;
      R a3, lmax;
      if (GTAB) {  // geometry record of this triangle's shape (layout stage; bitwise the oracle's geometry)
        const R *G = sXY + 12 * lv.w;
#pragma unroll
        for (int i = 0; i < 3; ++i) { g.nx[i] = G[i]; g.ny[i] = G[3 + i]; g.hl[i] = G[6 + i]; }
        a3 = G[9];
        lmax = G[10];
      } else {
        R x[3] = {sXY[2 * l[0]], sXY[2 * l[1]], sXY[2 * l[2]]}, y[3] = {sXY[2 * l[0] + 1], sXY[2 * l[1] + 1], sXY[2 * l[2] + 1]};
        tile_geometry(x, y, g, a3, lmax);
      }
      TriCore<R> kk;
      R pT[4];
      triangle_core(gamma, z, g, kk, pT, pN);  // stage 2: all matrices re-evaluated at W* (reading C12)
      bad |= !kk.ok;
      R X[4] = {pT[0], pT[1], pT[2], pT[3]};
      if (STAGE == 1) {
        const R *sS = reinterpret_cast<const R *>(buf + L.oS);
        st = lmax * Fast<R>::max(sS[l[0]], Fast<R>::max(sS[l[1]], sS[l[2]]));  // eq. 44-45
        if (STORE) {  // phi_0^N, phi_1^N and phi^T of W^n (phi_2^N follows from them, mrd_math.cuh): 12 values per triangle
          Cell<R> *o = reinterpret_cast<Cell<R> *>(io.phi12 + b * 12 * T) + tid;
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            o[(h * 3 + 0) * T] = Cell<R>{pN[0][2 * h], pN[0][2 * h + 1]};
            o[(h * 3 + 1) * T] = Cell<R>{pN[1][2 * h], pN[1][2 * h + 1]};
            o[(h * 3 + 2) * T] = Cell<R>{pT[2 * h], pT[2 * h + 1]};
          }
        }
      } else {
        // eq. 57 / 61: Phi^T = |T|/3 sum_j dW_j/dt + (phi^T(W^n) + phi^T(W*))/2;  eq. 62 per node
        const Vec4<R> *sD = reinterpret_cast<const Vec4<R> *>(buf + L.oD);
        R oN[3][4], oT[4];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const Cell<R> c0 = cell[h * HOFF + tid], c1 = cell[h * HOFF + T + tid], c2 = cell[h * HOFF + 2 * T + tid];
          oN[0][2 * h] = c0.a; oN[0][2 * h + 1] = c0.b;
          oN[1][2 * h] = c1.a; oN[1][2 * h + 1] = c1.b;
          oT[2 * h] = c2.a; oT[2 * h + 1] = c2.b;
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) oN[2][c] = (oT[c] - oN[0][c]) - oN[1][c];   // as stage 1 formed phi_2^N: bitwise its value
#pragma unroll
        for (int c = 0; c < 4; ++c) X[c] = R(0.5) * (oT[c] + pT[c]);
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          Vec4<R> d = sD[l[i]];
          R m[4] = {a3 * d.x, a3 * d.y, a3 * d.z, a3 * d.w};
#pragma unroll
          for (int c = 0; c < 4; ++c) {
            X[c] += m[c];
            pN[i][c] = m[c] + R(0.5) * (pN[i][c] + oN[i][c]);
          }
        }
        if (lump) {  // selective lumping (eq. 66-67): E_i = sum_j (|T| d_ij/3 - m^G_ij) dW_j/dt = |T|/12 (3 dW_i - sum_j dW_j)
          Vec4<R> d0 = sD[l[0]], d1 = sD[l[1]], d2 = sD[l[2]];
          R sm[4] = {d0.x + d1.x + d2.x, d0.y + d1.y + d2.y, d0.z + d1.z + d2.z, d0.w + d1.w + d2.w};
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            Vec4<R> d = sD[l[i]];
            R dv[4] = {d.x, d.y, d.z, d.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) pN[i][c] += (R(0.25) * a3) * (R(3) * dv[c] - sm[c]);
          }
        }
      }
      // The nodal N residuals go to shared memory now (their final place for scheme N); the LDA residuals are then
      // produced and blended in place -- 24 fewer values live at once than blending from registers.
      R th[4] = {0, 0, 0, 0};
      if (SCHEME == MRD_SCHEME_B) blend_theta(X, pN, bvar, th);  // eq. 53 (+ C10); Bmax / Bmin: L503
      if (SCHEME == MRD_SCHEME_BX)                               // eq. 54-56: one theta from the shock sensor of this stage's state
        th[0] = th[1] = th[2] = th[3] = bx_theta(z, g, a3, lmax, bxL, bxInv);
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) cell[h * HOFF + i * T + tid] = Cell<R>{pN[i][2 * h], pN[i][2 * h + 1]};
      if (SCHEME != MRD_SCHEME_N) {
        // eq. 50-51 (stage 2: eq. 63 with eq. 65): L_i = -K_i^+ N-hat X;  eq. 52: B_i = L_i + Theta (N_i - L_i)
        R q[4], Lw[3][4];
        to_symmetrising(gamma - R(1), kk, X, q);
        lda_from_symmetrised(kk, g, X, q, Lw);
        if (lump) {  // the same anti-diffusive term on the LDA residual (L567)
          const Vec4<R> *sD = reinterpret_cast<const Vec4<R> *>(buf + L.oD);
          Vec4<R> d0 = sD[l[0]], d1 = sD[l[1]], d2 = sD[l[2]];
          R sm[4] = {d0.x + d1.x + d2.x, d0.y + d1.y + d2.y, d0.z + d1.z + d2.z, d0.w + d1.w + d2.w};
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            Vec4<R> d = sD[l[i]];
            R dv[4] = {d.x, d.y, d.z, d.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) Lw[i][c] += (R(0.25) * a3) * (R(3) * dv[c] - sm[c]);
          }
        }
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            Cell<R> *r = cell + h * HOFF + i * T + tid;
            if (SCHEME == MRD_SCHEME_B || SCHEME == MRD_SCHEME_BX) {
              const Cell<R> n = *r;
              *r = Cell<R>{Lw[i][2 * h] + th[2 * h] * (n.a - Lw[i][2 * h]), Lw[i][2 * h + 1] + th[2 * h + 1] * (n.b - Lw[i][2 * h + 1])};
            } else {
              *r = Cell<R>{Lw[i][2 * h], Lw[i][2 * h + 1]};
            }
          }
      }
      if (STAGE == 1 && io.phi_dbg && valid) {
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          const Cell<R> c0 = cell[i * T + tid], c1 = cell[HOFF + i * T + tid];
          st4(&io.phi_dbg[3 * t + i], Vec4<R>{c0.a, c0.b, c1.a, c1.b});
        }
        io.sT_dbg[t] = st;
      }
    }
    if (!valid) {  // padding thread of the last tile: contributes nothing
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int h = 0; h < 2; ++h) cell[h * HOFF + i * T + tid] = Cell<R>{R(0), R(0)};
      st = R(0);
    }
    if (STAGE == 1) {
      sTx[tid] = st;
      sTx[T + tid] = st;
      sTx[2 * T + tid] = st;
    }
    __syncthreads();
    // ---- epilogue: per slot the ascending sum of its tile-local incidences; one partial per slot leaves the SM
    {
      const uint16_t *boff = plan + 4 * T, *ent = plan + 4 * T + td.offn;
      for (int j = tid; j < ns; j += T) {   // (padding slots have no incidences: their partial is zero and nobody reads it)
        R a[4], S;
        slot_sum<R, T, STAGE == 1>(cell, sTx, ent, boff[j], boff[j + 1], a, S);
        st4(&io.part[s0 + j], Vec4<R>{a[0], a[1], a[2], a[3]});
        if (STAGE == 1) io.partS[s0 + j] = S;
      }
    }
    // No second block barrier: a warp that is done goes on to the next tile (the other buffer, the other residual
    // area) while slower warps finish this epilogue; the LAST warp to leave refills buffer `cur` with tile k+2.
    // (Nobody runs more than one tile ahead: the barrier above needs every warp.)
    __syncwarp();
    if ((tid & 31) == 0) {
      __threadfence_block();
      if (atomicAdd(&done[cur], 1u) == NW - 1) {
        __threadfence_block();
        done[cur] = 0;
        const int64_t b2 = nb + gridDim.x;
        if (b2 < td.ntile) {
          fence_proxy_async();  // buffer `cur` was read through the generic proxy
          tile_stage_in<R, STAGE, GTAB>(td, L, buf, &bar[cur], b2, __ldg(td.tile_info + b2), __ldg(td.tile_info + b2 + 1), io.slotZ, io.slotS,
                                        io.slotD, io.phi12);
        }
      }
    }
    i0 = use_info(n0);
    i1 = use_info(n1);
  }
  if (bad) atomicOr(status, 1);
}

// ---------------------------------------------------------------------------------------------
// vertex side of the fused path: add the vertex's partials (ascending slot order)
// ---------------------------------------------------------------------------------------------
// S7 on the fused path: d_i = 2 V_i / sum of the vertex's partial s_T sums (eq. 44), block minimum -> atomicMin
template <class R>
__global__ void __launch_bounds__(256)
slot_dt_kernel(MeshDev<R> m, TileDev<R> td, Ctl *__restrict__ ctl, const R *__restrict__ partS) {
  MRD_CTL_GUARD(ctl)
  // grid-stride: a few blocks per SM, so that only ~10^3 atomicMin hit the one address (65 536 one-per-block atomics
  // serialise in L2 and took longer than the gather itself)
  // Four vertices per thread and pass, their loads issued together (the gather is a chain vslot_off -> vslot_ent -> partS of
  // dependent loads; every resident thread slot is taken already, so more loads in flight have to come from each thread).
  // The sum of a vertex still runs over its slots in ascending order.
  double d = __longlong_as_double(0x7FF0000000000000ll);
  const int64_t stride = (int64_t)gridDim.x * blockDim.x;
  constexpr int U = 4;
  for (int64_t i0 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i0 < m.nv; i0 += U * stride) {
    int32_t q0[U], q1[U], ent[U][4];
    R ps[U][4], vol[U];
    bool on[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int64_t i = i0 + u * stride;
      on[u] = i < m.nv && !(m.frozen && m.frozen[i] == 2);   // (2: halo vertex of a partition, its fan is incomplete here)
      q0[u] = on[u] ? __ldg(td.vslot_off + i) : 0;
      q1[u] = on[u] ? __ldg(td.vslot_off + i + 1) : 0;
      vol[u] = on[u] ? __ldg(m.vol + i) : R(1);
    }
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int k = 0; k < 4; ++k) ent[u][k] = q0[u] + k < q1[u] ? __ldg(td.vslot_ent + q0[u] + k) : -1;
#pragma unroll
    for (int u = 0; u < U; ++u)
#pragma unroll
      for (int k = 0; k < 4; ++k) ps[u][k] = ent[u][k] >= 0 ? __ldg(partS + ent[u][k]) : R(0);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (!on[u]) continue;
      R S = 0;
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (q0[u] + k < q1[u]) S += ps[u][k];
      for (int32_t q = q0[u] + 4; q < q1[u]; ++q) S += __ldg(partS + __ldg(td.vslot_ent + q));
      d = fmin(d, 2.0 * (double)vol[u] / (double)S);
    }
  }
  block_min_to_global(d, &ctl->dmin_bits);
}

// S8 / S10 / S12 on the fused path: gather the vertex's partials (ascending slot order), add the wall terms, update.
//   MODE 0: stage 1 of RK2   W* = W^n - dt/V sum        (Win -> Wout; Z*, dW/dt to the slots)
//   MODE 1: single stage     W^{n+1} = W^n - dt/V sum   (Win -> Wout; Z, |v|+c to the slots)        eq. 43
//   MODE 2: stage 2 of RK2   W^{n+1} = W* - dt/V sum    (in place: Win == Wout; Z, |v|+c to the slots) eq. 61
// Launch shape (measured at 4096^2, profiles/r02_experiments.md section 7): blocks of 128 threads; in fp64 enough of them resident
// that the three-level gather (vslot_off -> vslot_ent -> part) has more loads in flight -- 40 registers for the stage-1 update
// (24 bytes spilled), 32 for the final update (40 bytes spilled): 0.614 -> 0.585 ms and 0.509 -> 0.472 ms.  In fp32 the register
// caps lose (0.336 -> 0.395 ms for the stage-1 update), so there is no minimum (0).
template <class R> struct VtxShape;
template <> struct VtxShape<double> { static constexpr int threads = 128, minb_update = 12, minb_final = 16; };
template <> struct VtxShape<float> { static constexpr int threads = 128, minb_update = 0, minb_final = 0; };
template <class R, int MODE>
__global__ void __launch_bounds__(VtxShape<R>::threads, MODE == 2 ? VtxShape<R>::minb_final : VtxShape<R>::minb_update)
slot_gather_update_kernel(MeshDev<R> m, TileDev<R> td, R gamma, const Ctl *__restrict__ ctl,
                          const Vec4<R> *__restrict__ part, const Vec4<R> *__restrict__ wall_acc, const Vec4<R> *Win,
                          Vec4<R> *Wout, VertexSink<R> sink, int *status) {
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
  Vec4<R> w = Win[i];
  bool fr = m.frozen ? (m.frozen[i] != 0) : false;
  vertex_finish<R, MODE == 0>(gamma, dt, __ldg(m.vol + i), fr, w, a, i, Wout, sink, status);
}

}  // namespace mrd
