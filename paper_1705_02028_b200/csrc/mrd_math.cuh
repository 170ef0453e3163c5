// mrd_math.cuh -- per-triangle and per-vertex arithmetic of the residual-distribution sweep (device).
//
// Written from PAPER.md (arXiv:1705.02028); shares nothing with oracle/.  Templated on the scalar
// R = double | float.  The formulation is the exact similarity transform of the paper's matrices
// into the symmetrising variables dQ = (dp/c, du, dv, dp - c^2 drho) (unit reference density), in
// which K_i = (l_i/2) [[w, c n^T, 0], [c n, w I, 0], [0, 0, w]]:
//   - K_i^(+/-) (eq. 40-42; App. A eq. A10-A25) are applied as characteristic
//     projections with a = (l1+l2)/2, b = (l1-l2)/2 (the paper's l_12) and a - l3 (its l_123);
//   - sum_j K_j^- becomes a symmetric 3x3 block plus the entropy scalar, so N-hat (eq. 49)
//     is a 3x3 cofactor inverse and a reciprocal; the stagnation rule C8 is the scalar's 0/0 -> 0;
//   - residuals are mapped back to conserved variables before the blend of eq. 52-53 (L493-L503),
//     which is defined per conserved component.
#pragma once
#include <cuda_runtime.h>

namespace mrd {

// ---------------------------------------------------------------------------------------------
// scalar helpers: reciprocal / reciprocal square root by hardware seed + Newton steps (the fp64
// division and sqrt of CUDA are IEEE-rounded subroutine calls; 1-2 ulp is enough here, see
// DESIGN.md "Tolerance").  Arguments are positive and normal wherever these are used.
// ---------------------------------------------------------------------------------------------
template <class R> struct Fast;

template <> struct Fast<double> {
  static __device__ __forceinline__ double rcp(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    e = fma(-x, r, 1.0);
    r = fma(r, e, r);
    return r;
  }
  static __device__ __forceinline__ double rsqrt(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double hx = 0.5 * x;
    double e = fma(-hx * y, y, 0.5);
    y = fma(y, e, y);
    e = fma(-hx * y, y, 0.5);
    y = fma(y, e, y);
    return y;
  }
  // sqrt(x) for x >= 0 (exactly 0 for x = 0), given nothing else
  static __device__ __forceinline__ double sqrt0(double x) {
    if (!(x > 0.0)) return 0.0;
    double y = rsqrt(x);
    double s = x * y;
    double r = fma(-s, s, x);
    return fma(r, 0.5 * y, s);
  }
  static __device__ __forceinline__ double abs(double x) { return fabs(x); }
  static __device__ __forceinline__ double max(double a, double b) { return fmax(a, b); }
  static __device__ __forceinline__ double min(double a, double b) { return fmin(a, b); }
  static __device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
};

template <> struct Fast<float> {
  static __device__ __forceinline__ float rcp(float x) { return __frcp_rn(x); }
  static __device__ __forceinline__ float rsqrt(float x) { return rsqrtf(x); }
  static __device__ __forceinline__ float sqrt0(float x) { return x > 0.0f ? __fsqrt_rn(x) : 0.0f; }
  static __device__ __forceinline__ float abs(float x) { return fabsf(x); }
  static __device__ __forceinline__ float max(float a, float b) { return fmaxf(a, b); }
  static __device__ __forceinline__ float min(float a, float b) { return fminf(a, b); }
  static __device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
};

template <class R> struct Vec4 { R x, y, z, w; };
template <> struct __align__(32) Vec4<double> { double x, y, z, w; };
template <> struct __align__(16) Vec4<float> { float x, y, z, w; };

template <class R> __device__ __forceinline__ Vec4<R> ld4(const Vec4<R> *p) {
  return *p;
}
template <> __device__ __forceinline__ Vec4<double> ld4<double>(const Vec4<double> *p) {
  const double2 *q = reinterpret_cast<const double2 *>(p);
  double2 a = __ldg(q), b = __ldg(q + 1);
  return Vec4<double>{a.x, a.y, b.x, b.y};
}
template <> __device__ __forceinline__ Vec4<float> ld4<float>(const Vec4<float> *p) {
  float4 a = __ldg(reinterpret_cast<const float4 *>(p));
  return Vec4<float>{a.x, a.y, a.z, a.w};
}
template <class R> __device__ __forceinline__ void st4(Vec4<R> *p, const Vec4<R> &v);
template <> __device__ __forceinline__ void st4<double>(Vec4<double> *p, const Vec4<double> &v) {
  double2 *q = reinterpret_cast<double2 *>(p);
  q[0] = make_double2(v.x, v.y);
  q[1] = make_double2(v.z, v.w);
}
template <> __device__ __forceinline__ void st4<float>(Vec4<float> *p, const Vec4<float> &v) {
  *reinterpret_cast<float4 *>(p) = make_float4(v.x, v.y, v.z, v.w);
}

// ---------------------------------------------------------------------------------------------
// Per-vertex quantities: parameter vector Z = sqrt(rho) (1, u, v, h) (eq. 20
// L290-L294 and its 2D analogue L419, reading C1) with p from eq. 10 (L224), and the signal speed
// |v| + c, c^2 = gamma p / rho, of eq. 45 (L447-L449, reading C14).  Returns false when rho <= 0
// or p <= 0.
// ---------------------------------------------------------------------------------------------
template <class R>
__device__ __forceinline__ bool vertex_prepare(R gamma, const Vec4<R> &W, Vec4<R> &Z, R &speed, R &p_out) {
  using F = Fast<R>;
  const R g1 = gamma - R(1);
  R rho = W.x;
  bool ok = rho > R(0);
  R rs = ok ? rho : R(1);
  R ir = F::rcp(rs);
  R u = W.y * ir, v = W.z * ir;
  R ke2 = W.y * u + W.z * v;  // rho (u^2 + v^2)
  R p = g1 * (W.w - R(0.5) * ke2);
  p_out = p;
  ok = ok && (p > R(0));
  R ps = ok ? p : R(1);
  R h = (W.w + ps) * ir;
  R isr = F::rsqrt(rs);
  R s = rs * isr;  // sqrt(rho)
  s = F::fma_(F::fma_(-s, s, rs), R(0.5) * isr, s);
  Z.x = s;
  Z.y = s * u;
  Z.z = s * v;
  Z.w = s * h;
  speed = F::sqrt0(u * u + v * v) + F::sqrt0(gamma * ps * ir);
  return ok;
}

// fp64 per-vertex quantities, operation by operation as eq. 10, 20, 45 are written and without FMA contraction of
// the formulas themselves.  Quotients by rho use ONE reciprocal plus a residual correction each
// (q = a r; q += fma(-q, rho, a) r: correctly rounded except in rare half-ulp cases), square roots the analogous
// correction of x rsqrt(x).  This matters on fine meshes: the triangle kernels difference Z between neighbouring
// vertices (delta = Z_j - Z_1 ~ h), so an ulp of error in Z is 1/h ulps in every residual; with these forms Z and the
// signal speed equal the oracle's IEEE results bit for bit in all but rare cases, at a quarter of the instructions
// of CUDA's IEEE division/sqrt subroutines (the update kernels became fp64-bound with those).
__device__ __forceinline__ double div_by(double a, double rho, double r) {
  double q = a * r;
  return fma(fma(-q, rho, a), r, q);
}
__device__ __forceinline__ double sqrt_near(double x) {
  if (!(x > 0.0)) return 0.0;
  double y = Fast<double>::rsqrt(x);
  double sq = x * y;
  return fma(fma(-sq, sq, x), 0.5 * y, sq);
}
template <>
__device__ __forceinline__ bool vertex_prepare<double>(double gamma, const Vec4<double> &W, Vec4<double> &Z, double &speed,
                                                       double &p_out) {
  const double g1 = gamma - 1.0;
  double rho = W.x;
  bool ok = rho > 0.0;
  double rs = ok ? rho : 1.0;
  double r = Fast<double>::rcp(rs);
  r = fma(fma(-rs, r, 1.0), r, r);
  double u = div_by(W.y, rs, r), v = div_by(W.z, rs, r);
  double m2 = __dadd_rn(__dmul_rn(W.y, W.y), __dmul_rn(W.z, W.z));
  double p = __dmul_rn(g1, __dadd_rn(W.w, -div_by(__dmul_rn(0.5, m2), rs, r)));
  p_out = p;
  ok = ok && (p > 0.0);
  double ps = ok ? p : 1.0;
  double h = div_by(__dadd_rn(W.w, ps), rs, r);
  double sr = sqrt_near(rs);
  Z.x = sr;
  Z.y = __dmul_rn(sr, u);
  Z.z = __dmul_rn(sr, v);
  Z.w = __dmul_rn(sr, h);
  speed = __dadd_rn(sqrt_near(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v))), sqrt_near(div_by(__dmul_rn(gamma, ps), rs, r)));
  return ok;
}

// ---------------------------------------------------------------------------------------------
// One triangle at one state: everything the distribution needs.
// ---------------------------------------------------------------------------------------------
template <class R> struct TriGeom {
  R nx[3], ny[3];  // unit inward normal of the edge opposite node i (eq. 35; reading C4)
  R hl[3];         // l_i / 2 (eq. 37 with d = 2)
};

template <class R> struct TriCore {
  // linearised state (eq. 39)
  R u, v, hq2 /* (u^2+v^2)/2 */, c, c2, ic /* 1/c */, ic2, cg /* c/(gamma-1) */;
  // positive parts per edge: a+ = (l1+ + l2+)/2, b+ = (l1+ - l2+)/2, l3+
  R ap[3], bp[3], l3p[3];
  // N-hat (eq. 49): symmetric 3x3 inverse (00,01,02,11,12,22) and the entropy reciprocal
  R n00, n01, n02, n11, n12, n22, ns;
  bool ok;
  bool stagnant;  // stagnation rule C8 applied: the entropy part of N-hat is 0
};

// y = K x in the rotated frame of edge (nx, ny) with coefficients (a, b, l3):
//   y0 = a x0 + b xn,  yn = b x0 + a xn,  yt = l3 xt,  y3 = l3 x3,  (y1, y2) = rotation back of (yn, yt).
// ACC = false: y is overwritten; ACC = true: added to y.  Written as explicit FMA chains (the fp64 pipe is the
// binding unit of the sweep: every DADD saved counts).
template <bool ACC, class R>
__device__ __forceinline__ void apply_split(R a, R b, R l3, R nx, R ny, const R x[4], R y[4]) {
  using F = Fast<R>;
  R xn = F::fma_(nx, x[1], ny * x[2]);
  R xt = F::fma_(nx, x[2], -(ny * x[1]));
  R yn = F::fma_(b, x[0], a * xn);
  R yt = l3 * xt;
  if (ACC) {
    y[0] = F::fma_(a, x[0], F::fma_(b, xn, y[0]));
    y[1] = F::fma_(nx, yn, F::fma_(-ny, yt, y[1]));
    y[2] = F::fma_(ny, yn, F::fma_(nx, yt, y[2]));
    y[3] = F::fma_(l3, x[3], y[3]);
  } else {
    y[0] = F::fma_(a, x[0], b * xn);
    y[1] = F::fma_(nx, yn, -(ny * yt));
    y[2] = F::fma_(ny, yn, nx * yt);
    y[3] = l3 * x[3];
  }
}
// the unsplit K_i = (l_i/2)(A nx + B ny) applied to x: in symmetrising variables
//   y0 = wl x0 + cl (n.x),  (y1, y2) = wl (x1, x2) + cl x0 (nx, ny),  y3 = wl x3      (wl = l/2 w, cl = l/2 c)
template <bool ACC, class R>
__device__ __forceinline__ void apply_full(R wl, R cl, R nx, R ny, const R x[4], R y[4]) {
  using F = Fast<R>;
  R xn = F::fma_(nx, x[1], ny * x[2]);
  R t = cl * x[0];
  if (ACC) {
    y[0] = F::fma_(wl, x[0], F::fma_(cl, xn, y[0]));
    y[1] = F::fma_(wl, x[1], F::fma_(t, nx, y[1]));
    y[2] = F::fma_(wl, x[2], F::fma_(t, ny, y[2]));
    y[3] = F::fma_(wl, x[3], y[3]);
  } else {
    y[0] = F::fma_(wl, x[0], cl * xn);
    y[1] = F::fma_(wl, x[1], t * nx);
    y[2] = F::fma_(wl, x[2], t * ny);
    y[3] = wl * x[3];
  }
}

// symmetrising variables -> conserved variables (unit reference density)
template <class R> __device__ __forceinline__ void to_conserved(const TriCore<R> &k, const R q[4], R w[4]) {
  R drho = (k.c * q[0] - q[3]) * k.ic2;
  w[0] = drho;
  w[1] = k.u * drho + q[1];
  w[2] = k.v * drho + q[2];
  w[3] = k.cg * q[0] + k.hq2 * drho + k.u * q[1] + k.v * q[2];
}
// conserved -> symmetrising
template <class R> __device__ __forceinline__ void to_symmetrising(R g1, const TriCore<R> &k, const R w[4], R q[4]) {
  R dp = g1 * (w[3] - k.u * w[1] - k.v * w[2] + k.hq2 * w[0]);
  q[0] = dp * k.ic;
  q[1] = w[1] - k.u * w[0];
  q[2] = w[2] - k.v * w[0];
  q[3] = dp - k.c2 * w[0];
}

// S2-S5: from the three parameter vectors and the geometry to phi^T (eq. 36) and phi_i^N (eq. 48),
// both in conserved variables; `k` keeps what beta_i = -K_i^+ N-hat (eq. 51) needs.
template <class R>
__device__ __forceinline__ void triangle_core(R gamma, const Vec4<R> Z[3], const TriGeom<R> &g, TriCore<R> &k,
                                              R phiT[4], R phiN[3][4]) {
  using F = Fast<R>;
  const R g1 = gamma - R(1);
  const R third = R(1) / R(3);
  // eq. 39: Zbar, and u, v, h, c of the linearised state
  R zb0 = (Z[0].x + Z[1].x + Z[2].x) * third;
  R zb1 = (Z[0].y + Z[1].y + Z[2].y) * third;
  R zb2 = (Z[0].z + Z[1].z + Z[2].z) * third;
  R zb3 = (Z[0].w + Z[1].w + Z[2].w) * third;
  R iz = F::rcp(zb0);
  k.u = zb1 * iz;
  k.v = zb2 * iz;
  R h = zb3 * iz;
  k.hq2 = R(0.5) * (k.u * k.u + k.v * k.v);
  R c2 = g1 * (h - k.hq2);
  k.ok = c2 > R(0);
  c2 = k.ok ? c2 : R(1);
  k.c2 = c2;
  k.ic = F::rsqrt(c2);
  k.c = c2 * k.ic;
  k.ic2 = k.ic * k.ic;
  k.cg = k.c * F::rcp(g1);  // (an IEEE division of two block-uniform values costs ~25 instructions and a branch per thread)

  // O3 (reading C3): delta_j = D(Zbar)(Z_j - Z_0) mapped to symmetrising variables; the composition is
  //   drho = 2 zb0 d0, du = zb0 d1 - zb1 d0, dv = zb0 d2 - zb2 d0,
  //   dp = (g1/gamma) (zb3 d0 + zb0 d3 - zb1 d1 - zb2 d2)
  // (exactly zero when Z_j == Z_0, so uniform flow has zero residual, L237)
  const R gg = g1 * F::rcp(gamma);
  R dq[3][4];
  dq[0][0] = dq[0][1] = dq[0][2] = dq[0][3] = R(0);
#pragma unroll
  for (int j = 1; j < 3; ++j) {
    R d0 = Z[j].x - Z[0].x, d1 = Z[j].y - Z[0].y, d2 = Z[j].z - Z[0].z, d3 = Z[j].w - Z[0].w;
    R dp = gg * (zb3 * d0 + zb0 * d3 - zb1 * d1 - zb2 * d2);
    R drho = R(2) * zb0 * d0;
    dq[j][0] = dp * k.ic;
    dq[j][1] = zb0 * d1 - zb1 * d0;
    dq[j][2] = zb0 * d2 - zb2 * d0;
    dq[j][3] = dp - c2 * drho;
  }

  // O4: per edge the split eigenvalues (eq. 41-42) and the sums over edges.  With q = l_i/8 the halves
  // lambda^(+/-)/2 = q lambda +/- |q lambda| come out of one addition each (scaling by powers of two is exact).
  R s00 = 0, s01 = 0, s02 = 0, s11 = 0, s12 = 0, s22 = 0, s33 = 0;
  R accm[4] = {0, 0, 0, 0};   // sum_j K_j^- dq_j
  R phiq[4] = {0, 0, 0, 0};   // sum_j K_j dq_j = phi^T (eq. 36)
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    R nx = g.nx[i], ny = g.ny[i], hl = g.hl[i];
    R wn = F::fma_(k.u, nx, k.v * ny);
    R hq = R(0.25) * hl;
    R wq = hq * wn, cq = hq * k.c;            // (l_i/8) w, (l_i/8) c
    R l1q = wq + cq, l2q = wq - cq;
    R p1 = l1q + F::abs(l1q), p2 = l2q + F::abs(l2q);  // l1+/2, l2+/2
    R m1 = l1q - F::abs(l1q), m2 = l2q - F::abs(l2q);  // l1-/2, l2-/2
    R ap = p1 + p2, bp = p1 - p2, am = m1 + m2, bm = m1 - m2;
    R l3h = wq + wq;                          // l3/2
    R l3p = l3h + F::abs(l3h), l3m = l3h - F::abs(l3h);
    k.ap[i] = ap;
    k.bp[i] = bp;
    k.l3p[i] = l3p;
    // with nxx + nyy = 1: s11 = sum_j (a- - l3-) nxx + sum_j l3-, s22 likewise with nyy (two instructions fewer per edge
    // than accumulating a- nxx + l3- nyy); the entropy sum s33 is added after the loop
    R nxx = nx * nx, nyy = ny * ny, nxy = nx * ny;
    R dm = am - l3m;
    if (i == 0) {  // (0 + x is not x for x = -0, so the compiler keeps additions to a zero accumulator)
      s00 = am;
      s01 = bm * nx;
      s02 = bm * ny;
      s11 = dm * nxx;
      s12 = dm * nxy;
      s22 = dm * nyy;
      s33 = l3m;
    } else {
      s00 += am;
      s01 = F::fma_(bm, nx, s01);
      s02 = F::fma_(bm, ny, s02);
      s11 = F::fma_(dm, nxx, s11);
      s12 = F::fma_(dm, nxy, s12);
      s22 = F::fma_(dm, nyy, s22);
      s33 += l3m;
    }
    if (i == 1) {
      apply_split<false>(am, bm, l3m, nx, ny, dq[i], accm);
      apply_full<false>(hl * wn, hl * k.c, nx, ny, dq[i], phiq);
    } else if (i == 2) {
      apply_split<true>(am, bm, l3m, nx, ny, dq[i], accm);
      apply_full<true>(hl * wn, hl * k.c, nx, ny, dq[i], phiq);
    }
  }

  s11 += s33;
  s22 += s33;
  // O5: N-hat = (sum K^-)^-1: cofactor inverse of the symmetric 3x3 block, reciprocal of the entropy
  // scalar; stagnation rule (reading C8): u^2 + v^2 <= (1e-14 c)^2 -> entropy part of N-hat = 0
  R c00 = s11 * s22 - s12 * s12;
  R c01 = s02 * s12 - s01 * s22;
  R c02 = s01 * s12 - s02 * s11;
  R c11 = s00 * s22 - s02 * s02;
  R c12 = s01 * s02 - s00 * s12;
  R c22 = s00 * s11 - s01 * s01;
  R det = s00 * c00 + s01 * c01 + s02 * c02;
  R idet = F::rcp(det);  // det < 0 (negative definite block); rcp seeds handle the sign
  k.n00 = c00 * idet; k.n01 = c01 * idet; k.n02 = c02 * idet;
  k.n11 = c11 * idet; k.n12 = c12 * idet; k.n22 = c22 * idet;
  const R eps = R(1e-14);
  const bool stagnant = (R(2) * k.hq2 <= (eps * eps) * c2) || !(s33 < R(0));
  k.stagnant = stagnant;
  k.ns = stagnant ? R(0) : F::rcp(stagnant ? R(-1) : s33);

  // eq. 48: phi_i^N = K_i^+ (dq_i - N-hat sum_j K_j^- dq_j)
  R win[4];
  win[0] = k.n00 * accm[0] + k.n01 * accm[1] + k.n02 * accm[2];
  win[1] = k.n01 * accm[0] + k.n11 * accm[1] + k.n12 * accm[2];
  win[2] = k.n02 * accm[0] + k.n12 * accm[1] + k.n22 * accm[2];
  win[3] = k.ns * accm[3];
  // nodes 0 and 1 directly; node 2 from sum_i phi_i^N = phi^T, which holds identically because sum_i K_i = 0 and
  // N-hat sum_j K_j^- = I (in the stagnation case both entropy parts vanish): 8 additions instead of ~26 operations
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    R d[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) d[c] = i == 0 ? -win[c] : dq[i][c] - win[c];  // dq_0 = 0
    R y[4];
    apply_split<false>(k.ap[i], k.bp[i], k.l3p[i], g.nx[i], g.ny[i], d, y);
    to_conserved(k, y, phiN[i]);
  }
  to_conserved(k, phiq, phiT);
#pragma unroll
  for (int c = 0; c < 4; ++c) phiN[2][c] = (phiT[c] - phiN[0][c]) - phiN[1][c];
}

// eq. 50-51: out_i = beta_i X = -K_i^+ N-hat X for a conserved-variable vector X (phi^T in stage 1,
// Phi^T in stage 2: eq. 63 with eq. 65, reading C12).  Nodes 0 and 1 directly; node 2 from sum_i beta_i = I, which holds
// identically (sum_i K_i^+ = -sum_j K_j^- and N-hat is its inverse) except for the entropy component under the
// stagnation rule C8, where that part of N-hat is 0: there the three residuals add up to X minus its entropy part
// M (0, 0, 0, q_3) = -(q_3 / c^2) (1, u, v, (u^2 + v^2)/2).  8-13 instructions instead of the ~22 of a third projection.
template <class R>
__device__ __forceinline__ void lda_from_symmetrised(const TriCore<R> &k, const TriGeom<R> &g, const R X[4], const R q[4], R out[3][4]) {
  R y[4];
  y[0] = -(k.n00 * q[0] + k.n01 * q[1] + k.n02 * q[2]);
  y[1] = -(k.n01 * q[0] + k.n11 * q[1] + k.n12 * q[2]);
  y[2] = -(k.n02 * q[0] + k.n12 * q[1] + k.n22 * q[2]);
  y[3] = -(k.ns * q[3]);
#pragma unroll
  for (int i = 0; i < 2; ++i) {
    R z[4];
    apply_split<false>(k.ap[i], k.bp[i], k.l3p[i], g.nx[i], g.ny[i], y, z);
    to_conserved(k, z, out[i]);
  }
  const R e3 = k.stagnant ? q[3] * k.ic2 : R(0);
  out[2][0] = ((X[0] + e3) - out[0][0]) - out[1][0];
  out[2][1] = (Fast<R>::fma_(k.u, e3, X[1]) - out[0][1]) - out[1][1];
  out[2][2] = (Fast<R>::fma_(k.v, e3, X[2]) - out[0][2]) - out[1][2];
  out[2][3] = (Fast<R>::fma_(k.hq2, e3, X[3]) - out[0][3]) - out[1][3];
}
template <class R>
__device__ __forceinline__ void apply_beta(R gamma, const TriCore<R> &k, const TriGeom<R> &g, const R X[4], R out[3][4]) {
  R q[4];
  to_symmetrising(gamma - R(1), k, X, q);
  lda_from_symmetrised(k, g, X, q, out);
}

// eq. 52-53 (+ reading C10): Theta_kk = min(1, |X_k| / sum_j |N_j,k|), 0 when the denominator is 0;
// B_i = Theta N_i + (1 - Theta) LDA_i, written over N.
// Theta_kk of eq. 53 for all four components; bvar 1 / 2: all entries replaced by their maximum / minimum (Bmax / Bmin,
// L503)
// range in which the product of the four blend denominators (and its reciprocal) is safely a normal number
template <class R> struct ProductRange;
template <> struct ProductRange<double> {
  static __device__ __forceinline__ double lo() { return 1e-290; }
  static __device__ __forceinline__ double hi() { return 1e290; }
};
template <> struct ProductRange<float> {   // (the fp32 variant takes one reciprocal per component: never used)
  static __device__ __forceinline__ float lo() { return 1e-30f; }
  static __device__ __forceinline__ float hi() { return 1e30f; }
};
template <class R> __device__ __forceinline__ void blend_theta(const R X[4], const R N[3][4], int bvar, R th[4]) {
  using F = Fast<R>;
  // Theta = min(1, |X| / den), and 0 on a zero denominator (C10).  den = 0 means every nodal residual is exactly 0,
  // which makes X and the LDA residuals exactly 0 too, so the value taken there (1) changes nothing: B_i = 0.
  R den[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) den[c] = F::abs(N[0][c]) + F::abs(N[1][c]) + F::abs(N[2][c]);
  if (sizeof(R) == 8) {
    // fp64: the four reciprocals from ONE (seed + Newton) reciprocal of the product of the denominators (the seed
    // instruction and its fix-ups are the expensive part): 1/d_0 = d_1 (d_2 d_3) / P, ...  Zero denominators are replaced
    // by 1 (their Theta is 1 whatever the quotient); should the product leave the normal range (denominators below
    // ~1e-75 each), the components fall back to one reciprocal each.
    R d[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) d[c] = den[c] > R(0) ? den[c] : R(1);
    const R p01 = d[0] * d[1], p23 = d[2] * d[3], P = p01 * p23;
    if (P > ProductRange<R>::lo() && P < ProductRange<R>::hi()) {
      const R r = F::rcp(P);
      const R r01 = r * p23, r23 = r * p01;   // 1 / (d0 d1), 1 / (d2 d3)
      const R inv[4] = {r01 * d[1], r01 * d[0], r23 * d[3], r23 * d[2]};
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        R t = F::abs(X[c]) * inv[c];
        th[c] = (den[c] > R(0) && t < R(1)) ? t : R(1);
      }
    } else {
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        R t = F::abs(X[c]) * F::rcp(d[c]);
        th[c] = (den[c] > R(0) && t < R(1)) ? t : R(1);
      }
    }
  } else {
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      // Written so that a zero or denormal denominator (reciprocal inf, product inf or NaN) also lands on 1.
      R t = F::abs(X[c]) * F::rcp(den[c]);
      th[c] = t < R(1) ? t : R(1);
    }
  }
  if (bvar != 0) {
    R hi = F::max(F::max(th[0], th[1]), F::max(th[2], th[3]));
    R lo = F::min(F::min(th[0], th[1]), F::min(th[2], th[3]));
    R t = bvar == 1 ? hi : lo;
    th[0] = th[1] = th[2] = th[3] = t;
  }
}
// Bx (eq. 54-56; readings C23-C26): theta = min(1, s^2 l_max / L), s = (-L div v / (|v|_max - |v|_min))^+,
// div v of the linear interpolant of the vertex velocities = sum_j (u_j . n_j) l_j / (2|T|) (inward normals).
// Z = sqrt(rho) (1, u, v, h), so u_j = Z_j.y / Z_j.x.  area3 = |T|/3, hl = l/2; inv_range = 1 / (|v|_max - |v|_min) or 0.
template <class R>
__device__ __forceinline__ R bx_theta(const Vec4<R> z[3], const TriGeom<R> &g, R area3, R lmax, R Ldom, R inv_range) {
  using F = Fast<R>;
  R acc = R(0);
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    R iz = F::rcp(z[j].x);
    acc = F::fma_(F::fma_(z[j].y * iz, g.nx[j], (z[j].z * iz) * g.ny[j]), g.hl[j], acc);
  }
  R div = acc * F::rcp(R(3) * area3);
  R s = F::max(R(0), -(Ldom * div) * inv_range);
  R t = s * s * (lmax * F::rcp(Ldom));
  return t < R(1) ? t : R(1);
}

template <class R> __device__ __forceinline__ void blend(const R X[4], R N[3][4], const R L[3][4], int bvar) {
  R th[4];
  blend_theta(X, N, bvar, th);
#pragma unroll
  for (int c = 0; c < 4; ++c)
#pragma unroll
    for (int i = 0; i < 3; ++i) N[i][c] = L[i][c] + th[c] * (N[i][c] - L[i][c]);
}

}  // namespace mrd
