// mrd_predicates.cuh -- the exact geometric predicates of the mesh-generation layer as device functions (section 4.1.3,
// L665-L667; eq. 3, eq. 5): floating-point filters with a rigorous error bound, and the determinants in floating-point
// expansion arithmetic (error-free transformations TwoSum / TwoProduct with FMA; sums of non-overlapping components with zero
// elimination).  The sign of an expansion is the sign of its largest component.  Used by mrd_meshgen.cu (predicate entry
// points, Delaunay triangulator, point location).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

namespace mrdgen {

// ------------------------------------------------------------------------------------------------------------------
// Expansion arithmetic (device).  An expansion is a sum of doubles e[0..n) that do not overlap, in increasing magnitude, zeros
// removed.  All operations below are exact.
// ------------------------------------------------------------------------------------------------------------------
static __device__ __forceinline__ void two_sum(double a, double b, double &s, double &e) {
  s = __dadd_rn(a, b);
  const double bb = __dsub_rn(s, a);
  e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
static __device__ __forceinline__ void two_diff(double a, double b, double &s, double &e) { two_sum(a, -b, s, e); }
static __device__ __forceinline__ void two_prod(double a, double b, double &p, double &e) {
  p = __dmul_rn(a, b);
  e = __fma_rn(a, b, -p);
}
// h = e + b (e: expansion of length n, b: any double); returns the new length.  h may alias e.
static __device__ int grow(const double *e, int n, double b, double *h) {
  double Q = b;
  int m = 0;
  for (int i = 0; i < n; ++i) {
    double s, lo;
    two_sum(Q, e[i], s, lo);
    Q = s;
    if (lo != 0.0) h[m++] = lo;
  }
  if (Q != 0.0 || m == 0) h[m++] = Q;
  return m;
}
// e += f (both expansions); e must have room for n + m components
static __device__ int expansion_add(double *e, int n, const double *f, int m) {
  for (int j = 0; j < m; ++j) n = grow(e, n, f[j], e);
  return n;
}
// acc += s * (e[0..n) * b): the exact products go in one component at a time
static __device__ int add_scaled(double *acc, int na, const double *e, int n, double b, double s) {
  for (int i = 0; i < n; ++i) {
    double p, lo;
    two_prod(e[i], b, p, lo);
    if (lo != 0.0) na = grow(acc, na, s * lo, acc);
    if (p != 0.0) na = grow(acc, na, s * p, acc);
  }
  return na;
}
// acc += s * (e * f), e and f expansions
static __device__ int add_product(double *acc, int na, const double *e, int n, const double *f, int m, double s) {
  for (int j = 0; j < m; ++j) na = add_scaled(acc, na, e, n, f[j], s);
  return na;
}
static __device__ __forceinline__ int sign_of(const double *e, int n) {
  const double top = e[n - 1];
  return top > 0.0 ? 1 : (top < 0.0 ? -1 : 0);
}

// orient2d, exact: (ax - cx)(by - cy) - (ay - cy)(bx - cx) with every difference a two-component expansion
static __device__ int orient2d_exact(double2 a, double2 b, double2 c) {
  double A[2][2], Bv[2][2];
  int nA[2], nB[2];
  const double av[2] = {a.x, a.y}, bv[2] = {b.x, b.y}, cv[2] = {c.x, c.y};
  for (int k = 0; k < 2; ++k) {
    double s, lo;
    two_diff(av[k], cv[k], s, lo);
    nA[k] = 0;
    if (lo != 0.0) A[k][nA[k]++] = lo;
    if (s != 0.0 || nA[k] == 0) A[k][nA[k]++] = s;
    two_diff(bv[k], cv[k], s, lo);
    nB[k] = 0;
    if (lo != 0.0) Bv[k][nB[k]++] = lo;
    if (s != 0.0 || nB[k] == 0) Bv[k][nB[k]++] = s;
  }
  double acc[20];
  acc[0] = 0.0;
  int n = 1;
  n = add_product(acc, n, A[0], nA[0], Bv[1], nB[1], 1.0);    // + (ax - cx)(by - cy)
  n = add_product(acc, n, A[1], nA[1], Bv[0], nB[0], -1.0);   // - (ay - cy)(bx - cx)
  return sign_of(acc, n);
}

// incircle2d, exact (eq. 5): sum over the rows (a, b, c) of lift_row * minor_row with the rows translated by d
constexpr int MAXE = 1200;   // 3 x (12 x 16 x 2) = 1152 components at most
static __device__ int incircle2d_exact(double2 a, double2 b, double2 c, double2 d, double *acc, double *tmp) {
  const double px[3] = {a.x, b.x, c.x}, py[3] = {a.y, b.y, c.y};
  double X[3][2], Y[3][2];
  int nX[3], nY[3];
  for (int k = 0; k < 3; ++k) {
    double s, lo;
    two_diff(px[k], d.x, s, lo);
    nX[k] = 0;
    if (lo != 0.0) X[k][nX[k]++] = lo;
    if (s != 0.0 || nX[k] == 0) X[k][nX[k]++] = s;
    two_diff(py[k], d.y, s, lo);
    nY[k] = 0;
    if (lo != 0.0) Y[k][nY[k]++] = lo;
    if (s != 0.0 || nY[k] == 0) Y[k][nY[k]++] = s;
  }
  acc[0] = 0.0;
  int na = 1;
  for (int k = 0; k < 3; ++k) {
    const int i = (k + 1) % 3, j = (k + 2) % 3;   // cofactor of row k: + (x_i y_j - y_i x_j) for k = 0, 1, 2 (cyclic)
    double lift[16], minor[20];
    lift[0] = 0.0;
    int nl = 1;
    nl = add_product(lift, nl, X[k], nX[k], X[k], nX[k], 1.0);
    nl = add_product(lift, nl, Y[k], nY[k], Y[k], nY[k], 1.0);
    minor[0] = 0.0;
    int nm = 1;
    nm = add_product(minor, nm, X[i], nX[i], Y[j], nY[j], 1.0);
    nm = add_product(minor, nm, Y[i], nY[i], X[j], nX[j], -1.0);
    // acc += lift * minor, through tmp so that the inner sums stay short
    tmp[0] = 0.0;
    int nt = 1;
    nt = add_product(tmp, nt, lift, nl, minor, nm, 1.0);
    na = expansion_add(acc, na, tmp, nt);
  }
  return sign_of(acc, na);
}

// The same determinant when the six translations a - d, b - d, c - d are EXACT (no rounding: the usual case for neighbouring
// points, whose coordinates are within a factor 2 of each other): every factor is then a single double and the expansions stay
// short -- lift <= 4 components, minor <= 4, their product <= 32, the sum of the three <= 96 -- so they fit thread-local arrays
// and any thread can do it.  Returns the exact sign, or 2 when a translation is inexact (the caller falls back to
// incircle2d_exact with its 1152-component scratch).
static __device__ int incircle2d_exact_short(double2 a, double2 b, double2 c, double2 d) {
  const double px[3] = {a.x, b.x, c.x}, py[3] = {a.y, b.y, c.y};
  double X[3], Y[3];
  for (int k = 0; k < 3; ++k) {
    double lo;
    two_diff(px[k], d.x, X[k], lo);
    if (lo != 0.0) return 2;
    two_diff(py[k], d.y, Y[k], lo);
    if (lo != 0.0) return 2;
  }
  double acc[100], tmp[36];
  acc[0] = 0.0;
  int na = 1;
  for (int k = 0; k < 3; ++k) {
    const int i = (k + 1) % 3, j = (k + 2) % 3;
    double lift[8], minor[8];
    lift[0] = 0.0;
    int nl = 1;
    nl = add_product(lift, nl, &X[k], 1, &X[k], 1, 1.0);
    nl = add_product(lift, nl, &Y[k], 1, &Y[k], 1, 1.0);
    minor[0] = 0.0;
    int nm = 1;
    nm = add_product(minor, nm, &X[i], 1, &Y[j], 1, 1.0);
    nm = add_product(minor, nm, &Y[i], 1, &X[j], 1, -1.0);
    tmp[0] = 0.0;
    int nt = 1;
    nt = add_product(tmp, nt, lift, nl, minor, nm, 1.0);
    na = expansion_add(acc, na, tmp, nt);
  }
  return sign_of(acc, na);
}

constexpr double EPS = 1.1102230246251565e-16;   // 2^-53

// Filters: the determinant in plain fp64 and a bound on its rounding error.  Return +1 / -1 when the sign is certain, 2 when the
// exact evaluation has to decide.
// eq. 3: each product carries three roundings (two differences, one product), the difference one more: |error| <= 4 eps (|l| + |r|)
// to first order; 8 eps covers the higher orders with a wide margin
static __device__ __forceinline__ int orient2d_filter(double2 a, double2 b, double2 c) {
  const double l = __dmul_rn(__dsub_rn(a.x, c.x), __dsub_rn(b.y, c.y)), r = __dmul_rn(__dsub_rn(a.y, c.y), __dsub_rn(b.x, c.x));
  const double det = __dsub_rn(l, r);
  const double bound = 8.0 * EPS * (fabs(l) + fabs(r));
  return det > bound ? 1 : (det < -bound ? -1 : 2);
}
static __device__ __forceinline__ int orient2d_sign(double2 a, double2 b, double2 c) {
  const int s = orient2d_filter(a, b, c);
  return s != 2 ? s : orient2d_exact(a, b, c);
}
// eq. 5: every one of the six monomial groups lift * product goes through at most 9 roundings (a difference, a square or product,
// the sums, the final products and additions); |error| <= 10 eps * permanent to first order, 16 eps with margin
// (whatever contraction into FMAs the compiler applies only removes roundings)
static __device__ __forceinline__ int incircle2d_filter(double2 a, double2 b, double2 c, double2 d) {
  const double ax = a.x - d.x, ay = a.y - d.y, bx = b.x - d.x, by = b.y - d.y, cx = c.x - d.x, cy = c.y - d.y;
  const double al = ax * ax + ay * ay, bl = bx * bx + by * by, cl = cx * cx + cy * cy;
  const double bc1 = bx * cy, bc2 = by * cx, ca1 = cx * ay, ca2 = cy * ax, ab1 = ax * by, ab2 = ay * bx;
  const double det = al * (bc1 - bc2) + bl * (ca1 - ca2) + cl * (ab1 - ab2);
  const double perm = al * (fabs(bc1) + fabs(bc2)) + bl * (fabs(ca1) + fabs(ca2)) + cl * (fabs(ab1) + fabs(ab2));
  const double bound = 16.0 * EPS * perm;
  return det > bound ? 1 : (det < -bound ? -1 : 2);
}

}  // namespace mrdgen
