// mrd_meshgen.cu -- first slice of the mesh-generation layer (section 2.4 and 4.1): the two kernels every
// iteration of the parallel Delaunay refinement starts with, and the two geometric predicates everything else rests on.
//
//   test_quality   for every triangle the circumradius r of eq. 2 (L146), the circumradius-to-shortest-edge ratio beta
//                  (L118-L126), the flag "r > R or beta > B" (L150) and the circumcentre, where the new vertex goes (L150);
//   orient2d       the sign of the determinant of eq. 3 (L160), EXACT;
//   incircle2d     the sign of the determinant of eq. 5 (L198), EXACT.
//
// test_quality is written operation by operation with round-to-nearest intrinsics (no FMA contraction), so that it agrees
// bit for bit with the CPU oracle (oracle/meshgen.py), which evaluates the same formulas in the same order.
// The predicates must be exact (L162-L166, L665-L667: "mutually contradictory results inevitably lead to ... invalid
// triangulations").  The paper uses adaptive exact predicates; here: a floating-point FILTER with a rigorous error bound
// decides almost every test, and the rest go to a second kernel that evaluates the determinant exactly in floating-point
// expansion arithmetic (error-free transformations TwoSum / TwoProduct with FMA; sums of non-overlapping components with
// zero elimination).  The sign of an expansion is the sign of its largest component.
#include <cuda_runtime.h>

#include <cstdint>
#include <string>

#include "../../include/mrd.h"

namespace mrdgen {

// ------------------------------------------------------------------------------------------------------------------
// TestQuality (eq. 2): one thread per triangle
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
test_quality_kernel(int64_t nt, const double2 *__restrict__ xy, const int32_t *__restrict__ tri, double R, double B,
                    double *__restrict__ r_out, double *__restrict__ beta_out, double2 *__restrict__ cc_out,
                    uint8_t *__restrict__ bad_out, unsigned long long *__restrict__ n_bad) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int bad = 0;
  if (t < nt) {
    const double2 a = xy[tri[3 * t]], b = xy[tri[3 * t + 1]], c = xy[tri[3 * t + 2]];
    // eq. 3 / eq. 2: det = (ax - cx)(by - cy) - (ay - cy)(bx - cx)
    const double Ax = __dsub_rn(a.x, c.x), Ay = __dsub_rn(a.y, c.y), Bx = __dsub_rn(b.x, c.x), By = __dsub_rn(b.y, c.y);
    const double det = __dsub_rn(__dmul_rn(Ax, By), __dmul_rn(Ay, Bx));
    // edge lengths opposite a, b, c
    const double Cx = __dsub_rn(a.x, b.x), Cy = __dsub_rn(a.y, b.y);
    const double la2 = __dadd_rn(__dmul_rn(Bx, Bx), __dmul_rn(By, By));   // |b - c|^2
    const double lb2 = __dadd_rn(__dmul_rn(Ax, Ax), __dmul_rn(Ay, Ay));   // |a - c|^2
    const double lc2 = __dadd_rn(__dmul_rn(Cx, Cx), __dmul_rn(Cy, Cy));   // |a - b|^2
    const double la = __dsqrt_rn(la2), lb = __dsqrt_rn(lb2), lc = __dsqrt_rn(lc2);
    const double r = __ddiv_rn(__dmul_rn(__dmul_rn(la, lb), lc), __dmul_rn(2.0, det));   // eq. 2
    const double lmin = fmin(la, fmin(lb, lc));
    const double beta = __ddiv_rn(r, lmin);                                              // L120
    // circumcentre: c + (|A|^2 (By, -Bx) - |B|^2 (Ay, -Ax)) / (2 det), A = a - c, B = b - c
    const double d2 = __dmul_rn(2.0, det);
    const double ux = __ddiv_rn(__dsub_rn(__dmul_rn(lb2, By), __dmul_rn(la2, Ay)), d2);
    const double uy = __ddiv_rn(__dsub_rn(__dmul_rn(la2, Ax), __dmul_rn(lb2, Bx)), d2);
    r_out[t] = r;
    beta_out[t] = beta;
    cc_out[t] = make_double2(__dadd_rn(c.x, ux), __dadd_rn(c.y, uy));
    bad = (r > R || beta > B) ? 1 : 0;   // L150 (a triangle with det <= 0 has r <= 0 or inf: flagged by beta or not at all; the
    if (!(det > 0.0)) bad = 1;           //       mesh is counter-clockwise, so det <= 0 is itself a defect: flag it)
    bad_out[t] = (uint8_t)bad;
  }
  // count: warp ballot -> one atomic per warp
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_bad, (unsigned long long)__popc(m));
}

// ------------------------------------------------------------------------------------------------------------------
// Expansion arithmetic (device).  An expansion is a sum of doubles e[0..n) that do not overlap, in increasing magnitude, zeros
// removed.  All operations below are exact.
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void two_sum(double a, double b, double &s, double &e) {
  s = __dadd_rn(a, b);
  const double bb = __dsub_rn(s, a);
  e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void two_diff(double a, double b, double &s, double &e) { two_sum(a, -b, s, e); }
__device__ __forceinline__ void two_prod(double a, double b, double &p, double &e) {
  p = __dmul_rn(a, b);
  e = __fma_rn(a, b, -p);
}
// h = e + b (e: expansion of length n, b: any double); returns the new length.  h may alias e.
__device__ int grow(const double *e, int n, double b, double *h) {
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
__device__ int expansion_add(double *e, int n, const double *f, int m) {
  for (int j = 0; j < m; ++j) n = grow(e, n, f[j], e);
  return n;
}
// acc += s * (e[0..n) * b): the exact products go in one component at a time
__device__ int add_scaled(double *acc, int na, const double *e, int n, double b, double s) {
  for (int i = 0; i < n; ++i) {
    double p, lo;
    two_prod(e[i], b, p, lo);
    if (lo != 0.0) na = grow(acc, na, s * lo, acc);
    if (p != 0.0) na = grow(acc, na, s * p, acc);
  }
  return na;
}
// acc += s * (e * f), e and f expansions
__device__ int add_product(double *acc, int na, const double *e, int n, const double *f, int m, double s) {
  for (int j = 0; j < m; ++j) na = add_scaled(acc, na, e, n, f[j], s);
  return na;
}
__device__ __forceinline__ int sign_of(const double *e, int n) {
  const double top = e[n - 1];
  return top > 0.0 ? 1 : (top < 0.0 ? -1 : 0);
}

// orient2d, exact: (ax - cx)(by - cy) - (ay - cy)(bx - cx) with every difference a two-component expansion
__device__ int orient2d_exact(double2 a, double2 b, double2 c) {
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
__device__ int incircle2d_exact(double2 a, double2 b, double2 c, double2 d, double *acc, double *tmp) {
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

// ------------------------------------------------------------------------------------------------------------------
// Filter kernels: the determinant in plain fp64 and a bound on its rounding error; undecided tests go to a work list
// ------------------------------------------------------------------------------------------------------------------
constexpr double EPS = 1.1102230246251565e-16;   // 2^-53

__global__ void __launch_bounds__(256)
orient_filter_kernel(int64_t n, const double2 *__restrict__ xy, const int32_t *__restrict__ idx, int8_t *__restrict__ sign,
                     int32_t *__restrict__ work, unsigned long long *__restrict__ n_work) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const double2 a = xy[idx[3 * k]], b = xy[idx[3 * k + 1]], c = xy[idx[3 * k + 2]];
  const double l = __dmul_rn(__dsub_rn(a.x, c.x), __dsub_rn(b.y, c.y)), r = __dmul_rn(__dsub_rn(a.y, c.y), __dsub_rn(b.x, c.x));
  const double det = __dsub_rn(l, r);
  // each product carries three roundings (two differences, one product), the difference one more: |error| <= 4 eps (|l| + |r|)
  // to first order; 8 eps covers the higher orders with a wide margin
  const double bound = 8.0 * EPS * (fabs(l) + fabs(r));
  if (det > bound) sign[k] = 1;
  else if (det < -bound) sign[k] = -1;
  else {
    sign[k] = 2;
    work[atomicAdd(n_work, 1ull)] = (int32_t)k;
  }
}
__global__ void orient_exact_kernel(const unsigned long long *__restrict__ n_work, const int32_t *__restrict__ work,
                                    const double2 *__restrict__ xy, const int32_t *__restrict__ idx, int8_t *__restrict__ sign) {
  const int64_t nw = (int64_t)*n_work;
  for (int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; q < nw; q += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = work[q];
    sign[k] = (int8_t)orient2d_exact(xy[idx[3 * k]], xy[idx[3 * k + 1]], xy[idx[3 * k + 2]]);
  }
}

__global__ void __launch_bounds__(256)
incircle_filter_kernel(int64_t n, const double2 *__restrict__ xy, const int32_t *__restrict__ idx, int8_t *__restrict__ sign,
                       int32_t *__restrict__ work, unsigned long long *__restrict__ n_work) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const double2 a = xy[idx[4 * k]], b = xy[idx[4 * k + 1]], c = xy[idx[4 * k + 2]], d = xy[idx[4 * k + 3]];
  const double ax = a.x - d.x, ay = a.y - d.y, bx = b.x - d.x, by = b.y - d.y, cx = c.x - d.x, cy = c.y - d.y;
  const double al = ax * ax + ay * ay, bl = bx * bx + by * by, cl = cx * cx + cy * cy;
  const double bc1 = bx * cy, bc2 = by * cx, ca1 = cx * ay, ca2 = cy * ax, ab1 = ax * by, ab2 = ay * bx;
  const double det = al * (bc1 - bc2) + bl * (ca1 - ca2) + cl * (ab1 - ab2);
  // every one of the six monomial groups lift * product goes through at most 9 roundings (a difference, a square or product,
  // the sums, the final products and additions); |error| <= 10 eps * permanent to first order, 16 eps with margin
  // (whatever contraction into FMAs the compiler applies only removes roundings)
  const double perm = al * (fabs(bc1) + fabs(bc2)) + bl * (fabs(ca1) + fabs(ca2)) + cl * (fabs(ab1) + fabs(ab2));
  const double bound = 16.0 * EPS * perm;
  if (det > bound) sign[k] = 1;
  else if (det < -bound) sign[k] = -1;
  else {
    sign[k] = 2;
    work[atomicAdd(n_work, 1ull)] = (int32_t)k;
  }
}
__global__ void __launch_bounds__(32)
incircle_exact_kernel(const unsigned long long *__restrict__ n_work, const int32_t *__restrict__ work, const double2 *__restrict__ xy,
                      const int32_t *__restrict__ idx, int8_t *__restrict__ sign, double *__restrict__ scratch) {
  const int64_t nw = (int64_t)*n_work;
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double *acc = scratch + tid * (2 * MAXE), *tmp = acc + MAXE;   // per-thread scratch in global memory (the expansions are long)
  for (int64_t q = tid; q < nw; q += (int64_t)gridDim.x * blockDim.x) {
    const int64_t k = work[q];
    sign[k] = (int8_t)incircle2d_exact(xy[idx[4 * k]], xy[idx[4 * k + 1]], xy[idx[4 * k + 2]], xy[idx[4 * k + 3]], acc, tmp);
  }
}

}  // namespace mrdgen

extern "C" {

// (mrd_last_error lives in mrd_api.cu; this file reports through its hook)
int mrd_internal_set_error(int code, const char *msg);

namespace {
int gen_fail(int code, const std::string &msg) { return mrd_internal_set_error(code, msg.c_str()); }
#define GEN_TRY(expr)                                                                                   \
  do {                                                                                                  \
    cudaError_t e_ = (expr);                                                                            \
    if (e_ != cudaSuccess) return gen_fail(e_ == cudaErrorMemoryAllocation ? MRD_ENOMEM : MRD_ECUDA,    \
                                           std::string(#expr) + ": " + cudaGetErrorString(e_));         \
  } while (0)
}  // namespace

int mrd_meshgen_test_quality(int64_t n_triangle, const double *xy_dev, const int32_t *tri_dev, double R, double B, double *r_dev,
                             double *beta_dev, double *cc_dev, uint8_t *bad_dev, int64_t *n_bad, void *stream) {
  if (n_triangle < 0 || (n_triangle > 0 && (!xy_dev || !tri_dev || !r_dev || !beta_dev || !cc_dev || !bad_dev)))
    return gen_fail(MRD_EINVAL, "null argument");
  if (!(R > 0.0) || !(B > 0.0)) return gen_fail(MRD_EINVAL, "R and B must be positive");
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long *cnt = nullptr;
  GEN_TRY(cudaMalloc(&cnt, sizeof *cnt));
  GEN_TRY(cudaMemsetAsync(cnt, 0, sizeof *cnt, s));
  if (n_triangle > 0)
    mrdgen::test_quality_kernel<<<(unsigned)((n_triangle + 255) / 256), 256, 0, s>>>(n_triangle, (const double2 *)xy_dev, tri_dev, R, B, r_dev, beta_dev,
                                                                                     (double2 *)cc_dev, bad_dev, cnt);
  unsigned long long h = 0;
  cudaError_t e = cudaMemcpyAsync(&h, cnt, sizeof h, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(cnt);
  if (e != cudaSuccess) return gen_fail(MRD_ECUDA, std::string("test_quality: ") + cudaGetErrorString(e));
  if (n_bad) *n_bad = (int64_t)h;
  return MRD_OK;
}

static int predicate_impl(int which, int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  if (n < 0 || (n > 0 && (!xy_dev || !idx_dev || !sign_dev))) return gen_fail(MRD_EINVAL, "null argument");
  if (n > 0x7FFFFFF0ll) return gen_fail(MRD_EINVAL, "too many tests for 32-bit work lists");
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long *cnt = nullptr;
  int32_t *work = nullptr;
  double *scratch = nullptr;
  GEN_TRY(cudaMalloc(&cnt, sizeof *cnt));
  cudaError_t e = cudaMalloc(&work, sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
  const int exact_blocks = 148 * 4, exact_threads = 32;
  if (e == cudaSuccess && which == 1) e = cudaMalloc(&scratch, sizeof(double) * 2 * mrdgen::MAXE * (size_t)exact_blocks * exact_threads);
  if (e == cudaSuccess) e = cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  if (e == cudaSuccess && n > 0) {
    const unsigned nb = (unsigned)((n + 255) / 256);
    if (which == 0) {
      mrdgen::orient_filter_kernel<<<nb, 256, 0, s>>>(n, (const double2 *)xy_dev, idx_dev, sign_dev, work, cnt);
      mrdgen::orient_exact_kernel<<<exact_blocks, 128, 0, s>>>(cnt, work, (const double2 *)xy_dev, idx_dev, sign_dev);
    } else {
      mrdgen::incircle_filter_kernel<<<nb, 256, 0, s>>>(n, (const double2 *)xy_dev, idx_dev, sign_dev, work, cnt);
      mrdgen::incircle_exact_kernel<<<exact_blocks, exact_threads, 0, s>>>(cnt, work, (const double2 *)xy_dev, idx_dev, sign_dev, scratch);
    }
  }
  unsigned long long h = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, cnt, sizeof h, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  cudaFree(cnt);
  cudaFree(work);
  if (scratch) cudaFree(scratch);
  if (e != cudaSuccess) return gen_fail(e == cudaErrorMemoryAllocation ? MRD_ENOMEM : MRD_ECUDA, std::string("predicate: ") + cudaGetErrorString(e));
  if (n_exact) *n_exact = (int64_t)h;
  return MRD_OK;
}

int mrd_meshgen_orient2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  return predicate_impl(0, n, xy_dev, idx_dev, sign_dev, n_exact, stream);
}
int mrd_meshgen_incircle2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  return predicate_impl(1, n, xy_dev, idx_dev, sign_dev, n_exact, stream);
}

}  // extern "C"
