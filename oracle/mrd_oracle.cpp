// mrd_oracle.cpp -- CPU ORACLE for the residual-distribution sweep of arXiv:1705.02028.
//
// TEST INFRASTRUCTURE, NOT THE PRODUCT.  Plain, slow, fp64, written from PAPER.md only, following
// the algorithm step by step in the paper's order and notation (the
// readings C1-C22 of passages where the paper is silent or garbled are listed in DESIGN.md).
// It shares no code with paper_1705_02028_b200/ (the CUDA path) and must not be used by it.
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): flux-Jacobian finite differences, K R = R Lambda,
// R R^-1 = I, A10-A25 == R diag(l) R^-1, Simpson contour integral of the flux, sum(beta_i) = I,
// sum(phi_i^N) = phi^T, symmetrising-variable block form, stagnation limit, uniform flow == 0 exactly,
// conservation, permutation invariance, Heun reduction, Sod vs exact Riemann solution, vortex order ~ 2.
// Wall boundary term (eq. 68-71): pinned by v_n = 0 -> 0, by the mass balance, by the oblique-wall
// uniform-flow test, and its stage-2 averaging (reading C15) by the Heun reduction of RK2 with scheme N on
// a mesh with walls and oblique flow (tests/test_oracle_step.py).  No function here is "parity unpinned".
#include "mrd_oracle.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <unordered_map>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

thread_local std::string g_err;
int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}

// ------------------------------------------------------------------------------------------
// Scalar helpers: the per-triangle routines are templates over the scalar so that the same
// text can be run with a counting type (orc_count_ops); `double` is what every result uses.
// ------------------------------------------------------------------------------------------
struct OpCounts {
  int64_t add = 0, mul = 0, div = 0, sqrt = 0, abs = 0, cmp = 0;
};
thread_local OpCounts g_ops;

struct Cnt {
  double v;
  Cnt() : v(0.0) {}
  Cnt(double x) : v(x) {}
};
inline Cnt operator+(Cnt a, Cnt b) { g_ops.add++; return Cnt(a.v + b.v); }
inline Cnt operator-(Cnt a, Cnt b) { g_ops.add++; return Cnt(a.v - b.v); }
inline Cnt operator-(Cnt a) { return Cnt(-a.v); }
inline Cnt operator*(Cnt a, Cnt b) { g_ops.mul++; return Cnt(a.v * b.v); }
inline Cnt operator/(Cnt a, Cnt b) { g_ops.div++; return Cnt(a.v / b.v); }
inline Cnt &operator+=(Cnt &a, Cnt b) { a = a + b; return a; }
inline Cnt &operator-=(Cnt &a, Cnt b) { a = a - b; return a; }
inline bool operator<(Cnt a, Cnt b) { g_ops.cmp++; return a.v < b.v; }
inline bool operator>(Cnt a, Cnt b) { g_ops.cmp++; return a.v > b.v; }
inline bool operator<=(Cnt a, Cnt b) { g_ops.cmp++; return a.v <= b.v; }
inline bool operator==(Cnt a, Cnt b) { g_ops.cmp++; return a.v == b.v; }

inline double Sqrt(double x) { return std::sqrt(x); }
inline double Abs(double x) { return std::fabs(x); }
inline double Max(double a, double b) { return a > b ? a : b; }
inline double Min(double a, double b) { return a < b ? a : b; }
inline Cnt Sqrt(Cnt x) { g_ops.sqrt++; return Cnt(std::sqrt(x.v)); }
inline Cnt Abs(Cnt x) { g_ops.abs++; return Cnt(std::fabs(x.v)); }
inline Cnt Max(Cnt a, Cnt b) { g_ops.cmp++; return a.v > b.v ? a : b; }
inline Cnt Min(Cnt a, Cnt b) { g_ops.cmp++; return a.v < b.v ? a : b; }

// row-major 4x4 helpers
template <class R> inline void matvec4(const R *M, const R *x, R *y) {
  for (int r = 0; r < 4; ++r) {
    R s = M[4 * r + 0] * x[0];
    for (int c = 1; c < 4; ++c) s = s + M[4 * r + c] * x[c];
    y[r] = s;
  }
}

// Gauss-Jordan inversion with partial pivoting of the n x n matrix stored with row stride `ld`
// (O5).  Returns false when a pivot is exactly zero.
template <class R> bool gauss_jordan(const R *A, int n, int ld, R *Ainv, int ldinv) {
  R a[4][8];
  for (int r = 0; r < n; ++r)
    for (int c = 0; c < n; ++c) {
      a[r][c] = A[r * ld + c];
      a[r][n + c] = R(r == c ? 1.0 : 0.0);
    }
  for (int k = 0; k < n; ++k) {
    int piv = k;
    R best = Abs(a[k][k]);
    for (int r = k + 1; r < n; ++r) {
      R cand = Abs(a[r][k]);
      if (cand > best) { best = cand; piv = r; }
    }
    if (best == R(0.0)) return false;
    if (piv != k)
      for (int c = 0; c < 2 * n; ++c) std::swap(a[k][c], a[piv][c]);
    R inv = R(1.0) / a[k][k];
    for (int c = 0; c < 2 * n; ++c) a[k][c] = a[k][c] * inv;
    for (int r = 0; r < n; ++r) {
      if (r == k) continue;
      R f = a[r][k];
      for (int c = 0; c < 2 * n; ++c) a[r][c] = a[r][c] - f * a[k][c];
    }
  }
  for (int r = 0; r < n; ++r)
    for (int c = 0; c < n; ++c) Ainv[r * ldinv + c] = a[r][n + c];
  return true;
}

// ------------------------------------------------------------------------------------------
// O1. Geometry of one triangle with counter-clockwise vertices x[0..2] (already unwrapped).
// n_i = inward normal of the edge opposite node i, scaled with the edge length (eq. 35):
// the edge runs from vertex i+1 to vertex i+2, e = x_{i+2} - x_{i+1}, n_i = (-e_y, e_x).
// ------------------------------------------------------------------------------------------
template <class R> struct Geom {
  R nx[3], ny[3];  // UNIT inward normals (reading C4)
  R len[3];        // edge lengths l_i = |n_i|
  R area;          // |T|
  R lmax;          // longest edge (eq. 44)
};

template <class R> void triangle_geometry(const R x[3][2], Geom<R> &g) {
  for (int i = 0; i < 3; ++i) {
    int a = (i + 1) % 3, b = (i + 2) % 3;
    R ex = x[b][0] - x[a][0], ey = x[b][1] - x[a][1];
    R l = Sqrt(ex * ex + ey * ey);
    g.len[i] = l;
    g.nx[i] = -ey / l;
    g.ny[i] = ex / l;
  }
  R ax = x[1][0] - x[0][0], ay = x[1][1] - x[0][1];
  R bx = x[2][0] - x[0][0], by = x[2][1] - x[0][1];
  g.area = R(0.5) * (ax * by - ay * bx);
  g.lmax = Max(g.len[0], Max(g.len[1], g.len[2]));
}

// ------------------------------------------------------------------------------------------
// S1/O2. Parameter vector Z = sqrt(rho) (1, u, v, h)  (eq. 20 L290-L294 in 1D; its 2D analogue,
// L419, reading C1), with p from eq. 10 (L224) and h = (e + p)/rho (L227).
// ------------------------------------------------------------------------------------------
template <class R> bool parameter_vector(R gamma, const R W[4], R Z[4], R *speed /* |v| + c, eq. 45 */) {
  R rho = W[0];
  if (!(rho > R(0.0))) return false;
  R u = W[1] / rho, v = W[2] / rho;
  R p = (gamma - R(1.0)) * (W[3] - R(0.5) * (W[1] * W[1] + W[2] * W[2]) / rho);
  if (!(p > R(0.0))) return false;
  R h = (W[3] + p) / rho;
  R s = Sqrt(rho);
  Z[0] = s;
  Z[1] = s * u;
  Z[2] = s * v;
  Z[3] = s * h;
  if (speed) *speed = Sqrt(u * u + v * v) + Sqrt(gamma * p / rho);  // eq. 45 with c^2 = gamma p / rho (C14)
  return true;
}

// ------------------------------------------------------------------------------------------
// App. A eq. A2 (L1272-L1278): K = A nx + B ny for conserved variables, times `half_len` = l_i/2
// (eq. 37 with d = 2 and the unit normal, reading C4).
// ------------------------------------------------------------------------------------------
template <class R> void euler_K(R gamma, R u, R v, R h, R nx, R ny, R half_len, R K[16]) {
  R g1 = gamma - R(1.0), g2 = gamma - R(2.0);
  R w = u * nx + v * ny;
  R alpha = g1 * (u * u + v * v) / R(2.0);
  K[0] = R(0.0);               K[1] = nx;                   K[2] = ny;                   K[3] = R(0.0);
  K[4] = alpha * nx - u * w;   K[5] = w - g2 * u * nx;      K[6] = u * ny - g1 * v * nx; K[7] = g1 * nx;
  K[8] = alpha * ny - v * w;   K[9] = v * nx - g1 * u * ny; K[10] = w - g2 * v * ny;     K[11] = g1 * ny;
  K[12] = (alpha - h) * w;     K[13] = h * nx - g1 * u * w; K[14] = h * ny - g1 * v * w; K[15] = gamma * w;
  for (int k = 0; k < 16; ++k) K[k] = K[k] * half_len;
}

// ------------------------------------------------------------------------------------------
// App. A eq. A10-A25 (L1309-L1350): K^(+/-) = R diag(l1,l2,l3,l3) R^-1 in closed form, given
// l_k (already including the factor l_i/2).  Readings C7: h_c = h/c; plain u, v in A23-A24;
// |n| = 1; each K_{r,c} taken once (the extraction duplicates A10, A11, A16).
// ------------------------------------------------------------------------------------------
template <class R>
void euler_K_split(R gamma, R u, R v, R h, R c, R nx, R ny, R l1, R l2, R l3, R K[16]) {
  R g1 = gamma - R(1.0), g2 = gamma - R(2.0);
  R w = u * nx + v * ny;
  R alpha = g1 * (u * u + v * v) / R(2.0);
  R ac = alpha / c, uc = u / c, vc = v / c, hc = h / c;
  R l123 = (l1 + l2 - R(2.0) * l3) / R(2.0);
  R l12 = (l1 - l2) / R(2.0);
  K[0] = ac / c * l123 - w / c * l12 + l3;                                        // A10
  K[1] = -g1 * uc / c * l123 + nx / c * l12;                                      // A11
  K[2] = -g1 * vc / c * l123 + ny / c * l12;                                      // A12
  K[3] = g1 / (c * c) * l123;                                                     // A13
  K[4] = (ac * uc - w * nx) * l123 + (ac * nx - uc * w) * l12;                    // A14
  K[5] = (nx * nx - g1 * uc * uc) * l123 - g2 * uc * nx * l12 + l3;               // A15
  K[6] = (nx * ny - g1 * uc * vc) * l123 + (uc * ny - g1 * vc * nx) * l12;        // A16
  K[7] = g1 * uc / c * l123 + g1 * nx / c * l12;                                  // (A17)
  K[8] = (ac * vc - w * ny) * l123 + (ac * ny - vc * w) * l12;                    // A18
  K[9] = (nx * ny - g1 * uc * vc) * l123 + (vc * nx - g1 * uc * ny) * l12;        // A19
  K[10] = (ny * ny - g1 * vc * vc) * l123 - g2 * vc * ny * l12 + l3;              // A20
  K[11] = g1 * vc / c * l123 + g1 * ny / c * l12;                                 // A21
  K[12] = (ac * hc - w * w) * l123 + w * (ac - hc) * l12;                         // A22
  K[13] = (w * nx - u - ac * uc) * l123 + (hc * nx - g1 * uc * w) * l12;          // A23
  K[14] = (w * ny - v - ac * vc) * l123 + (hc * ny - g1 * vc * w) * l12;          // A24
  K[15] = g1 * hc / c * l123 + g1 * w / c * l12 + l3;                             // A25
}

// ------------------------------------------------------------------------------------------
// Everything one triangle needs at one state (O2-O6): linearised state, K_i, K_i^+, K_i^-,
// N-hat, the differences delta_j, phi^T and phi_i^N.
// ------------------------------------------------------------------------------------------
template <class R> struct Core {
  R u, v, h, c;          // linearised state (eq. 39)
  R K[3][16], Kp[3][16], Km[3][16];
  R sumKm[16], Nhat[16];
  R delta[3][4];         // D(Zbar) (Z_j - Z_1)   (O3)
  R phiT[4];             // eq. 36
  R phiN[3][4];          // eq. 48
  R speed[3];            // |v_j| + c_j at the vertices (eq. 45)
};

const double STAGNATION_EPS = 1e-14;  // reading C8

template <class R> int triangle_core(R gamma, const R W[3][4], const Geom<R> &g, Core<R> &o) {
  // O2: Z_j, Zbar (eq. 39), linearised u, v, h, c
  R Z[3][4];
  for (int j = 0; j < 3; ++j)
    if (!parameter_vector(gamma, W[j], Z[j], &o.speed[j])) return ORC_ENONPHYSICAL;
  R Zb[4];
  for (int k = 0; k < 4; ++k) Zb[k] = (Z[0][k] + Z[1][k] + Z[2][k]) / R(3.0);
  o.u = Zb[1] / Zb[0];
  o.v = Zb[2] / Zb[0];
  o.h = Zb[3] / Zb[0];
  R g1 = gamma - R(1.0);
  R c2 = g1 * (o.h - R(0.5) * (o.u * o.u + o.v * o.v));
  if (!(c2 > R(0.0))) return ORC_ENONPHYSICAL;
  o.c = Sqrt(c2);

  // O3: delta_j = D(Zbar) (Z_j - Z_1), D = dW/dZ at Zbar (reading C3)
  for (int j = 0; j < 3; ++j) {
    R d[4];
    for (int k = 0; k < 4; ++k) d[k] = Z[j][k] - Z[0][k];
    o.delta[j][0] = R(2.0) * Zb[0] * d[0];
    o.delta[j][1] = Zb[1] * d[0] + Zb[0] * d[1];
    o.delta[j][2] = Zb[2] * d[0] + Zb[0] * d[2];
    o.delta[j][3] = (Zb[3] * d[0] + g1 * Zb[1] * d[1] + g1 * Zb[2] * d[2] + Zb[0] * d[3]) / gamma;
  }

  // O4: K_i (A2), K_i^+ and K_i^- (A10-A25 with l_k = (l_i/2) lambda_k^(+/-), eq. 41-42), reading C22:
  // both signs evaluated directly, never as K - K^+.
  for (int k = 0; k < 16; ++k) o.sumKm[k] = R(0.0);
  for (int i = 0; i < 3; ++i) {
    R nx = g.nx[i], ny = g.ny[i], hl = g.len[i] / R(2.0);
    R w = o.u * nx + o.v * ny;
    R lam[3] = {w + o.c, w - o.c, w};
    R lp[3], lm[3];
    for (int k = 0; k < 3; ++k) {
      lp[k] = hl * (R(0.5) * (lam[k] + Abs(lam[k])));  // eq. 42
      lm[k] = hl * (R(0.5) * (lam[k] - Abs(lam[k])));
    }
    euler_K(gamma, o.u, o.v, o.h, nx, ny, hl, o.K[i]);
    euler_K_split(gamma, o.u, o.v, o.h, o.c, nx, ny, lp[0], lp[1], lp[2], o.Kp[i]);
    euler_K_split(gamma, o.u, o.v, o.h, o.c, nx, ny, lm[0], lm[1], lm[2], o.Km[i]);
    for (int k = 0; k < 16; ++k) o.sumKm[k] = o.sumKm[k] + o.Km[i][k];
  }

  // O5: N-hat = (sum_j K_j^-)^-1 (eq. 49) with the stagnation rule C8
  for (int k = 0; k < 16; ++k) o.Nhat[k] = R(0.0);
  R q2 = o.u * o.u + o.v * o.v;
  R lim = R(STAGNATION_EPS) * o.c;
  bool ok;
  if (q2 <= lim * lim) {
    ok = gauss_jordan(o.sumKm + 5, 3, 4, o.Nhat + 5, 4);  // rows/columns 2-4 (1-based)
  } else {
    ok = gauss_jordan(o.sumKm, 4, 4, o.Nhat, 4);
  }
  if (!ok) return ORC_ENONPHYSICAL;

  // O6: phi^T = sum_i K_i delta_i (eq. 36);  phi_i^N = K_i^+ (delta_i - Nhat sum_j K_j^- delta_j) (eq. 48)
  R tmp[4], win[4], acc[4];
  for (int k = 0; k < 4; ++k) { o.phiT[k] = R(0.0); acc[k] = R(0.0); }
  for (int i = 0; i < 3; ++i) {
    matvec4(o.K[i], o.delta[i], tmp);
    for (int k = 0; k < 4; ++k) o.phiT[k] = o.phiT[k] + tmp[k];
    matvec4(o.Km[i], o.delta[i], tmp);
    for (int k = 0; k < 4; ++k) acc[k] = acc[k] + tmp[k];
  }
  matvec4(o.Nhat, acc, win);
  for (int i = 0; i < 3; ++i) {
    R d[4];
    for (int k = 0; k < 4; ++k) d[k] = o.delta[i][k] - win[k];
    matvec4(o.Kp[i], d, o.phiN[i]);
  }
  return ORC_OK;
}

// beta_i x = -K_i^+ Nhat x  (eq. 51)
template <class R> void apply_beta(const Core<R> &o, const R x[4], R out[3][4]) {
  R y[4];
  matvec4(o.Nhat, x, y);
  for (int i = 0; i < 3; ++i) {
    R t[4];
    matvec4(o.Kp[i], y, t);
    for (int k = 0; k < 4; ++k) out[i][k] = -t[k];
  }
}

// eq. 52-53 (+ reading C10): Theta_kk = min(1, |phi_k| / sum_j |phi^N_{j,k}|), 0 when the denominator is 0
// Bmax / Bmin (L503): "setting all diagonal values of Theta to theta, [where] theta can be taken to be either the
// maximum (Bmax) or the minimum (Bmin) over all Theta_kk".
// Bx (eq. 54): one scalar theta from the shock sensor (bx_theta below), passed in as theta_bx.
template <class R>
void blend(int scheme, const R phiT[4], const R phiN[3][4], const R phiLDA[3][4], R theta[4], R phiB[3][4],
           R theta_bx = R(0.0)) {
  for (int k = 0; k < 4; ++k) {
    R den = Abs(phiN[0][k]) + Abs(phiN[1][k]) + Abs(phiN[2][k]);
    R th = R(0.0);
    if (den > R(0.0)) th = Min(R(1.0), Abs(phiT[k]) / den);
    if (scheme == ORC_SCHEME_N) th = R(1.0);
    if (scheme == ORC_SCHEME_LDA) th = R(0.0);
    if (scheme == ORC_SCHEME_BX) th = theta_bx;
    theta[k] = th;
  }
  if (scheme == ORC_SCHEME_BMAX || scheme == ORC_SCHEME_BMIN) {
    R t = theta[0];
    for (int k = 1; k < 4; ++k) t = scheme == ORC_SCHEME_BMAX ? Max(t, theta[k]) : Min(t, theta[k]);
    for (int k = 0; k < 4; ++k) theta[k] = t;
  }
  for (int k = 0; k < 4; ++k)
    for (int i = 0; i < 3; ++i) phiB[i][k] = theta[k] * phiN[i][k] + (R(1.0) - theta[k]) * phiLDA[i][k];
}

// Bx shock sensor, eq. 55-56 (L509-L517), readings C23-C26 of DESIGN.md:
//   s = ( -L div v / (|v|_max - |v|_min) )^+ ,  theta = min(1, s^2 h)
// * div v: divergence of the LINEAR interpolant of the vertex velocities u_j = m_j / rho_j on the triangle,
//   sum_j (u_j . n_j) l_j / (2 |T|) with the inward normal n_j opposite vertex j (grad N_j = n_j l_j / (2|T|));
// * |v|_max, |v|_min: extremes of the vertex speeds over the WHOLE mesh at the state the stage is evaluated at
//   (only then is s = O(1) in smooth flow, as L517 says); equal extremes (e.g. fluid at rest): s = 0;
// * L: the domain size = the larger side of the domain's bounding box (the period where periodic);
// * h: "a measure of the size of the element" made dimensionless with L: l_max^T / L (l_max as in eq. 44);
//   theta is clamped to 1 (a blend coefficient).
template <class R> struct BxCtx {
  R L;       // domain size
  R vrange;  // |v|_max - |v|_min of the stage's state
};
template <class R> R bx_theta(const R W[3][4], const Geom<R> &g, const BxCtx<R> &bx) {
  R div = R(0.0);
  for (int j = 0; j < 3; ++j) {
    R u = W[j][1] / W[j][0], v = W[j][2] / W[j][0];
    div = div + (u * g.nx[j] + v * g.ny[j]) * g.len[j];
  }
  div = div / (R(2.0) * g.area);
  if (!(bx.vrange > R(0.0))) return R(0.0);
  R s = Max(R(0.0), -(bx.L * div) / bx.vrange);  // eq. 56
  return Min(R(1.0), s * s * (g.lmax / bx.L));   // eq. 55
}

template <class R> struct Stage1Out {
  R phiT[4], phiN[3][4], phiLDA[3][4], phiB[3][4], theta[4], sT;
};

template <class R>
int triangle_stage1(R gamma, int scheme, const R W[3][4], const Geom<R> &g, Core<R> &core, Stage1Out<R> &o,
                    const BxCtx<R> *bx = nullptr) {
  int rc = triangle_core(gamma, W, g, core);
  if (rc) return rc;
  for (int k = 0; k < 4; ++k) o.phiT[k] = core.phiT[k];
  for (int i = 0; i < 3; ++i)
    for (int k = 0; k < 4; ++k) o.phiN[i][k] = core.phiN[i][k];
  apply_beta(core, core.phiT, o.phiLDA);  // eq. 50
  blend(scheme, o.phiT, o.phiN, o.phiLDA, o.theta, o.phiB, (scheme == ORC_SCHEME_BX && bx) ? bx_theta(W, g, *bx) : R(0.0));
  // O7 / eq. 44-45: s_T = l_max * max_j (|v_j| + c_j)
  o.sT = g.lmax * Max(core.speed[0], Max(core.speed[1], core.speed[2]));
  return ORC_OK;
}

template <class R> struct Stage2Out {
  R PhiT[4], PhiN[3][4], PhiLDA[3][4], PhiB[3][4], theta[4];
};

// O9: total residuals of the second Runge-Kutta stage (eq. 57, 61-65; reading C12)
// `lumping` = 1: selective lumping (eq. 66-67): the anti-diffusive term
//   sum_j (|T| delta_ij / 3 - m^G_ij) dW_j/dt,  m^G_ij = |T|/12 (delta_ij + 1)  (Galerkin mass matrix)
// is added to BOTH Phi_i^N and Phi_i^LDA ("Phi_i can be either Phi_i^LDA or Phi_i^N", L567) before they are "mixed in
// the usual way" (L572); it sums to zero over the nodes, so Phi^T and conservation are unchanged.
template <class R>
int triangle_stage2(R gamma, int scheme, const R Wn[3][4], const R Ws[3][4], const Geom<R> &g, R dt,
                    const R phiT_n[4], const R phiN_n[3][4], Core<R> &core, Stage2Out<R> &o, int lumping = 0,
                    const BxCtx<R> *bx = nullptr) {
  int rc = triangle_core(gamma, Ws, g, core);  // all matrices re-evaluated at W*
  if (rc) return rc;
  R third = g.area / R(3.0);
  R dW[3][4];
  for (int j = 0; j < 3; ++j)
    for (int k = 0; k < 4; ++k) dW[j][k] = (Ws[j][k] - Wn[j][k]) / dt;
  for (int k = 0; k < 4; ++k) {
    // eq. 57 with eq. 60-61 time averaging: Phi^T = |T|/3 sum_j dW_j/dt + (phi^T(W^n) + phi^T(W*))/2
    o.PhiT[k] = third * (dW[0][k] + dW[1][k] + dW[2][k]) + R(0.5) * (phiT_n[k] + core.phiT[k]);
    for (int i = 0; i < 3; ++i)  // eq. 62
      o.PhiN[i][k] = third * dW[i][k] + R(0.5) * (core.phiN[i][k] + phiN_n[i][k]);
  }
  apply_beta(core, o.PhiT, o.PhiLDA);  // eq. 63 with eq. 65: Phi_i^LDA = beta_i(W*) Phi^T
  if (lumping == 1) {
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 4; ++k) {
        R extra = R(0.0);
        for (int j = 0; j < 3; ++j) {
          R lumped = (i == j) ? g.area / R(3.0) : R(0.0);                       // |T| delta_ij / 3
          R galerkin = g.area / R(12.0) * ((i == j) ? R(2.0) : R(1.0));         // eq. 67
          extra = extra + (lumped - galerkin) * dW[j][k];                       // eq. 66
        }
        o.PhiN[i][k] = o.PhiN[i][k] + extra;
        o.PhiLDA[i][k] = o.PhiLDA[i][k] + extra;
      }
  }
  // Bx in stage 2: the sensor of the state the matrices are evaluated at, W* (as C12)
  blend(scheme, o.PhiT, o.PhiN, o.PhiLDA, o.theta, o.PhiB, (scheme == ORC_SCHEME_BX && bx) ? bx_theta(Ws, g, *bx) : R(0.0));
  return ORC_OK;
}

// eq. 68-71 (L586-L602): weak reflecting wall, edge a-b, OUTWARD unit normal n (reading C15), alpha = 0.75
template <class R>
bool wall_edge(R gamma, const R Wa[4], const R Wb[4], R nx, R ny, R len, R Pa[4], R Pb[4]) {
  const R alpha = R(0.75);
  R Fa[4], Fb[4];
  const R *Ws[2] = {Wa, Wb};
  R *Fs[2] = {Fa, Fb};
  for (int s = 0; s < 2; ++s) {
    const R *W = Ws[s];
    R rho = W[0];
    if (!(rho > R(0.0))) return false;
    R u = W[1] / rho, v = W[2] / rho;
    R p = (gamma - R(1.0)) * (W[3] - R(0.5) * (W[1] * W[1] + W[2] * W[2]) / rho);
    R h = (W[3] + p) / rho;
    R vn = u * nx + v * ny;
    Fs[s][0] = -(rho * vn);  // eq. 68
    Fs[s][1] = -(rho * u * vn);
    Fs[s][2] = -(rho * v * vn);
    Fs[s][3] = -(rho * h * vn);
  }
  for (int k = 0; k < 4; ++k) {
    Pa[k] = len / R(2.0) * (alpha * Fa[k] + (R(1.0) - alpha) * Fb[k]);  // eq. 70
    Pb[k] = len / R(2.0) * ((R(1.0) - alpha) * Fa[k] + alpha * Fb[k]);  // eq. 71
  }
  return true;
}

}  // namespace

// ============================================================================================
// The mesh object and the time stepper (O1, O7-O10)
// ============================================================================================
struct orc_mesh {
  double gamma, cfl;
  int scheme, time_order;
  int lumping = 0;  // 0 = global lumping (all tests of the paper, L576); 1 = selective lumping (eq. 66-67)
  double period[2];
  int64_t nv, nt, ne;
  std::vector<double> xy;            // [nv][2]
  std::vector<int32_t> tri;          // [nt][3], CCW
  std::vector<uint8_t> flag;         // [nv]
  std::vector<int32_t> wedge;        // [ne][2]
  std::vector<double> wnx, wny, wlen;  // wall-edge outward unit normal and length
  std::vector<Geom<double>> geo;     // [nt]
  std::vector<double> vol;           // [nv]  V_i = sum |T|/3 (reading C5)
  std::vector<double> W, Wic, Ws;    // [4][nv]
  std::vector<double> phi, phiN_n, phiT_n, sT;  // per-triangle scratch: [nt][3][4], [nt][3][4], [nt][4], [nt]
  std::vector<double> acc;           // [nv][4]
  std::vector<double> wallN;         // [ne][2][4] stage-1 wall terms
  double Ldom = 1.0;                 // domain size L of eq. 56 (Bx)
  int nthreads = 1;
  double t = 0.0;
  bool has_state = false;
};

namespace {

inline double min_image(double d, double period) {
  if (period > 0.0) {
    if (d > 0.5 * period) d -= period;
    else if (d < -0.5 * period) d += period;
  }
  return d;
}

// vertex coordinates of triangle t, the 2nd and 3rd unwrapped relative to the first (reading C19)
void triangle_xy(const orc_mesh *m, int64_t t, double x[3][2]) {
  const int32_t *v = &m->tri[3 * t];
  x[0][0] = m->xy[2 * v[0]];
  x[0][1] = m->xy[2 * v[0] + 1];
  for (int j = 1; j < 3; ++j)
    for (int d = 0; d < 2; ++d)
      x[j][d] = x[0][d] + min_image(m->xy[2 * v[j] + d] - x[0][d], m->period[d]);
}

void gather(const orc_mesh *m, const std::vector<double> &W, int64_t t, double w[3][4]) {
  const int32_t *v = &m->tri[3 * t];
  for (int j = 0; j < 3; ++j)
    for (int k = 0; k < 4; ++k) w[j][k] = W[k * m->nv + v[j]];
}

}  // namespace

extern "C" {

const char *orc_last_error(void) { return g_err.c_str(); }

int orc_mesh_create(orc_mesh **out, double gamma, double cfl, int scheme, int time_order, double period_x,
                    double period_y, int64_t nv, const double *xy, int64_t nt, const int32_t *tri,
                    const uint8_t *vertex_flag, int64_t ne, const int32_t *wall_edge) {
  if (!out || !xy || !tri || nv < 3 || nt < 1) return fail(ORC_EINVAL, "null or empty mesh");
  if (!(gamma > 1.0) || !(cfl > 0.0)) return fail(ORC_EINVAL, "gamma must be > 1 and cfl > 0");
  if (scheme < 0 || scheme > 5 || (time_order != 1 && time_order != 2)) return fail(ORC_EINVAL, "bad scheme/time_order");
  if (ne < 0 || (ne > 0 && !wall_edge)) return fail(ORC_EINVAL, "bad wall edge list");
  orc_mesh *m = new (std::nothrow) orc_mesh();
  if (!m) return fail(ORC_ENOMEM, "out of memory");
  m->gamma = gamma; m->cfl = cfl; m->scheme = scheme; m->time_order = time_order;
  m->period[0] = period_x; m->period[1] = period_y;
  m->nv = nv; m->nt = nt; m->ne = ne;
  m->xy.assign(xy, xy + 2 * nv);
  m->tri.assign(tri, tri + 3 * nt);
  m->flag.assign(nv, 0);
  if (vertex_flag) m->flag.assign(vertex_flag, vertex_flag + nv);
  m->geo.resize(nt);
  m->vol.assign(nv, 0.0);
  std::vector<int> deg(nv, 0);
  for (int64_t t = 0; t < nt; ++t) {
    int32_t *v = &m->tri[3 * t];
    for (int j = 0; j < 3; ++j)
      if (v[j] < 0 || v[j] >= nv) { delete m; return fail(ORC_EINVAL, "triangle index out of range"); }
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) { delete m; return fail(ORC_EINVAL, "degenerate triangle"); }
    double x[3][2];
    triangle_xy(m, t, x);
    double cross = (x[1][0] - x[0][0]) * (x[2][1] - x[0][1]) - (x[1][1] - x[0][1]) * (x[2][0] - x[0][0]);
    if (cross == 0.0) { delete m; return fail(ORC_EINVAL, "zero-area triangle"); }
    if (cross < 0.0) {  // make counter-clockwise
      std::swap(v[1], v[2]);
      triangle_xy(m, t, x);
    }
    triangle_geometry(x, m->geo[t]);
    for (int j = 0; j < 3; ++j) {
      m->vol[v[j]] += m->geo[t].area / 3.0;  // O1: V_i = sum_{T ni i} |T|/3
      deg[v[j]]++;
    }
  }
  for (int64_t i = 0; i < nv; ++i)
    if (deg[i] == 0) { delete m; return fail(ORC_EINVAL, "vertex without triangle"); }
  {  // domain size L of eq. 56: larger side of the bounding box, the period where periodic (reading C25)
    double lo[2] = {xy[0], xy[1]}, hi[2] = {xy[0], xy[1]};
    for (int64_t i = 0; i < nv; ++i)
      for (int d = 0; d < 2; ++d) {
        lo[d] = std::min(lo[d], xy[2 * i + d]);
        hi[d] = std::max(hi[d], xy[2 * i + d]);
      }
    double side[2];
    for (int d = 0; d < 2; ++d) side[d] = m->period[d] > 0.0 ? m->period[d] : hi[d] - lo[d];
    m->Ldom = std::max(side[0], side[1]);
  }
  // wall edges: outward unit normal = away from the third vertex of the one triangle holding the edge
  if (ne > 0) {
    m->wedge.assign(wall_edge, wall_edge + 2 * ne);
    m->wnx.resize(ne); m->wny.resize(ne); m->wlen.resize(ne);
    // the one triangle holding each wall edge: hash the wall edges, then one pass over the triangles
    std::unordered_map<uint64_t, int64_t> edge_of;
    auto key = [](int32_t a, int32_t b) { return ((uint64_t)(uint32_t)std::min(a, b) << 32) | (uint32_t)std::max(a, b); };
    for (int64_t e = 0; e < ne; ++e) {
      int32_t a = m->wedge[2 * e], b = m->wedge[2 * e + 1];
      if (a < 0 || a >= nv || b < 0 || b >= nv || a == b) { delete m; return fail(ORC_EINVAL, "bad wall edge"); }
      if (!edge_of.emplace(key(a, b), e).second) { delete m; return fail(ORC_EINVAL, "duplicate wall edge"); }
    }
    std::vector<int64_t> tri_of(ne, -1);
    std::vector<int> count_of(ne, 0);
    for (int64_t t = 0; t < nt; ++t) {
      const int32_t *v = &m->tri[3 * t];
      for (int j = 0; j < 3; ++j) {
        auto it = edge_of.find(key(v[j], v[(j + 1) % 3]));
        if (it != edge_of.end()) { tri_of[it->second] = t; count_of[it->second]++; }
      }
    }
    for (int64_t e = 0; e < ne; ++e) {
      int32_t a = m->wedge[2 * e], b = m->wedge[2 * e + 1];
      if (count_of[e] != 1) { delete m; return fail(ORC_EINVAL, "wall edge must belong to exactly one triangle"); }
      int64_t found = tri_of[e];
      const int32_t *v = &m->tri[3 * found];
      double x[3][2];
      triangle_xy(m, found, x);
      int ia = (v[0] == a ? 0 : (v[1] == a ? 1 : 2)), ib = (v[0] == b ? 0 : (v[1] == b ? 1 : 2)), ic = 3 - ia - ib;
      double ex = x[ib][0] - x[ia][0], ey = x[ib][1] - x[ia][1];
      double len = std::sqrt(ex * ex + ey * ey);
      double nx = ey / len, ny = -ex / len;
      double mx = 0.5 * (x[ia][0] + x[ib][0]), my = 0.5 * (x[ia][1] + x[ib][1]);
      if (nx * (x[ic][0] - mx) + ny * (x[ic][1] - my) > 0.0) { nx = -nx; ny = -ny; }
      m->wnx[e] = nx; m->wny[e] = ny; m->wlen[e] = len;
    }
  }
  m->W.assign(4 * nv, 0.0);
  m->Wic.assign(4 * nv, 0.0);
  m->Ws.assign(4 * nv, 0.0);
  m->phi.assign(12 * nt, 0.0);
  m->phiN_n.assign(12 * nt, 0.0);
  m->phiT_n.assign(4 * nt, 0.0);
  m->sT.assign(nt, 0.0);
  m->acc.assign(4 * nv, 0.0);
  m->wallN.assign(8 * (ne > 0 ? ne : 1), 0.0);
  *out = m;
  return ORC_OK;
}

void orc_mesh_destroy(orc_mesh *m) { delete m; }

int orc_set_lumping(orc_mesh *m, int lumping) {
  if (!m || (lumping != 0 && lumping != 1)) return fail(ORC_EINVAL, "lumping must be 0 (global) or 1 (selective)");
  m->lumping = lumping;
  return ORC_OK;
}

int orc_set_num_threads(orc_mesh *m, int n) {
  if (!m || n < 1) return fail(ORC_EINVAL, "bad thread count");
  m->nthreads = n;
  return ORC_OK;
}

int orc_set_state(orc_mesh *m, const double *W) {
  if (!m || !W) return fail(ORC_EINVAL, "null argument");
  m->W.assign(W, W + 4 * m->nv);
  m->Wic = m->W;
  m->t = 0.0;
  m->has_state = true;
  return ORC_OK;
}

int orc_get_state(const orc_mesh *m, double *W) {
  if (!m || !W) return fail(ORC_EINVAL, "null argument");
  std::memcpy(W, m->W.data(), sizeof(double) * 4 * m->nv);
  return ORC_OK;
}

int orc_get_geometry(const orc_mesh *m, double *area, double *vol) {
  if (!m) return fail(ORC_EINVAL, "null argument");
  if (area) for (int64_t t = 0; t < m->nt; ++t) area[t] = m->geo[t].area;
  if (vol) std::memcpy(vol, m->vol.data(), sizeof(double) * m->nv);
  return ORC_OK;
}

int orc_get_diagnostics(const orc_mesh *m, double totals[4], double *min_rho, double *min_p) {
  if (!m) return fail(ORC_EINVAL, "null argument");
  double tot[4] = {0, 0, 0, 0}, mr = INFINITY, mp = INFINITY;
  for (int64_t i = 0; i < m->nv; ++i) {
    double w[4];
    for (int k = 0; k < 4; ++k) { w[k] = m->W[k * m->nv + i]; tot[k] += m->vol[i] * w[k]; }
    double p = (m->gamma - 1.0) * (w[3] - 0.5 * (w[1] * w[1] + w[2] * w[2]) / w[0]);
    mr = std::min(mr, w[0]);
    mp = std::min(mp, p);
  }
  if (totals) for (int k = 0; k < 4; ++k) totals[k] = tot[k];
  if (min_rho) *min_rho = mr;
  if (min_p) *min_p = mp;
  return ORC_OK;
}

}  // extern "C"

namespace {

// |v|_max - |v|_min over all vertices of the state W (Bx, eq. 56)
BxCtx<double> bx_context(const orc_mesh *m, const std::vector<double> &W) {
  double vmax = 0.0, vmin = INFINITY;
  for (int64_t i = 0; i < m->nv; ++i) {
    double u = W[m->nv + i] / W[i], v = W[2 * m->nv + i] / W[i];
    double a = std::sqrt(u * u + v * v);
    vmax = std::max(vmax, a);
    vmin = std::min(vmin, a);
  }
  return BxCtx<double>{m->Ldom, vmax - vmin};
}

// Stage-1 triangle loop over the state `W`: fills m->phi (scheme residuals), m->phiN_n, m->phiT_n, m->sT.
int stage1_triangles(orc_mesh *m, const std::vector<double> &W, double *dump_LDA, double *dump_B) {
  int bad = 0;
  BxCtx<double> bx{m->Ldom, 0.0};
  if (m->scheme == ORC_SCHEME_BX) bx = bx_context(m, W);
#pragma omp parallel for schedule(static) num_threads(m->nthreads) reduction(| : bad)
  for (int64_t t = 0; t < m->nt; ++t) {
    double w[3][4];
    gather(m, W, t, w);
    Core<double> core;
    Stage1Out<double> o;
    if (triangle_stage1(m->gamma, m->scheme, w, m->geo[t], core, o, &bx)) { bad |= 1; continue; }
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 4; ++k) {
        m->phi[12 * t + 4 * i + k] = o.phiB[i][k];
        m->phiN_n[12 * t + 4 * i + k] = o.phiN[i][k];
        if (dump_LDA) dump_LDA[12 * t + 4 * i + k] = o.phiLDA[i][k];
        if (dump_B) dump_B[12 * t + 4 * i + k] = o.phiB[i][k];
      }
    for (int k = 0; k < 4; ++k) m->phiT_n[4 * t + k] = o.phiT[k];
    m->sT[t] = o.sT;
  }
  return bad ? ORC_ENONPHYSICAL : ORC_OK;
}

int stage2_triangles(orc_mesh *m, double dt) {
  int bad = 0;
  BxCtx<double> bx{m->Ldom, 0.0};
  if (m->scheme == ORC_SCHEME_BX) bx = bx_context(m, m->Ws);
#pragma omp parallel for schedule(static) num_threads(m->nthreads) reduction(| : bad)
  for (int64_t t = 0; t < m->nt; ++t) {
    double wn[3][4], ws[3][4], pN[3][4], pT[4];
    gather(m, m->W, t, wn);
    gather(m, m->Ws, t, ws);
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 4; ++k) pN[i][k] = m->phiN_n[12 * t + 4 * i + k];
    for (int k = 0; k < 4; ++k) pT[k] = m->phiT_n[4 * t + k];
    Core<double> core;
    Stage2Out<double> o;
    if (triangle_stage2(m->gamma, m->scheme, wn, ws, m->geo[t], dt, pT, pN, core, o, m->lumping, &bx)) { bad |= 1; continue; }
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 4; ++k) m->phi[12 * t + 4 * i + k] = o.PhiB[i][k];
  }
  return bad ? ORC_ENONPHYSICAL : ORC_OK;
}

// scatter-add of the per-triangle distributed residuals into the per-vertex accumulators, in
// triangle order (reading C20), i.e. the sum over T containing i of eq. 43 / 60 / 61
void scatter(orc_mesh *m) {
  std::fill(m->acc.begin(), m->acc.end(), 0.0);
  for (int64_t t = 0; t < m->nt; ++t) {
    const int32_t *v = &m->tri[3 * t];
    for (int i = 0; i < 3; ++i)
      for (int k = 0; k < 4; ++k) m->acc[4 * (int64_t)v[i] + k] += m->phi[12 * t + 4 * i + k];
  }
}

int one_step(orc_mesh *m, double t_end, double *dt_out) {
  const int64_t nv = m->nv;
  // --- stage 1 residuals and signal speeds at W^n
  int rc = stage1_triangles(m, m->W, nullptr, nullptr);
  if (rc) return fail(rc, "non-physical state met in stage 1");
  // --- O7: dt = CFL * min_i 2 V_i / sum_{T ni i} s_T  (eq. 44), clipped to t_end (reading C13)
  std::vector<double> S(nv, 0.0);
  for (int64_t t = 0; t < m->nt; ++t)
    for (int i = 0; i < 3; ++i) S[m->tri[3 * t + i]] += m->sT[t];
  double bound = INFINITY;
  for (int64_t i = 0; i < nv; ++i) bound = std::min(bound, 2.0 * m->vol[i] / S[i]);
  double dt = m->cfl * bound;
  if (t_end > 0.0 && m->t + dt > t_end) dt = t_end - m->t;
  // --- O8: W* = W^n - dt/V_i [sum_T phi_i + wall terms]  (eq. 60 / eq. 43)
  scatter(m);
  for (int64_t e = 0; e < m->ne; ++e) {
    int32_t a = m->wedge[2 * e], b = m->wedge[2 * e + 1];
    double wa[4], wb[4];
    for (int k = 0; k < 4; ++k) { wa[k] = m->W[k * nv + a]; wb[k] = m->W[k * nv + b]; }
    double *Pa = &m->wallN[8 * e], *Pb = &m->wallN[8 * e + 4];
    if (!wall_edge(m->gamma, wa, wb, m->wnx[e], m->wny[e], m->wlen[e], Pa, Pb))
      return fail(ORC_ENONPHYSICAL, "non-physical state on a wall edge");
    for (int k = 0; k < 4; ++k) { m->acc[4 * (int64_t)a + k] += Pa[k]; m->acc[4 * (int64_t)b + k] += Pb[k]; }
  }
  for (int64_t i = 0; i < nv; ++i)
    for (int k = 0; k < 4; ++k)
      m->Ws[k * nv + i] = m->flag[i] ? m->Wic[k * nv + i] : m->W[k * nv + i] - dt / m->vol[i] * m->acc[4 * i + k];
  if (m->time_order == 2) {
    // --- O9-O10: second stage (eq. 61)
    rc = stage2_triangles(m, dt);
    if (rc) return fail(rc, "non-physical state met in stage 2");
    scatter(m);
    for (int64_t e = 0; e < m->ne; ++e) {
      int32_t a = m->wedge[2 * e], b = m->wedge[2 * e + 1];
      double wa[4], wb[4], Pa[4], Pb[4];
      for (int k = 0; k < 4; ++k) { wa[k] = m->Ws[k * nv + a]; wb[k] = m->Ws[k * nv + b]; }
      if (!wall_edge(m->gamma, wa, wb, m->wnx[e], m->wny[e], m->wlen[e], Pa, Pb))
        return fail(ORC_ENONPHYSICAL, "non-physical state on a wall edge");
      for (int k = 0; k < 4; ++k) {  // reading C15: (Phi^c(W^n) + Phi^c(W*)) / 2
        m->acc[4 * (int64_t)a + k] += 0.5 * (m->wallN[8 * e + k] + Pa[k]);
        m->acc[4 * (int64_t)b + k] += 0.5 * (m->wallN[8 * e + 4 + k] + Pb[k]);
      }
    }
    for (int64_t i = 0; i < nv; ++i)
      for (int k = 0; k < 4; ++k)
        m->Ws[k * nv + i] = m->flag[i] ? m->Wic[k * nv + i] : m->Ws[k * nv + i] - dt / m->vol[i] * m->acc[4 * i + k];
  }
  // positivity of the new state (so that a failed step leaves W at the last completed step)
  for (int64_t i = 0; i < nv; ++i) {
    double r = m->Ws[i], mx = m->Ws[nv + i], my = m->Ws[2 * nv + i], e = m->Ws[3 * nv + i];
    double p = (m->gamma - 1.0) * (e - 0.5 * (mx * mx + my * my) / r);
    if (!(r > 0.0) || !(p > 0.0)) return fail(ORC_ENONPHYSICAL, "update produced rho <= 0 or p <= 0");
  }
  m->W.swap(m->Ws);
  m->t += dt;
  *dt_out = dt;
  return ORC_OK;
}

}  // namespace

extern "C" {

int orc_step(orc_mesh *m, int64_t max_steps, double t_end, int64_t *steps_done, double *t, double *dt_last) {
  if (!m || !m->has_state) return fail(ORC_EINVAL, "no state set");
  int64_t n = 0;
  double dt = 0.0;
  int rc = ORC_OK;
  while (n < max_steps && !(t_end > 0.0 && m->t >= t_end)) {
    rc = one_step(m, t_end, &dt);
    if (rc) break;
    ++n;
  }
  if (steps_done) *steps_done = n;
  if (t) *t = m->t;
  if (dt_last) *dt_last = dt;
  return rc;
}

int orc_dump_stage1(orc_mesh *m, double *phiT, double *phiN, double *phiLDA, double *phiB, double *sT) {
  if (!m || !m->has_state) return fail(ORC_EINVAL, "no state set");
  int rc = stage1_triangles(m, m->W, phiLDA, phiB);
  if (rc) return fail(rc, "non-physical state");
  if (phiT) std::memcpy(phiT, m->phiT_n.data(), sizeof(double) * 4 * m->nt);
  if (phiN) std::memcpy(phiN, m->phiN_n.data(), sizeof(double) * 12 * m->nt);
  if (sT) std::memcpy(sT, m->sT.data(), sizeof(double) * m->nt);
  return ORC_OK;
}

void orc_euler_matrices(double gamma, double u, double v, double h, double nx, double ny, double len, double K[16],
                        double Kp[16], double Km[16]) {
  double c = std::sqrt((gamma - 1.0) * (h - 0.5 * (u * u + v * v)));
  double hl = len / 2.0;
  double w = u * nx + v * ny;
  double lam[3] = {w + c, w - c, w}, lp[3], lm[3];
  for (int k = 0; k < 3; ++k) {
    lp[k] = hl * (0.5 * (lam[k] + std::fabs(lam[k])));
    lm[k] = hl * (0.5 * (lam[k] - std::fabs(lam[k])));
  }
  if (K) euler_K(gamma, u, v, h, nx, ny, hl, K);
  if (Kp) euler_K_split(gamma, u, v, h, c, nx, ny, lp[0], lp[1], lp[2], Kp);
  if (Km) euler_K_split(gamma, u, v, h, c, nx, ny, lm[0], lm[1], lm[2], Km);
}

void orc_euler_matrices_l(double gamma, double u, double v, double h, double nx, double ny, double l1, double l2,
                          double l3, double K[16]) {
  double c = std::sqrt((gamma - 1.0) * (h - 0.5 * (u * u + v * v)));
  euler_K_split(gamma, u, v, h, c, nx, ny, l1, l2, l3, K);
}

void orc_eigenvectors(double gamma, double u, double v, double h, double nx, double ny, double R[16],
                      double Rinv[16], double lambda[4]) {
  double g1 = gamma - 1.0;
  double c = std::sqrt(g1 * (h - 0.5 * (u * u + v * v)));
  double w = u * nx + v * ny, alpha = g1 * (u * u + v * v) / 2.0;
  double ac = alpha / c, uc = u / c, vc = v / c;
  // eq. A7 (columns = e1..e4 of eq. A3-A6)
  double Rm[16] = {1, 1, 0, 1,
                   u + c * nx, u - c * nx, -ny, u,
                   v + c * ny, v - c * ny, nx, v,
                   h + c * w, h - c * w, v * nx - u * ny, alpha / g1};
  // eq. A8 with the 4th column corrected (reading C7), |n| = 1
  double s = 1.0 / (2.0 * c);
  double Ri[16] = {s * (ac - w), s * (nx - g1 * uc), s * (ny - g1 * vc), s * (g1 / c),
                   s * (ac + w), s * (-nx - g1 * uc), s * (-ny - g1 * vc), s * (g1 / c),
                   s * (2 * c * (u * ny - v * nx)), s * (-2 * c * ny), s * (2 * c * nx), 0.0,
                   s * (2 * c - 2 * ac), s * (2 * g1 * uc), s * (2 * g1 * vc), s * (-2 * g1 / c)};
  if (R) std::memcpy(R, Rm, sizeof Rm);
  if (Rinv) std::memcpy(Rinv, Ri, sizeof Ri);
  if (lambda) { lambda[0] = w + c; lambda[1] = w - c; lambda[2] = w; lambda[3] = w; }
}

int orc_triangle_stage1(double gamma, const double *W, const double *xy, double *phiT, double *phiN,
                        double *phiLDA, double *phiB, double *theta, double *sT, double *Nhat, double *sumKm) {
  double w[3][4], x[3][2];
  std::memcpy(w, W, sizeof w);
  std::memcpy(x, xy, sizeof x);
  Geom<double> g;
  triangle_geometry(x, g);
  if (!(g.area > 0.0)) return fail(ORC_EINVAL, "triangle must be counter-clockwise");
  Core<double> core;
  Stage1Out<double> o;
  int rc = triangle_stage1(gamma, ORC_SCHEME_B, w, g, core, o);
  if (rc) return fail(rc, "non-physical state");
  if (phiT) std::memcpy(phiT, o.phiT, sizeof o.phiT);
  if (phiN) std::memcpy(phiN, o.phiN, sizeof o.phiN);
  if (phiLDA) std::memcpy(phiLDA, o.phiLDA, sizeof o.phiLDA);
  if (phiB) std::memcpy(phiB, o.phiB, sizeof o.phiB);
  if (theta) std::memcpy(theta, o.theta, sizeof o.theta);
  if (sT) *sT = o.sT;
  if (Nhat) std::memcpy(Nhat, core.Nhat, sizeof core.Nhat);
  if (sumKm) std::memcpy(sumKm, core.sumKm, sizeof core.sumKm);
  return ORC_OK;
}

static thread_local int g_stage2_lumping = 0;
void orc_triangle_stage2_lumping(int lumping) { g_stage2_lumping = lumping; }

int orc_triangle_stage2(double gamma, const double *Wn, const double *Ws, const double *xy, double dt,
                        const double *phiT_n, const double *phiN_n, double *PhiT, double *PhiN, double *PhiLDA,
                        double *PhiB) {
  double wn[3][4], ws[3][4], x[3][2], pT[4], pN[3][4];
  std::memcpy(wn, Wn, sizeof wn);
  std::memcpy(ws, Ws, sizeof ws);
  std::memcpy(x, xy, sizeof x);
  std::memcpy(pT, phiT_n, sizeof pT);
  std::memcpy(pN, phiN_n, sizeof pN);
  Geom<double> g;
  triangle_geometry(x, g);
  if (!(g.area > 0.0)) return fail(ORC_EINVAL, "triangle must be counter-clockwise");
  Core<double> core;
  Stage2Out<double> o;
  int rc = triangle_stage2(gamma, ORC_SCHEME_B, wn, ws, g, dt, pT, pN, core, o, g_stage2_lumping);
  if (rc) return fail(rc, "non-physical state");
  if (PhiT) std::memcpy(PhiT, o.PhiT, sizeof o.PhiT);
  if (PhiN) std::memcpy(PhiN, o.PhiN, sizeof o.PhiN);
  if (PhiLDA) std::memcpy(PhiLDA, o.PhiLDA, sizeof o.PhiLDA);
  if (PhiB) std::memcpy(PhiB, o.PhiB, sizeof o.PhiB);
  return ORC_OK;
}

void orc_wall_edge(double gamma, const double *Wa, const double *Wb, double nx, double ny, double len,
                   double *Phi_a, double *Phi_b) {
  wall_edge(gamma, Wa, Wb, nx, ny, len, Phi_a, Phi_b);
}

int orc_count_ops(double gamma, const double *W, const double *xy, int stage, int scheme, int64_t counts[6]) {
  Cnt w[3][4], x[3][2];
  for (int j = 0; j < 3; ++j) {
    for (int k = 0; k < 4; ++k) w[j][k] = Cnt(W[4 * j + k]);
    for (int d = 0; d < 2; ++d) x[j][d] = Cnt(xy[2 * j + d]);
  }
  Geom<Cnt> g;
  triangle_geometry(x, g);  // geometry is precomputed per mesh: not counted
  g_ops = OpCounts();
  Core<Cnt> core;
  int rc;
  if (stage == 1) {
    Stage1Out<Cnt> o;
    rc = triangle_stage1(Cnt(gamma), scheme, w, g, core, o);
  } else {
    Stage1Out<Cnt> o1;
    rc = triangle_stage1(Cnt(gamma), scheme, w, g, core, o1);
    g_ops = OpCounts();
    Stage2Out<Cnt> o;
    if (!rc) rc = triangle_stage2(Cnt(gamma), scheme, w, w, g, Cnt(1.0), o1.phiT, o1.phiN, core, o);
  }
  counts[0] = g_ops.add; counts[1] = g_ops.mul; counts[2] = g_ops.div;
  counts[3] = g_ops.sqrt; counts[4] = g_ops.abs; counts[5] = g_ops.cmp;
  return rc ? fail(rc, "non-physical state") : ORC_OK;
}

}  // extern "C"
