// mrd_meshgen.cu -- the mesh-generation layer (section 2.3-2.4 and 4.1): parallel Delaunay refinement
// of bounded domains on the GPU, entry points mrd_meshgen_* of include/mrd.h.
//
//   test_quality    for every triangle the circumradius r of eq. 2 (L146), the circumradius-to-shortest-edge ratio beta
//                   (L118-L126), the flag "r > R or beta > B" (L150) and the circumcentre, where the new vertex goes (L150);
//   orient2d        the sign of the determinant of eq. 3 (L160), EXACT (also without any allocation: orient2d_static);
//   incircle2d      the sign of the determinant of eq. 5 (L198), EXACT;
//   build_edges     triangleEdges and edgeTriangles from triangleVertices (section 4.1.2);
//   delaunay_flip   flips of independent sets of edges until every edge is locally Delaunay (section 2.4.6, 4.1.5);
//   find_triangle   the triangle containing a point, by walking (section 2.4.2);
//   refine          the six steps of section 2.4 with the parallel insertion set of section 4.1.1 and the re-sort of 4.1.4.
//
// test_quality is written operation by operation with round-to-nearest intrinsics (no FMA contraction), so that it agrees
// bit for bit with the CPU oracle (oracle/meshgen.py), which evaluates the same formulas in the same order.
// The predicates must be exact (L162-L166, L665-L667: "mutually contradictory results inevitably lead to ... invalid
// triangulations").  The paper uses adaptive exact predicates; here (mrd_predicates.cuh): a floating-point FILTER with a
// rigorous error bound decides almost every test; the rest are evaluated exactly in floating-point expansion arithmetic
// (error-free transformations TwoSum / TwoProduct with FMA; sums of non-overlapping components with zero elimination) -- in
// place, in short thread-local expansions, when the translations of the test are exact, else by threads that own 19 KB of
// scratch each.  The sign of an expansion is the sign of its largest component.
// Every integer decision of the refinement (candidate order, priorities, numbering) is a function of the input alone, so the
// result is, array for array, the oracle's; DESIGN.md section 9c lists the readings M1-M16 behind that.
#include <cuda_runtime.h>
#include <cooperative_groups.h>

#include <algorithm>
#include <cstdint>
#include <cub/device/device_merge_sort.cuh>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/device/device_select.cuh>
#include <mutex>
#include <string>
#include <thrust/iterator/counting_iterator.h>

#include "../../include/mrd.h"
#include "mrd_predicates.cuh"

// Scratch of mrd_meshgen_orient2d_static (the entry point that allocates nothing): 256 bytes that hold the length of the work
// list, then the work list itself (one int32 per test the filter could not decide).  4 MB + 256 B, held by every GPU that loads
// the library until the process exits.  In HOST code this name is a stand-in, not a device address: the host takes the
// address once per device with cudaGetSymbolAddress (static_scratch_of below) and passes THAT to the kernels.
#define MRD_STATIC_MAX_TESTS (1 << 20)
static __device__ __align__(256) unsigned char g_static_scratch[256 + sizeof(int32_t) * MRD_STATIC_MAX_TESTS];

namespace mrdgen {

// ------------------------------------------------------------------------------------------------------------------
// TestQuality (eq. 2): one thread per triangle
// ------------------------------------------------------------------------------------------------------------------
// Size bound as a function of space (section 2.3.1; reading M16): factors on a grid over a rectangle, interpolated
// bilinearly at the circumcentre, one IEEE operation at a time in the oracle's order.  g == nullptr: the factor is 1.
struct SizeGrid {
  const double *g;        // [ny][nx], row-major
  int nx, ny;
  double x0, y0, sx, sy;  // sx = (nx - 1) / (x1 - x0)
  __device__ __forceinline__ double at(double2 p) const {
    const double fx = fmin(fmax(__dmul_rn(__dsub_rn(p.x, x0), sx), 0.0), (double)(nx - 1));
    const double fy = fmin(fmax(__dmul_rn(__dsub_rn(p.y, y0), sy), 0.0), (double)(ny - 1));
    const double fi = fmin(floor(fx), (double)(nx - 2)), fj = fmin(floor(fy), (double)(ny - 2));
    const int i = (int)fi, j = (int)fj;
    const double tx = __dsub_rn(fx, fi), ty = __dsub_rn(fy, fj), ux = __dsub_rn(1.0, tx), uy = __dsub_rn(1.0, ty);
    const double *row = g + (int64_t)j * nx + i;
    const double g0 = __dadd_rn(__dmul_rn(row[0], ux), __dmul_rn(row[1], tx));
    const double g1 = __dadd_rn(__dmul_rn(row[nx], ux), __dmul_rn(row[nx + 1], tx));
    return __dadd_rn(__dmul_rn(g0, uy), __dmul_rn(g1, ty));
  }
};
__global__ void __launch_bounds__(256)
test_quality_kernel(int64_t nt, const double2 *__restrict__ xy, const int32_t *__restrict__ tri, double R, double B,
                    double *__restrict__ r_out, double *__restrict__ beta_out, double2 *__restrict__ cc_out,
                    uint8_t *__restrict__ bad_out, unsigned long long *__restrict__ n_bad, SizeGrid size) {
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
    const double2 cc = make_double2(__dadd_rn(c.x, ux), __dadd_rn(c.y, uy));
    cc_out[t] = cc;
    if (size.g && det > 0.0) R = __dmul_rn(R, size.at(cc));
    bad = (r > R || beta > B) ? 1 : 0;   // L150 (a triangle with det <= 0 has r <= 0 or inf: flagged by beta or not at all; the
    if (!(det > 0.0)) bad = 1;           //       mesh is counter-clockwise, so det <= 0 is itself a defect: flag it)
    bad_out[t] = (uint8_t)bad;
  }
  // count: warp ballot -> one atomic per warp
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_bad, (unsigned long long)__popc(m));
}

// ------------------------------------------------------------------------------------------------------------------
// Filter kernels: the determinant in plain fp64 and a bound on its rounding error; undecided tests go to a work list
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
orient_filter_kernel(int64_t n, const double2 *__restrict__ xy, const int32_t *__restrict__ idx, int8_t *__restrict__ sign,
                     int32_t *__restrict__ work, unsigned long long *__restrict__ n_work) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n) return;
  const int sg = orient2d_filter(xy[idx[3 * k]], xy[idx[3 * k + 1]], xy[idx[3 * k + 2]]);
  sign[k] = (int8_t)sg;
  if (sg == 2) work[atomicAdd(n_work, 1ull)] = (int32_t)k;
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
  const int sg = incircle2d_filter(xy[idx[4 * k]], xy[idx[4 * k + 1]], xy[idx[4 * k + 2]], xy[idx[4 * k + 3]]);
  sign[k] = (int8_t)sg;
  if (sg == 2) work[atomicAdd(n_work, 1ull)] = (int32_t)k;
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

// ------------------------------------------------------------------------------------------------------------------
// Mesh data structure (section 4.1.2): triangleEdges and edgeTriangles from triangleVertices
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
edge_keys_kernel(int64_t n, const int32_t *__restrict__ tv, int bits, unsigned long long *__restrict__ key, int32_t *__restrict__ val) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int64_t t = i / 3;
  const int k = (int)(i - 3 * t);
  const unsigned a = (unsigned)tv[3 * t + (k + 1) % 3], b = (unsigned)tv[3 * t + (k + 2) % 3];   // edge k is opposite local vertex k
  key[i] = ((unsigned long long)min(a, b) << bits) | max(a, b);   // `bits` >= the width of a vertex number: sorts by (smaller, larger)
  val[i] = (int32_t)i;
}
__global__ void __launch_bounds__(256)
edge_heads_kernel(int64_t n, const unsigned long long *__restrict__ key, int32_t *__restrict__ head) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) head[i] = (i == 0 || key[i] != key[i - 1]) ? 1 : 0;
}
// incl = inclusive sum of head: sorted entry i belongs to edge incl[i] - 1
__global__ void __launch_bounds__(256)
edge_fill_kernel(int64_t n, const unsigned long long *__restrict__ key, const int32_t *__restrict__ val, const int32_t *__restrict__ incl,
                 int32_t *__restrict__ te, int32_t *__restrict__ et, int *__restrict__ err) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t e = incl[i] - 1;
  const int slot = (i > 0 && key[i] == key[i - 1]) ? 1 : 0;
  if (i > 1 && key[i] == key[i - 2]) { *err = 1; return; }      // an edge with three triangles
  te[val[i]] = e;
  et[2 * (int64_t)e + slot] = val[i] / 3;                        // (the sort is stable: ascending triangle order)
}

// ------------------------------------------------------------------------------------------------------------------
// Delaunay triangulator (section 2.4.6, 4.1.5)
// ------------------------------------------------------------------------------------------------------------------
struct FlipCounters { unsigned long long n_work, n_bad, n_flip, n_next, n_exact; };

// Bookkeeping of the refinement's in-place renumbering (reading M15), all optional (null members: nothing is recorded):
// T[t] / E[e] = 1 when triangle slot t / edge slot e received a new content (its old triangle / edge does not exist any
// more, or the slot is new); list / n: the edges whose quadrilateral changed, once each (mark[e] = -1), as the first
// candidates of the flip loop.
struct Touch {
  uint8_t *T, *E;
  int32_t *mark, *list;
  unsigned long long *n;
  __device__ __forceinline__ void tri(int32_t t) const { if (T) T[t] = 1; }
  __device__ __forceinline__ void edge(int32_t e) const { if (E) E[e] = 1; }
  // (one atomicAdd on the list's length per thread, not per edge: up to 3 M increments of one address serialise in L2)
  struct Pending { int32_t e[8]; int n; };
  __device__ __forceinline__ void check(int32_t e, Pending &p) const {
    if (list && atomicExch(mark + e, -1) != -1) p.e[p.n++] = e;
  }
  __device__ __forceinline__ void flush(const Pending &p) const {
    if (p.n == 0) return;
    const unsigned long long base = atomicAdd(n, (unsigned long long)p.n);
    for (int q = 0; q < p.n; ++q) list[base + q] = p.e[q];
  }
};

struct Quad { int32_t t1, t2; double2 a, b, c, d; };
static __device__ __forceinline__ bool load_quad(int32_t e, const double2 *xy, const int32_t *tv, const int32_t *te, const int32_t *et, Quad &q) {
  q.t1 = et[2 * (int64_t)e];
  q.t2 = et[2 * (int64_t)e + 1];
  if (q.t2 < 0) return false;                                    // a boundary edge: Delaunay by definition
  const int32_t *e2 = te + 3 * (int64_t)q.t2;
  const int k2 = e2[0] == e ? 0 : (e2[1] == e ? 1 : 2);
  const int32_t *v1 = tv + 3 * (int64_t)q.t1;
  q.a = xy[v1[0]]; q.b = xy[v1[1]]; q.c = xy[v1[2]];
  q.d = xy[tv[3 * (int64_t)q.t2 + k2]];                          // "the one vertex of T' that is not part of T" (L192)
  return true;
}
// E is not Delaunay: note it and bid for its two triangles (independent set of section 4.1.5: the higher edge number wins;
// the iteration stamp in the upper half outbids every bid of an earlier iteration, so the locks are never reset)
static __device__ __forceinline__ void bid(int32_t e, const Quad &q, unsigned long long stamp, int8_t *state, unsigned long long *lock) {
  state[e] = 1;
  atomicMax(lock + q.t1, stamp | (unsigned)e);
  atomicMax(lock + q.t2, stamp | (unsigned)e);
}
// (counters: one atomic per warp, not per thread -- millions of increments of one address serialise in L2)
__global__ void __launch_bounds__(256)
check_edge_kernel(int64_t n, const int32_t *__restrict__ cand, const double2 *__restrict__ xy, const int32_t *__restrict__ tv,
                  const int32_t *__restrict__ te, const int32_t *__restrict__ et, int8_t *__restrict__ state,
                  unsigned long long *__restrict__ lock, unsigned long long stamp, int32_t *__restrict__ work, FlipCounters *c,
                  const unsigned long long *__restrict__ n_dev) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (n_dev) n = min(n, (int64_t)*n_dev);                          // (the host knows only an upper bound of the list's length)
  bool exact = false;
  if (i < n) {
    const int32_t e = cand ? cand[i] : (int32_t)i;
    Quad q;
    if (!load_quad(e, xy, tv, te, et, q)) state[e] = 0;
    else {
      int sg = incircle2d_filter(q.a, q.b, q.c, q.d);
      if (sg == 2) {                                               // exact, in place when the translations are exact
        sg = incircle2d_exact_short(q.a, q.b, q.c, q.d);
        exact = sg != 2;
      }
      if (sg == 2) work[atomicAdd(&c->n_work, 1ull)] = e;          // rare
      else if (sg == 1) { bid(e, q, stamp, state, lock); bad = true; }
      else state[e] = 0;
    }
  }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad), mx = __ballot_sync(0xFFFFFFFFu, exact);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(&c->n_bad, (unsigned long long)__popc(m));
  if ((threadIdx.x & 31) == 0 && mx) atomicAdd(&c->n_exact, (unsigned long long)__popc(mx));
}
__global__ void __launch_bounds__(32)
check_edge_exact_kernel(const int32_t *__restrict__ work, const double2 *__restrict__ xy, const int32_t *__restrict__ tv,
                        const int32_t *__restrict__ te, const int32_t *__restrict__ et, int8_t *__restrict__ state,
                        unsigned long long *__restrict__ lock, unsigned long long stamp, FlipCounters *c, double *__restrict__ scratch) {
  const int64_t nw = (int64_t)c->n_work;
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  double *acc = scratch + tid * (2 * MAXE), *tmp = acc + MAXE;
  for (int64_t w = tid; w < nw; w += (int64_t)gridDim.x * blockDim.x) {
    const int32_t e = work[w];
    Quad q;
    load_quad(e, xy, tv, te, et, q);
    if (incircle2d_exact(q.a, q.b, q.c, q.d, acc, tmp) > 0) {
      bid(e, q, stamp, state, lock);
      atomicAdd(&c->n_bad, 1ull);
    } else state[e] = 0;                                         // zero: four cocircular vertices, left alone
  }
  if (tid == 0) c->n_exact += (unsigned long long)nw;
}
__global__ void __launch_bounds__(256)
flip_kernel(int64_t n, const int32_t *__restrict__ cand, int32_t *__restrict__ tv, int32_t *__restrict__ te, int32_t *__restrict__ et,
            int8_t *__restrict__ state, const unsigned long long *__restrict__ lock, unsigned long long stamp, int32_t iter,
            int32_t *__restrict__ mark, int32_t *__restrict__ next, FlipCounters *c, const unsigned long long *__restrict__ n_dev,
            Touch touch) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (n_dev) n = min(n, (int64_t)*n_dev);
  int32_t items[4];                                              // this thread's candidates for the next iteration
  int cnt = 0;
  bool flipped = false;
  const int32_t e = i < n ? (cand ? cand[i] : (int32_t)i) : -1;
  if (e >= 0 && state[e] == 1) {
    const int32_t t1 = et[2 * (int64_t)e], t2 = et[2 * (int64_t)e + 1];
    const unsigned long long mine = stamp | (unsigned)e;
    if (lock[t1] != mine || lock[t2] != mine) {                  // lost a triangle to another edge: try again next iteration
      if (atomicExch(mark + e, iter) != iter) items[cnt++] = e;
    } else {
      // flip (L102): a opposite E in t1 = (a, b, c), d opposite E in t2 = (d, c, b)  ->  t1 = (a, b, d), t2 = (a, d, c)
      int32_t *v1 = tv + 3 * (int64_t)t1, *v2 = tv + 3 * (int64_t)t2, *e1 = te + 3 * (int64_t)t1, *e2 = te + 3 * (int64_t)t2;
      const int i1 = e1[0] == e ? 0 : (e1[1] == e ? 1 : 2), i2 = e2[0] == e ? 0 : (e2[1] == e ? 1 : 2);
      const int32_t a = v1[i1], b = v1[(i1 + 1) % 3], cc = v1[(i1 + 2) % 3], d = v2[i2];
      const int32_t e_ca = e1[(i1 + 1) % 3], e_ab = e1[(i1 + 2) % 3], e_bd = e2[(i2 + 1) % 3], e_dc = e2[(i2 + 2) % 3];
      v1[0] = a; v1[1] = b; v1[2] = d;
      e1[0] = e_bd; e1[1] = e; e1[2] = e_ab;
      v2[0] = a; v2[1] = d; v2[2] = cc;
      e2[0] = e_dc; e2[1] = e_ca; e2[2] = e;
      // repair edgeTriangles of the two edges that changed sides (section 4.1.5; in place: every thread rewrites only the
      // entry that names one of ITS two triangles, which no other flip of this iteration can name)
      int32_t *f = et + 2 * (int64_t)e_bd;
      f[f[0] == t2 ? 0 : 1] = t1;
      f = et + 2 * (int64_t)e_ca;
      f[f[0] == t1 ? 0 : 1] = t2;
      state[e] = 0;                                              // "E' would be locally Delaunay" (L102)
      touch.tri(t1);
      touch.tri(t2);
      touch.edge(e);
      const int32_t outer[4] = {e_ca, e_ab, e_bd, e_dc};         // their quadrilaterals changed: check them next
#pragma unroll
      for (int j = 0; j < 4; ++j)
        if (atomicExch(mark + outer[j], iter) != iter) items[cnt++] = outer[j];
      flipped = true;
    }
  }
  // append to the next list: warp prefix sum, one atomic per warp
  const int lane = threadIdx.x & 31;
  int incl = cnt;
#pragma unroll
  for (int dlt = 1; dlt < 32; dlt <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, dlt);
    if (lane >= dlt) incl += v;
  }
  const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
  unsigned long long base = 0;
  if (lane == 31 && total) base = atomicAdd(&c->n_next, (unsigned long long)total);
  base = __shfl_sync(0xFFFFFFFFu, base, 31);
  for (int j = 0; j < cnt; ++j) next[base + incl - cnt + j] = items[j];
  const unsigned fm = __ballot_sync(0xFFFFFFFFu, flipped);
  if (lane == 0 && fm) atomicAdd(&c->n_flip, (unsigned long long)__popc(fm));
}

// Small candidate sets (the late iterations of a flip loop, the late iterations of a refinement): the whole loop check -> flip ->
// check -> ... in ONE cooperative launch with grid-wide barriers between the phases, instead of three launches and a counter
// read-back per iteration.  Same decisions as check_edge_kernel / flip_kernel (the independent set does not depend on which
// thread looks at which edge).  A test that needs the long expansions cannot be done here (no scratch): the loop stops BEFORE
// that iteration changes anything and the host path takes over from it.
struct FlipLoopState {
  unsigned long long n_bad[2], n_next[2];   // indexed by the parity of the iteration
  unsigned long long n_flip, n_exact;       // accumulated
  unsigned long long n_cur;                 // out: candidates of the iteration the loop stopped at
  int done_iters, converged, abort;         // out
};
__global__ void __launch_bounds__(256)
flip_loop_kernel(int64_t n0, const unsigned long long *__restrict__ n0_dev, int32_t iter0, int max_iters, int32_t *list0, int32_t *list1,
                 const double2 *__restrict__ xy, int32_t *tv, int32_t *te, int32_t *et, int8_t *state, unsigned long long *lock,
                 int32_t *mark, FlipLoopState *st, Touch touch) {
  cooperative_groups::grid_group grid = cooperative_groups::this_grid();
  const int64_t total = (int64_t)gridDim.x * blockDim.x, gtid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int lane = threadIdx.x & 31;
  int64_t n = n0_dev ? min(n0, (int64_t)*n0_dev) : n0;
  int it = 0;
  bool converged = false;
  for (; it < max_iters; ++it) {
    const int32_t iter = iter0 + it;
    const int p = iter & 1;
    const unsigned long long stamp = (unsigned long long)iter << 32;
    const int32_t *cur = p ? list0 : list1;                       // (the host loop: next = list[iter & 1])
    int32_t *nxt = p ? list1 : list0;
    // ---- check
    for (int64_t base = 0; base < n; base += total) {
      const int64_t i = base + gtid;
      bool bad = false, exact = false;
      if (i < n) {
        const int32_t e = cur[i];
        Quad q;
        if (!load_quad(e, xy, tv, te, et, q)) state[e] = 0;
        else {
          int sg = incircle2d_filter(q.a, q.b, q.c, q.d);
          if (sg == 2) {
            sg = incircle2d_exact_short(q.a, q.b, q.c, q.d);
            exact = sg != 2;
          }
          if (sg == 2) st->abort = 1;
          else if (sg == 1) { bid(e, q, stamp, state, lock); bad = true; }
          else state[e] = 0;
        }
      }
      const unsigned m = __ballot_sync(0xFFFFFFFFu, bad), mx = __ballot_sync(0xFFFFFFFFu, exact);
      if (lane == 0 && m) atomicAdd(&st->n_bad[p], (unsigned long long)__popc(m));
      if (lane == 0 && mx) atomicAdd(&st->n_exact, (unsigned long long)__popc(mx));
    }
    grid.sync();
    if (*(volatile int *)&st->abort) break;                        // (uniform: read after the barrier, written only before it)
    if (*(volatile unsigned long long *)&st->n_bad[p] == 0) { converged = true; ++it; break; }   // (this iteration counts: it found every edge locally Delaunay)
    if (gtid == 0) { st->n_bad[p ^ 1] = 0; st->n_next[p ^ 1] = 0; }   // for the next iteration; nobody reads them before the next barrier
    // ---- flip
    for (int64_t base = 0; base < n; base += total) {
      const int64_t i = base + gtid;
      int32_t items[4];
      int cnt = 0;
      bool flipped = false;
      const int32_t e = i < n ? cur[i] : -1;
      if (e >= 0 && state[e] == 1) {
        const int32_t t1 = et[2 * (int64_t)e], t2 = et[2 * (int64_t)e + 1];
        const unsigned long long mine = stamp | (unsigned)e;
        if (lock[t1] != mine || lock[t2] != mine) {
          if (atomicExch(mark + e, iter) != iter) items[cnt++] = e;
        } else {
          int32_t *v1 = tv + 3 * (int64_t)t1, *v2 = tv + 3 * (int64_t)t2, *e1 = te + 3 * (int64_t)t1, *e2 = te + 3 * (int64_t)t2;
          const int i1 = e1[0] == e ? 0 : (e1[1] == e ? 1 : 2), i2 = e2[0] == e ? 0 : (e2[1] == e ? 1 : 2);
          const int32_t a = v1[i1], b = v1[(i1 + 1) % 3], cc = v1[(i1 + 2) % 3], d = v2[i2];
          const int32_t e_ca = e1[(i1 + 1) % 3], e_ab = e1[(i1 + 2) % 3], e_bd = e2[(i2 + 1) % 3], e_dc = e2[(i2 + 2) % 3];
          v1[0] = a; v1[1] = b; v1[2] = d;
          e1[0] = e_bd; e1[1] = e; e1[2] = e_ab;
          v2[0] = a; v2[1] = d; v2[2] = cc;
          e2[0] = e_dc; e2[1] = e_ca; e2[2] = e;
          int32_t *f = et + 2 * (int64_t)e_bd;
          f[f[0] == t2 ? 0 : 1] = t1;
          f = et + 2 * (int64_t)e_ca;
          f[f[0] == t1 ? 0 : 1] = t2;
          state[e] = 0;
          touch.tri(t1);
          touch.tri(t2);
          touch.edge(e);
          const int32_t outer[4] = {e_ca, e_ab, e_bd, e_dc};
#pragma unroll
          for (int j = 0; j < 4; ++j)
            if (atomicExch(mark + outer[j], iter) != iter) items[cnt++] = outer[j];
          flipped = true;
        }
      }
      int incl = cnt;
#pragma unroll
      for (int dlt = 1; dlt < 32; dlt <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, dlt);
        if (lane >= dlt) incl += v;
      }
      const int tot = __shfl_sync(0xFFFFFFFFu, incl, 31);
      unsigned long long bs = 0;
      if (lane == 31 && tot) bs = atomicAdd(&st->n_next[p], (unsigned long long)tot);
      bs = __shfl_sync(0xFFFFFFFFu, bs, 31);
      for (int j = 0; j < cnt; ++j) nxt[bs + incl - cnt + j] = items[j];
      const unsigned fm = __ballot_sync(0xFFFFFFFFu, flipped);
      if (lane == 0 && fm) atomicAdd(&st->n_flip, (unsigned long long)__popc(fm));
    }
    grid.sync();
    n = (int64_t)*(volatile unsigned long long *)&st->n_next[p];
  }
  if (gtid == 0) {
    st->done_iters = it;
    st->converged = converged ? 1 : 0;
    st->n_cur = (unsigned long long)n;
  }
}

// input check of the triangulator and the refinement: every triangle counter-clockwise (exact ORIENT2D > 0), vertex numbers in range
__global__ void __launch_bounds__(256)
validate_kernel(int64_t nt, int64_t nv, const double2 *__restrict__ xy, const int32_t *__restrict__ tv, unsigned long long *__restrict__ n_bad) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (t < nt) {
    const int32_t a = tv[3 * t], b = tv[3 * t + 1], c = tv[3 * t + 2];
    bad = a < 0 || b < 0 || c < 0 || a >= nv || b >= nv || c >= nv || a == b || b == c || a == c;
    if (!bad) bad = orient2d_sign(xy[a], xy[b], xy[c]) <= 0;
  }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_bad, (unsigned long long)__popc(m));
}

// the edge tables describe a triangulation: every edge is listed by the triangle(s) edgeTriangles names for it, at the local
// place opposite the vertex that is not on it, and its two triangles run along it in opposite directions (two counter-clockwise
// triangles that run along a shared edge in the same direction lie on the same side of it: they overlap)
__global__ void __launch_bounds__(256)
validate_edges_kernel(int64_t ne, int64_t nt, const int32_t *__restrict__ tv, const int32_t *__restrict__ te, const int32_t *__restrict__ et,
                      unsigned long long *__restrict__ n_bad) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (e < ne) {
    const int32_t t1 = et[2 * e], t2 = et[2 * e + 1];
    bad = t1 < 0 || t1 >= nt || t2 >= nt || t1 == t2;
    if (!bad) {
      const int32_t *E1 = te + 3 * (int64_t)t1, *V1 = tv + 3 * (int64_t)t1;
      const int k1 = E1[0] == e ? 0 : E1[1] == e ? 1 : E1[2] == e ? 2 : -1;
      bad = k1 < 0;
      if (!bad && t2 >= 0) {
        const int32_t *E2 = te + 3 * (int64_t)t2, *V2 = tv + 3 * (int64_t)t2;
        const int k2 = E2[0] == e ? 0 : E2[1] == e ? 1 : E2[2] == e ? 2 : -1;
        bad = k2 < 0 || V1[(k1 + 1) % 3] != V2[(k2 + 2) % 3] || V1[(k1 + 2) % 3] != V2[(k2 + 1) % 3];
      }
    }
  }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_bad, (unsigned long long)__popc(m));
}
// every triangle's three edges exist and name the triangle
__global__ void __launch_bounds__(256)
validate_sides_kernel(int64_t nt, int64_t ne, const int32_t *__restrict__ te, const int32_t *__restrict__ et, unsigned long long *__restrict__ n_bad) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool bad = false;
  if (t < nt)
    for (int k = 0; k < 3; ++k) {
      const int32_t e = te[3 * t + k];
      bad |= e < 0 || e >= ne || (et[2 * (int64_t)e] != t && et[2 * (int64_t)e + 1] != t);
    }
  const unsigned m = __ballot_sync(0xFFFFFFFFu, bad);
  if ((threadIdx.x & 31) == 0 && m) atomicAdd(n_bad, (unsigned long long)__popc(m));
}

// ------------------------------------------------------------------------------------------------------------------
// Point location (section 2.4.2)
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
find_triangle_kernel(int64_t np, const double2 *__restrict__ p, const int32_t *__restrict__ t0, int64_t max_steps,
                     const double2 *__restrict__ xy, const int32_t *__restrict__ tv, const int32_t *__restrict__ te,
                     const int32_t *__restrict__ et, int32_t *__restrict__ t_out, int8_t *__restrict__ code_out, int *__restrict__ err) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= np) return;
  const double2 P = p[i];
  int32_t t = t0[i];
  for (int64_t step = 0; step < max_steps; ++step) {
    const int32_t *v = tv + 3 * (int64_t)t;
    const double2 A = xy[v[0]], B = xy[v[1]], C = xy[v[2]];
    // the edge (a, b) is opposite local vertex 2, (b, c) opposite 0, (c, a) opposite 1; cross the first with p strictly outside
    int s[3];
    int out = -1;
    s[0] = orient2d_sign(A, B, P);
    if (s[0] < 0) out = 2;
    else {
      s[1] = orient2d_sign(B, C, P);
      if (s[1] < 0) out = 0;
      else {
        s[2] = orient2d_sign(C, A, P);
        if (s[2] < 0) out = 1;
      }
    }
    if (out < 0) {
      const int z0 = s[0] == 0, z1 = s[1] == 0, z2 = s[2] == 0;
      int code = 0;
      if (z0 + z1 + z2 == 1) code = 1 + (z0 ? 2 : (z1 ? 0 : 1));
      else if (z0 + z1 + z2 >= 2) code = 4 + ((z0 && z1) ? 1 : ((z1 && z2) ? 2 : 0));   // the vertex the two edges share
      t_out[i] = t;
      code_out[i] = (int8_t)code;
      return;
    }
    const int32_t e = te[3 * (int64_t)t + out];
    const int32_t n0 = et[2 * (int64_t)e], n1 = et[2 * (int64_t)e + 1];
    const int32_t nxt = n0 != t ? n0 : n1;
    if (nxt < 0) {
      t_out[i] = -1 - t;
      code_out[i] = 0;
      return;
    }
    t = nxt;
  }
  *err = 1;
}

// ------------------------------------------------------------------------------------------------------------------
// Delaunay refinement (section 2.4) with the parallel insertion set of section 4.1.1
// ------------------------------------------------------------------------------------------------------------------
constexpr int CAVITY_MAX = 64;   // reading M11
enum { KIND_NONE = 0, KIND_TRI = 1, KIND_EDGE = 2, KIND_SEG = 3 };

// i(v) of L648 (reading M10): 32-bit mix of (seed, iteration, bad triangle) above the bad triangle's number
static __device__ __forceinline__ unsigned long long priority_of(unsigned seed, unsigned iteration, unsigned t) {
  if (seed == 0xFFFFFFFFu) return ((unsigned long long)t << 32) | t;   // MRD_MESHGEN_PRIORITY_REGULAR: i(v_n) = n (L654, Fig. 8)
  unsigned x = t * 2654435761u + iteration * 40503u + seed;
  x ^= x >> 15;
  x *= 2246822519u;
  x ^= x >> 13;
  x *= 3266489917u;
  x ^= x >> 16;
  return ((unsigned long long)x << 32) | t;
}
static __device__ __forceinline__ int local_of(const int32_t *row, int32_t x) { return row[0] == x ? 0 : (row[1] == x ? 1 : 2); }
static __device__ __forceinline__ int32_t across(const int32_t *et, int32_t e, int32_t t) {
  const int32_t n0 = et[2 * (int64_t)e], n1 = et[2 * (int64_t)e + 1];
  return n0 != t ? n0 : n1;
}
// eq. 4 (L172), one IEEE operation at a time
static __device__ __forceinline__ bool encroaches(double2 u, double2 w, double2 p) {
  const double ux = __dsub_rn(u.x, p.x), uy = __dsub_rn(u.y, p.y), wx = __dsub_rn(w.x, p.x), wy = __dsub_rn(w.y, p.y);
  return __dadd_rn(__dmul_rn(ux, wx), __dmul_rn(uy, wy)) < 0.0;
}
// the segments of triangle t that p encroaches upon: lowest edge number so far in (best_e, best_t)
static __device__ __forceinline__ void test_segments(int32_t t, double2 p, const double2 *xy, const int32_t *tv, const int32_t *te,
                                                     const int32_t *et, int32_t &best_e, int32_t &best_t) {
  const int32_t *v = tv + 3 * (int64_t)t, *ed = te + 3 * (int64_t)t;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const int32_t e = ed[k];
    if (et[2 * (int64_t)e + 1] < 0 && (best_e < 0 || e < best_e) && encroaches(xy[v[(k + 1) % 3]], xy[v[(k + 2) % 3]], p)) {
      best_e = e;
      best_t = t;
    }
  }
}
// all triangles that have x as a vertex (L176), starting from t: around x one way until back at t or at the boundary, then
// the other way
static __device__ void around_vertex(int32_t x, int32_t t, double2 p, const double2 *xy, const int32_t *tv, const int32_t *te,
                                     const int32_t *et, int32_t &best_e, int32_t &best_t) {
  test_segments(t, p, xy, tv, te, et, best_e, best_t);
  for (int dir = 1; dir <= 2; ++dir) {
    int32_t cur = t;
    for (int guard = 0; guard < 4096; ++guard) {
      const int k = local_of(tv + 3 * (int64_t)cur, x);
      const int32_t nxt = across(et, te[3 * (int64_t)cur + (k + dir) % 3], cur);   // both edges opposite k+1 and k+2 contain x
      if (nxt < 0) break;
      if (nxt == t) return;                                        // closed fan: everything seen
      test_segments(nxt, p, xy, tv, te, et, best_e, best_t);
      cur = nxt;
    }
  }
}
static __device__ __forceinline__ double2 midpoint(double2 u, double2 w) {
  return make_double2(__dmul_rn(0.5, __dadd_rn(u.x, w.x)), __dmul_rn(0.5, __dadd_rn(u.y, w.y)));
}
// near[v] = 1 when a triangle that has v as a vertex has a segment for an edge: only around such vertices can the rotation of
// around_vertex meet a segment, so the encroachment test of all other vertices is skipped (same result, most candidates are
// far from every segment)
__global__ void __launch_bounds__(256)
near_segment_kernel(int64_t ne, const int32_t *__restrict__ et, const int32_t *__restrict__ tv, uint8_t *__restrict__ near) {
  const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= ne || et[2 * e + 1] >= 0) return;
  const int32_t *v = tv + 3 * (int64_t)et[2 * e];
  near[v[0]] = 1; near[v[1]] = 1; near[v[2]] = 1;
}
// sections 2.4.2-2.4.3 for the circumcentre of every bad triangle (oracle/meshgen.py: candidate)
__global__ void __launch_bounds__(128)
candidate_kernel(int64_t nc, const int32_t *__restrict__ cand, const double2 *__restrict__ cc, int64_t max_steps,
                 const double2 *__restrict__ xy, const int32_t *__restrict__ tv, const int32_t *__restrict__ te,
                 const int32_t *__restrict__ et, int8_t *__restrict__ kind, double2 *__restrict__ pt, int32_t *__restrict__ t_ins,
                 int32_t *__restrict__ e_ins, int *__restrict__ err, const uint8_t *__restrict__ near) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nc) return;
  const int32_t tb = cand[j];
  const double2 P = cc[tb];
  int32_t t = tb;
  int code = -1, out = -1;
  for (int64_t step = 0; step < max_steps; ++step) {               // the walk of find_triangle_kernel, keeping the exit edge
    const int32_t *v = tv + 3 * (int64_t)t;
    const double2 A = xy[v[0]], B = xy[v[1]], C = xy[v[2]];
    int s0, s1 = 1, s2 = 1;
    out = -1;
    s0 = orient2d_sign(A, B, P);
    if (s0 < 0) out = 2;
    else {
      s1 = orient2d_sign(B, C, P);
      if (s1 < 0) out = 0;
      else {
        s2 = orient2d_sign(C, A, P);
        if (s2 < 0) out = 1;
      }
    }
    if (out < 0) {
      const int z0 = s0 == 0, z1 = s1 == 0, z2 = s2 == 0;
      code = 0;
      if (z0 + z1 + z2 == 1) code = 1 + (z0 ? 2 : (z1 ? 0 : 1));
      else if (z0 + z1 + z2 >= 2) code = 4;
      break;
    }
    const int32_t nxt = across(et, te[3 * (int64_t)t + out], t);
    if (nxt < 0) break;                                            // left the triangulation through edge `out` of t
    t = nxt;
    out = -1;
  }
  int8_t kd = KIND_NONE;
  double2 p = P;
  int32_t ti = t, ei = -1;
  if (code < 0 && out < 0) { *err = 1; return; }                    // the walk did not end
  if (code < 0) {                                                  // outside: split the segment it left through (M8)
    ei = te[3 * (int64_t)t + out];
    const int32_t *v = tv + 3 * (int64_t)t;
    p = midpoint(xy[v[(out + 1) % 3]], xy[v[(out + 2) % 3]]);
    kd = KIND_SEG;
  } else if (code >= 4) {
    kd = KIND_NONE;
  } else {
    int32_t t2 = -1;
    if (code >= 1) {
      ei = te[3 * (int64_t)t + code - 1];
      if (et[2 * (int64_t)ei + 1] < 0) {                           // on a segment: split it
        const int32_t *v = tv + 3 * (int64_t)t;
        p = midpoint(xy[v[code % 3]], xy[v[(code + 1) % 3]]);
        kd = KIND_SEG;
      } else {
        kd = KIND_EDGE;
        ti = et[2 * (int64_t)ei];
        t2 = et[2 * (int64_t)ei + 1];
      }
    } else kd = KIND_TRI;
    if (kd != KIND_SEG) {                                          // eq. 4 around every vertex of the insertion triangle(s)
      int32_t best_e = -1, best_t = -1;
      const int32_t *v = tv + 3 * (int64_t)ti;
      for (int k = 0; k < 3; ++k)
        if (near[v[k]]) around_vertex(v[k], ti, P, xy, tv, te, et, best_e, best_t);
      if (t2 >= 0) {
        const int32_t x4 = tv[3 * (int64_t)t2 + local_of(te + 3 * (int64_t)t2, ei)];                    // the fourth vertex
        if (near[x4]) around_vertex(x4, t2, P, xy, tv, te, et, best_e, best_t);
      }
      if (best_e >= 0) {
        const int k = local_of(te + 3 * (int64_t)best_t, best_e);
        const int32_t *u = tv + 3 * (int64_t)best_t;
        p = midpoint(xy[u[(k + 1) % 3]], xy[u[(k + 2) % 3]]);
        kd = KIND_SEG;
        ti = best_t;
        ei = best_e;
      }
    }
  }
  kind[j] = kd;
  pt[j] = p;
  t_ins[j] = ti;
  e_ins[j] = ei;
}

// section 4.1.1: the cavity of p from its insertion triangle(s); returns its size, -1 when it exceeds CAVITY_MAX, and -2 when
// EXACT is false and the filter could not decide one of the INCIRCLE2D tests (the candidate then goes to the exact kernel)
template <bool EXACT>
static __device__ int cavity_of(double2 p, int8_t kd, int32_t ti, int32_t ei, const double2 *xy, const int32_t *tv, const int32_t *te,
                                const int32_t *et, int32_t *list, double *acc, double *tmp) {
  int n = 0;
  if (kd == KIND_EDGE) { list[n++] = et[2 * (int64_t)ei]; list[n++] = et[2 * (int64_t)ei + 1]; }
  else list[n++] = ti;
  for (int head = 0; head < n; ++head) {
    const int32_t t = list[head];
    for (int k = 0; k < 3; ++k) {
      const int32_t nb = across(et, te[3 * (int64_t)t + k], t);
      if (nb < 0) continue;
      bool seen = false;
      for (int q = 0; q < n; ++q) seen |= list[q] == nb;
      if (seen) continue;
      const int32_t *v = tv + 3 * (int64_t)nb;
      const double2 A = xy[v[0]], B = xy[v[1]], C = xy[v[2]];
      int sg = incircle2d_filter(A, B, C, p);
      if (sg == 2) sg = incircle2d_exact_short(A, B, C, p);       // exact translations (neighbouring points): short expansions
      if (sg == 2) {
        if (!EXACT) return -2;
        sg = incircle2d_exact(A, B, C, p, acc, tmp);
      }
      if (sg > 0) {
        if (n == CAVITY_MAX) return -1;
        list[n++] = nb;
      }
    }
  }
  return n;
}
// Reading M11: a cavity that does not fit the per-thread list is walked without a list.  The cavity of a point in a Delaunay
// triangulation has no vertex inside it (the fan from the new vertex over its rim IS the new triangulation), so under "shares an
// edge" its triangles form a tree, and the walk follows the outline of that tree (L640-L646: "by always checking the neighbours
// in anti-clockwise order"): arrived in t through its local edge k it tries k+1 and k+2 and then leaves through k again; the
// root tries its edges 0, 1, 2 once.  A triangle is tested again when the walk comes back to it from a child -- the actions are
// idempotent.  PASS 1 claims every triangle on arrival, PASS 2 compares every one.  Returns 1 (PASS 2: 0 when a triangle
// carries another priority), -2 when EXACT is false and the filter cannot decide a test, -1 when the walk does not close within
// 4 nt + 16 moves (the input was not a Delaunay triangulation): the candidate waits.
template <int PASS, bool EXACT>
static __device__ int cavity_walk(double2 p, int8_t kd, int32_t ti, int32_t ei, const double2 *xy, const int32_t *tv, const int32_t *te,
                                  const int32_t *et, int64_t nt, unsigned long long pr, unsigned long long *claim, double *acc,
                                  double *tmp) {
  const int32_t root = kd == KIND_EDGE ? et[2 * (int64_t)ei] : ti;
  const int32_t root2 = kd == KIND_EDGE ? et[2 * (int64_t)ei + 1] : -1;
  if (PASS == 1) atomicMax(claim + root, pr);
  else if (claim[root] != pr) return 0;
  int32_t t = root;
  int k = -1;                                                     // root: the last of its edges that was tried
  for (int64_t moves = 0; moves < 4 * nt + 16; ++moves) {
    int go = -1;
    const bool at_root = t == root;
    for (int d = 1; d <= (at_root ? 2 - k : 2) && go < 0; ++d) {
      const int q = at_root ? k + d : (k + d) % 3;
      const int32_t nb = across(et, te[3 * (int64_t)t + q], t);
      if (nb < 0) continue;
      int sg = 1;
      if (nb != root && nb != root2) {
        const int32_t *v = tv + 3 * (int64_t)nb;
        const double2 A = xy[v[0]], B = xy[v[1]], C = xy[v[2]];
        sg = incircle2d_filter(A, B, C, p);
        if (sg == 2) sg = incircle2d_exact_short(A, B, C, p);
        if (sg == 2) {
          if (!EXACT) return -2;
          sg = incircle2d_exact(A, B, C, p, acc, tmp);
        }
      }
      if (sg > 0) go = q;
    }
    if (go < 0) {
      if (at_root) return 1;                                      // the outline is closed
      go = k;                                                     // back to where this triangle was entered from
    }
    const int32_t e = te[3 * (int64_t)t + go];
    const int32_t nb = across(et, e, t);
    if (PASS == 1) atomicMax(claim + nb, pr);
    else if (claim[nb] != pr) return 0;
    k = local_of(te + 3 * (int64_t)nb, e);
    t = nb;
  }
  return -1;
}
// pass 1: claim the cavity's triangles; pass 2: selected when every one of them still carries this candidate's priority.
// n > 0: the cavity is in `list`; n == -1: it did not fit (cavity_walk); n == -3: nothing to insert
template <int PASS, bool EXACT>
static __device__ __forceinline__ void cavity_act(int64_t j, int n, const int32_t *list, int8_t kd, unsigned long long pr, int8_t *kind,
                                                  unsigned long long *claim, int32_t *sel, int32_t *seg, const double2 *pt,
                                                  const int32_t *t_ins, const int32_t *e_ins, const double2 *xy, const int32_t *tv,
                                                  const int32_t *te, const int32_t *et, int64_t nt, double *acc, double *tmp,
                                                  int32_t *work, unsigned long long *n_work) {
  if (PASS == 1) {
    if (n == -1) {
      const int r = cavity_walk<1, EXACT>(pt[j], kd, t_ins[j], e_ins[j], xy, tv, te, et, nt, pr, claim, acc, tmp);
      if (r == -2) work[atomicAdd(n_work, 1ull)] = (int32_t)j;     // only when EXACT is false: the exact kernel walks it again
      else if (r < 0) kind[j] = KIND_NONE;
      return;
    }
    if (n < 0) kind[j] = KIND_NONE;                                // nothing to insert: waits
    for (int q = 0; q < n; ++q) atomicMax(claim + list[q], pr);
  } else {
    bool mine = n > 0;
    for (int q = 0; q < n; ++q) mine &= claim[list[q]] == pr;
    if (n == -1) {
      const int r = cavity_walk<2, EXACT>(pt[j], kd, t_ins[j], e_ins[j], xy, tv, te, et, nt, pr, claim, acc, tmp);
      if (r == -2) return;                                         // in the work list of pass 1: the exact kernel decides
      mine = r == 1;
    }
    sel[j] = mine ? 1 : 0;
    seg[j] = (mine && kd == KIND_SEG) ? 1 : 0;
  }
}
// one thread per candidate, filter and short exact evaluation only; the candidates with a test that needs the long expansions
// are listed for cavity_exact_kernel.  Pass 1 keeps the cavities it finds in a pool (one atomic per warp reserves the room;
// off[j] = -1 when the pool is full), pass 2 reads them back instead of walking the mesh again.
template <int PASS>
__global__ void __launch_bounds__(128)
cavity_kernel(int64_t nc, const int32_t *__restrict__ cand, int8_t *__restrict__ kind, const double2 *__restrict__ pt,
              const int32_t *__restrict__ t_ins, const int32_t *__restrict__ e_ins, const double2 *__restrict__ xy,
              const int32_t *__restrict__ tv, const int32_t *__restrict__ te, const int32_t *__restrict__ et,
              unsigned long long *__restrict__ claim, unsigned seed, unsigned iteration, int32_t *__restrict__ sel,
              int32_t *__restrict__ seg, int32_t *__restrict__ work, unsigned long long *__restrict__ n_work,
              int32_t *__restrict__ pool, unsigned long long *__restrict__ pool_n, int64_t pool_cap, int32_t *__restrict__ off,
              int64_t nt) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = j < nc;
  int32_t list[CAVITY_MAX];
  const int8_t kd = live ? kind[j] : (int8_t)KIND_NONE;
  int n = -3;
  if (PASS == 2 && live && off[j] >= 0) {                         // found in pass 1
    const int32_t *src = pool + off[j];
    n = src[0];
    for (int q = 0; q < n; ++q) list[q] = src[1 + q];
  } else if (live && kd != KIND_NONE) {
    n = cavity_of<false>(pt[j], kd, t_ins[j], e_ins[j], xy, tv, te, et, list, nullptr, nullptr);
  }
  if (PASS == 1) {
    // room in the pool: 1 + n entries for every cavity found here, reserved once per warp
    const int want = (live && n > 0) ? n + 1 : 0;
    const int lane = threadIdx.x & 31;
    int incl = want;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
      if (lane >= d) incl += v;
    }
    const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    unsigned long long base = 0;
    if (lane == 31 && total) base = atomicAdd(pool_n, (unsigned long long)total);
    base = __shfl_sync(0xFFFFFFFFu, base, 31);
    if (live) {
      int32_t o = -1;
      if (want && (int64_t)(base + incl) <= pool_cap) {
        o = (int32_t)(base + incl - want);
        pool[o] = n;
        for (int q = 0; q < n; ++q) pool[o + 1 + q] = list[q];
      }
      off[j] = o;
    }
  }
  if (!live) return;
  if (n == -2) {                                                  // undecided: pass 1 lists it, pass 2 finds it in that list
    if (PASS == 1) work[atomicAdd(n_work, 1ull)] = (int32_t)j;
    return;
  }
  cavity_act<PASS, false>(j, n, list, kd, priority_of(seed, iteration, (unsigned)cand[j]), kind, claim, sel, seg, pt, t_ins, e_ins, xy,
                          tv, te, et, nt, nullptr, nullptr, work, n_work);
}
// the listed candidates again, with the exact INCIRCLE2D where the filter fails.  Grid-stride with few threads: every thread
// owns a slice of the expansion scratch.  One exact evaluation is a serial chain of ~10^4 operations on expansions in global
// memory (~100 us), so pass 1 keeps the cavities it found (the first CAVITY_STORE work items) and pass 2 reads them back
// instead of finding them again: both passes walk the work list of pass 1.
constexpr int CAVITY_STORE = 1 << 15;
template <int PASS>
__global__ void __launch_bounds__(32)
cavity_exact_kernel(const unsigned long long *__restrict__ n_work, const int32_t *__restrict__ work, const int32_t *__restrict__ cand,
                    int8_t *__restrict__ kind, const double2 *__restrict__ pt, const int32_t *__restrict__ t_ins,
                    const int32_t *__restrict__ e_ins, const double2 *__restrict__ xy, const int32_t *__restrict__ tv,
                    const int32_t *__restrict__ te, const int32_t *__restrict__ et, unsigned long long *__restrict__ claim, unsigned seed,
                    unsigned iteration, int32_t *__restrict__ sel, int32_t *__restrict__ seg, double *__restrict__ scratch,
                    int32_t *__restrict__ store, int64_t nt) {
  const int64_t tid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x, nw = (int64_t)*n_work;
  double *acc = scratch + tid * (2 * MAXE), *tmp = acc + MAXE;
  int32_t list[CAVITY_MAX];
  for (int64_t w = tid; w < nw; w += (int64_t)gridDim.x * blockDim.x) {
    const int64_t j = work[w];
    const int8_t kd = kind[j];
    int32_t *st = store + w * (CAVITY_MAX + 1);
    int n;
    if (PASS == 2 && w < CAVITY_STORE) {
      n = st[0];
      for (int q = 0; q < n; ++q) list[q] = st[1 + q];
    } else {
      n = kd == KIND_NONE ? -3 : cavity_of<true>(pt[j], kd, t_ins[j], e_ins[j], xy, tv, te, et, list, acc, tmp);
      if (PASS == 1 && w < CAVITY_STORE) {
        st[0] = n;
        for (int q = 0; q < n; ++q) st[1 + q] = list[q];
      }
    }
    cavity_act<PASS, true>(j, n, list, kd, priority_of(seed, iteration, (unsigned)cand[j]), kind, claim, sel, seg, pt, t_ins, e_ins, xy, tv,
                           te, et, nt, acc, tmp, nullptr, nullptr);
  }
}
static __device__ __forceinline__ void swap_side(int32_t *et, int32_t e, int32_t from, int32_t to) {
  int32_t *f = et + 2 * (int64_t)e;
  f[f[0] == from ? 0 : 1] = to;
}
static __device__ __forceinline__ void put3(int32_t *row, int32_t a, int32_t b, int32_t c) { row[0] = a; row[1] = b; row[2] = c; }
// section 2.4.4 for every selected candidate (oracle/meshgen.py: insert_vertex); rank / segrank: exclusive sums of sel / seg
__global__ void __launch_bounds__(128)
insert_kernel(int64_t nc, const int8_t *__restrict__ kind, const double2 *__restrict__ pt, const int32_t *__restrict__ t_ins,
              const int32_t *__restrict__ e_ins, const int32_t *__restrict__ sel, const int32_t *__restrict__ rank,
              const int32_t *__restrict__ segrank, int32_t nv, int32_t nt, int32_t ne, double2 *__restrict__ xy,
              int32_t *__restrict__ tv, int32_t *__restrict__ te, int32_t *__restrict__ et, Touch touch) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= nc || !sel[j]) return;
  const int32_t v = nv + rank[j];
  const int32_t tn = nt + 2 * rank[j] - segrank[j], en = ne + 3 * rank[j] - segrank[j];   // SEG adds 1 / 2, the others 2 / 3
  xy[v] = pt[j];
  Touch::Pending pend;
  pend.n = 0;
  const int32_t t = t_ins[j], e = e_ins[j];
  int32_t *V = tv + 3 * (int64_t)t, *E = te + 3 * (int64_t)t;
  if (kind[j] == KIND_TRI) {
    const int32_t a = V[0], b = V[1], c = V[2], e0 = E[0], e1 = E[1], e2 = E[2];
    const int32_t t1 = tn, t2 = tn + 1, f0 = en, f1 = en + 1, f2 = en + 2;      // f0 = (v, a), f1 = (v, b), f2 = (v, c)
    put3(V, a, b, v); put3(E, f1, f0, e2);
    put3(tv + 3 * (int64_t)t1, b, c, v); put3(te + 3 * (int64_t)t1, f2, f1, e0);
    put3(tv + 3 * (int64_t)t2, c, a, v); put3(te + 3 * (int64_t)t2, f0, f2, e1);
    et[2 * (int64_t)f0] = t; et[2 * (int64_t)f0 + 1] = t2;
    et[2 * (int64_t)f1] = t; et[2 * (int64_t)f1 + 1] = t1;
    et[2 * (int64_t)f2] = t1; et[2 * (int64_t)f2 + 1] = t2;
    swap_side(et, e0, t, t1);
    swap_side(et, e1, t, t2);
    touch.tri(t); touch.tri(t1); touch.tri(t2);
    touch.edge(f0); touch.edge(f1); touch.edge(f2);
    touch.check(e0, pend); touch.check(e1, pend); touch.check(e2, pend); touch.check(f0, pend); touch.check(f1, pend); touch.check(f2, pend);
    touch.flush(pend);
    return;
  }
  const int i1 = local_of(E, e);
  const int32_t a = V[i1], b = V[(i1 + 1) % 3], c = V[(i1 + 2) % 3];           // E = (b, c), a opposite
  const int32_t e_ca = E[(i1 + 1) % 3], e_ab = E[(i1 + 2) % 3];
  if (kind[j] == KIND_SEG) {
    const int32_t n1 = tn, g0 = en, g1 = en + 1;                               // E becomes (b, v); g0 = (v, c); g1 = (a, v)
    put3(V, a, b, v); put3(E, e, g1, e_ab);
    put3(tv + 3 * (int64_t)n1, a, v, c); put3(te + 3 * (int64_t)n1, g0, e_ca, g1);
    et[2 * (int64_t)g0] = n1; et[2 * (int64_t)g0 + 1] = -1;
    et[2 * (int64_t)g1] = t; et[2 * (int64_t)g1 + 1] = n1;
    swap_side(et, e_ca, t, n1);
    touch.tri(t); touch.tri(n1);
    touch.edge(e); touch.edge(g0); touch.edge(g1);               // E = (b, c) is (b, v) now
    touch.check(e, pend); touch.check(g0, pend); touch.check(g1, pend); touch.check(e_ca, pend); touch.check(e_ab, pend);
    touch.flush(pend);
    return;
  }
  const int32_t t2 = across(et, e, t);
  int32_t *V2 = tv + 3 * (int64_t)t2, *E2 = te + 3 * (int64_t)t2;
  const int i2 = local_of(E2, e);
  const int32_t d = V2[i2], e_bd = E2[(i2 + 1) % 3], e_dc = E2[(i2 + 2) % 3];
  const int32_t n1 = tn, n2 = tn + 1, g0 = en, g1 = en + 1, g2 = en + 2;       // g0 = (v, c), g1 = (a, v), g2 = (v, d)
  put3(V, a, b, v); put3(E, e, g1, e_ab);
  put3(tv + 3 * (int64_t)n1, a, v, c); put3(te + 3 * (int64_t)n1, g0, e_ca, g1);
  put3(V2, d, v, b); put3(E2, e, e_bd, g2);
  put3(tv + 3 * (int64_t)n2, d, c, v); put3(te + 3 * (int64_t)n2, g0, g2, e_dc);
  et[2 * (int64_t)g0] = n1; et[2 * (int64_t)g0 + 1] = n2;
  et[2 * (int64_t)g1] = t; et[2 * (int64_t)g1 + 1] = n1;
  et[2 * (int64_t)g2] = t2; et[2 * (int64_t)g2 + 1] = n2;
  swap_side(et, e_ca, t, n1);
  swap_side(et, e_dc, t2, n2);
  touch.tri(t); touch.tri(n1); touch.tri(t2); touch.tri(n2);
  touch.edge(e); touch.edge(g0); touch.edge(g1); touch.edge(g2);
  touch.check(e, pend); touch.check(g0, pend); touch.check(g1, pend); touch.check(g2, pend);
  touch.check(e_ca, pend); touch.check(e_ab, pend); touch.check(e_bd, pend); touch.check(e_dc, pend);
  touch.flush(pend);
}
// Morton value of every vertex (section 4.1.4; reading M14): 21 bits per coordinate, x in the even places
static __device__ __forceinline__ unsigned long long spread21(unsigned v) {
  unsigned long long x = v & 0x1FFFFFull;
  x = (x | (x << 16)) & 0x0000FFFF0000FFFFull;
  x = (x | (x << 8)) & 0x00FF00FF00FF00FFull;
  x = (x | (x << 4)) & 0x0F0F0F0F0F0F0F0Full;
  x = (x | (x << 2)) & 0x3333333333333333ull;
  x = (x | (x << 1)) & 0x5555555555555555ull;
  return x;
}
__global__ void __launch_bounds__(256)
morton_keys_kernel(int64_t nv, const double2 *__restrict__ xy, double x0, double y0, double sx, double sy,
                   unsigned long long *__restrict__ key, int32_t *__restrict__ idx) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  const double2 p = xy[i];
  const double fx = floor(__dmul_rn(__dsub_rn(p.x, x0), sx)), fy = floor(__dmul_rn(__dsub_rn(p.y, y0), sy));
  const unsigned ix = (unsigned)fmin(2097151.0, fmax(0.0, fx)), iy = (unsigned)fmin(2097151.0, fmax(0.0, fy));
  key[i] = spread21(ix) | (spread21(iy) << 1);
  idx[i] = (int32_t)i;
}
// order[i] = old number of the vertex that becomes i
__global__ void __launch_bounds__(256)
vertex_permute_kernel(int64_t nv, const int32_t *__restrict__ order, const double2 *__restrict__ xy, double2 *__restrict__ xy_new,
                      int32_t *__restrict__ number) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  const int32_t o = order[i];
  xy_new[i] = xy[o];
  number[o] = (int32_t)i;
}
__global__ void __launch_bounds__(256)
relabel_kernel(int64_t n, const int32_t *__restrict__ number, int32_t *__restrict__ tv) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) tv[i] = number[tv[i]];
}
// ---- in-place renumbering (reading M15; oracle/meshgen.py: renumber_in_place) ---------------------------------------------
// S: the touched triangle slots in ascending order.  Rotate their rows (tv and te together) to the smallest vertex; sort keys.
__global__ void __launch_bounds__(256)
touched_keys_kernel(int64_t ns, const int32_t *__restrict__ S, int32_t *__restrict__ tv, int32_t *__restrict__ te, int bits,
                    unsigned long long *__restrict__ key_lo, int32_t *__restrict__ idx) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ns) return;
  int32_t *v = tv + 3 * (int64_t)S[i], *ed = te + 3 * (int64_t)S[i];
  const int32_t a = v[0], b = v[1], c = v[2], ea = ed[0], eb = ed[1], ec = ed[2];
  const int r = (a < b && a < c) ? 0 : ((b < a && b < c) ? 1 : 2);
  const int32_t x = r == 0 ? a : (r == 1 ? b : c), y = r == 0 ? b : (r == 1 ? c : a), z = r == 0 ? c : (r == 1 ? a : b);
  put3(v, x, y, z);
  put3(ed, r == 0 ? ea : (r == 1 ? eb : ec), r == 0 ? eb : (r == 1 ? ec : ea), r == 0 ? ec : (r == 1 ? ea : eb));
  key_lo[i] = ((unsigned long long)(unsigned)y << bits) | (unsigned)z;
  idx[i] = (int32_t)i;
}
// small touched sets: the whole triple as ONE key for a merge sort (a handful of launches instead of two radix sorts)
struct TriKey { int32_t a, b, c; };
struct TriKeyLess {
  __device__ __forceinline__ bool operator()(const TriKey &x, const TriKey &y) const {
    return x.a != y.a ? x.a < y.a : (x.b != y.b ? x.b < y.b : x.c < y.c);
  }
};
struct U64Less {
  __device__ __forceinline__ bool operator()(unsigned long long x, unsigned long long y) const { return x < y; }
};
__global__ void __launch_bounds__(256)
touched_triples_kernel(int64_t ns, const int32_t *__restrict__ S, int32_t *__restrict__ tv, int32_t *__restrict__ te,
                       TriKey *__restrict__ key, int32_t *__restrict__ idx) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= ns) return;
  int32_t *v = tv + 3 * (int64_t)S[i], *ed = te + 3 * (int64_t)S[i];
  const int32_t a = v[0], b = v[1], c = v[2], ea = ed[0], eb = ed[1], ec = ed[2];
  const int r = (a < b && a < c) ? 0 : ((b < a && b < c) ? 1 : 2);
  const int32_t x = r == 0 ? a : (r == 1 ? b : c), y = r == 0 ? b : (r == 1 ? c : a), z = r == 0 ? c : (r == 1 ? a : b);
  put3(v, x, y, z);
  put3(ed, r == 0 ? ea : (r == 1 ? eb : ec), r == 0 ? eb : (r == 1 ? ec : ea), r == 0 ? ec : (r == 1 ? ea : eb));
  key[i] = TriKey{x, y, z};
  idx[i] = (int32_t)i;
}
__global__ void __launch_bounds__(256)
touched_first_kernel(int64_t ns, const int32_t *__restrict__ S, const int32_t *__restrict__ tv, const int32_t *__restrict__ idx,
                     unsigned *__restrict__ key_hi) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < ns) key_hi[i] = (unsigned)tv[3 * (int64_t)S[idx[i]]];
}
// order[r]: which entry of S holds the r-th smallest triple.  It moves to slot S[r].
__global__ void __launch_bounds__(256)
tri_map_kernel(int64_t ns, const int32_t *__restrict__ S, const int32_t *__restrict__ order, const int32_t *__restrict__ tv,
               const int32_t *__restrict__ te, int32_t *__restrict__ tri_map, int32_t *__restrict__ tmp_tv, int32_t *__restrict__ tmp_te) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= ns) return;
  const int32_t told = S[order[r]];
  tri_map[told] = S[r];
  const int32_t *v = tv + 3 * (int64_t)told, *ed = te + 3 * (int64_t)told;
  put3(tmp_tv + 3 * r, v[0], v[1], v[2]);
  put3(tmp_te + 3 * r, ed[0], ed[1], ed[2]);
}
// SE: the touched edge slots in ascending order; key = (smaller end point, larger end point)
__global__ void __launch_bounds__(256)
touched_edge_keys_kernel(int64_t nse, const int32_t *__restrict__ SE, const int32_t *__restrict__ tv, const int32_t *__restrict__ te,
                         const int32_t *__restrict__ et, int bits, unsigned long long *__restrict__ key, int32_t *__restrict__ idx) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nse) return;
  const int32_t e = SE[i], t = et[2 * (int64_t)e];
  const int k = local_of(te + 3 * (int64_t)t, e);
  const unsigned u = (unsigned)tv[3 * (int64_t)t + (k + 1) % 3], w = (unsigned)tv[3 * (int64_t)t + (k + 2) % 3];
  key[i] = ((unsigned long long)min(u, w) << bits) | max(u, w);
  idx[i] = (int32_t)i;
}
__global__ void __launch_bounds__(256)
edge_map_kernel(int64_t nse, const int32_t *__restrict__ SE, const int32_t *__restrict__ order, const int32_t *__restrict__ et,
                int32_t *__restrict__ edge_map, int2 *__restrict__ tmp_et) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nse) return;
  const int32_t eold = SE[order[r]];
  edge_map[eold] = SE[r];
  tmp_et[r] = make_int2(et[2 * (int64_t)eold], et[2 * (int64_t)eold + 1]);
}
// where, in the pair of an UNTOUCHED edge, a touched triangle is named (read before anything is rewritten)
__global__ void __launch_bounds__(256)
side_pos_kernel(int64_t ns, const int32_t *__restrict__ S, const int32_t *__restrict__ order, const int32_t *__restrict__ tmp_te,
                const uint8_t *__restrict__ touch_e, const int32_t *__restrict__ et, int8_t *__restrict__ jpos) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= 3 * ns) return;
  const int64_t r = q / 3;
  const int32_t eold = tmp_te[q], told = S[order[r]];
  jpos[q] = touch_e[eold] ? (int8_t)-1 : (int8_t)(et[2 * (int64_t)eold] == told ? 0 : 1);
}
// the rows go to their new slots, with the new numbers of the edges and triangles they name
__global__ void __launch_bounds__(256)
renumber_scatter_kernel(int64_t ns, int64_t nse, const int32_t *__restrict__ S, const int32_t *__restrict__ SE,
                        const int32_t *__restrict__ tmp_tv, const int32_t *__restrict__ tmp_te, const int2 *__restrict__ tmp_et,
                        const int8_t *__restrict__ jpos, const uint8_t *__restrict__ touch_e, const int32_t *__restrict__ tri_map,
                        const int32_t *__restrict__ edge_map, int32_t *__restrict__ tv, int32_t *__restrict__ te, int32_t *__restrict__ et) {
  const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (r < ns) {
    const int32_t s = S[r];
    put3(tv + 3 * (int64_t)s, tmp_tv[3 * r], tmp_tv[3 * r + 1], tmp_tv[3 * r + 2]);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int32_t eold = tmp_te[3 * r + k];
      if (touch_e[eold]) te[3 * (int64_t)s + k] = edge_map[eold];
      else {
        te[3 * (int64_t)s + k] = eold;
        et[2 * (int64_t)eold + jpos[3 * r + k]] = s;                // an untouched edge keeps its slot; its neighbour moved
      }
    }
  }
  if (r < nse) {                                                   // a touched edge lies between touched triangles only
    const int2 p = tmp_et[r];
    const int32_t x = tri_map[p.x], y = p.y >= 0 ? tri_map[p.y] : -1;
    *reinterpret_cast<int2 *>(et + 2 * (int64_t)SE[r]) = (y >= 0 && x > y) ? make_int2(y, x) : make_int2(x, y);
  }
}
// neighbours in ascending order (one 8-byte load and store per pair: two threads that meet at an edge write the same value)
__global__ void __launch_bounds__(256)
renumber_order_kernel(int64_t ns, const int32_t *__restrict__ S, const int32_t *__restrict__ te, int32_t *__restrict__ et) {
  const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= 3 * ns) return;
  int2 *pair = reinterpret_cast<int2 *>(et + 2 * (int64_t)te[3 * (int64_t)S[q / 3] + q % 3]);
  const int2 p = *pair;
  if (p.y >= 0 && p.x > p.y) *pair = make_int2(p.y, p.x);
}

// canonical order (reading M12): rotate every triangle to its smallest vertex; sort keys (second, third) and (first)
__global__ void __launch_bounds__(256)
canonical_keys_kernel(int64_t nt, int32_t *__restrict__ tv, int bits, unsigned long long *__restrict__ key_lo, int32_t *__restrict__ idx) {
  const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nt) return;
  int32_t *v = tv + 3 * t;
  const int32_t a = v[0], b = v[1], c = v[2];
  const int r = (a < b && a < c) ? 0 : ((b < a && b < c) ? 1 : 2);
  const int32_t x = r == 0 ? a : (r == 1 ? b : c), y = r == 0 ? b : (r == 1 ? c : a), z = r == 0 ? c : (r == 1 ? a : b);
  v[0] = x; v[1] = y; v[2] = z;
  key_lo[t] = ((unsigned long long)(unsigned)y << bits) | (unsigned)z;
  idx[t] = (int32_t)t;
}
__global__ void __launch_bounds__(256)
gather_first_kernel(int64_t nt, const int32_t *__restrict__ tv, const int32_t *__restrict__ idx, unsigned *__restrict__ key_hi) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nt) key_hi[i] = (unsigned)tv[3 * (int64_t)idx[i]];
}
__global__ void __launch_bounds__(256)
gather_rows_kernel(int64_t nt, const int32_t *__restrict__ src, const int32_t *__restrict__ idx, int32_t *__restrict__ dst) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nt) return;
  const int32_t *s = src + 3 * (int64_t)idx[i];
  dst[3 * i] = s[0]; dst[3 * i + 1] = s[1]; dst[3 * i + 2] = s[2];
}

}  // namespace mrdgen

extern "C" {

// (mrd_last_error lives in mrd_api.cu; this file reports through its hook)
int mrd_internal_set_error(int code, const char *msg);

namespace {
int gen_fail(int code, const std::string &msg) { return mrd_internal_set_error(code, msg.c_str()); }
int cuda_fail(const char *what, cudaError_t e) {
  return gen_fail(e == cudaErrorMemoryAllocation ? MRD_ENOMEM : MRD_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// Work space kept between calls: cudaMalloc / cudaFree of the scratch arrays cost milliseconds, the kernels microseconds.
// One block per process, grown on demand, carved up by every call (which holds the lock until it has synchronised its
// stream); a small pinned host block receives the counters.  mrd_meshgen_release() frees both.
struct Arena {
  std::mutex mu;
  int dev = -1;
  char *base = nullptr;
  size_t cap = 0;
  unsigned long long *pinned = nullptr;   // 16 words
  cudaError_t reserve(size_t bytes) {
    int d = 0;
    cudaError_t e = cudaGetDevice(&d);
    if (e != cudaSuccess) return e;
    if (d != dev || bytes > cap) {
      if (base) cudaFree(base);
      base = nullptr;
      cap = 0;
      dev = d;
      e = cudaMalloc(&base, bytes);
      if (e != cudaSuccess) return e;
      cap = bytes;
    }
    if (!pinned) e = cudaHostAlloc(&pinned, 16 * sizeof(unsigned long long), cudaHostAllocDefault);
    return e;
  }
  void release() {
    if (base) cudaFree(base);
    if (pinned) cudaFreeHost(pinned);
    base = nullptr;
    pinned = nullptr;
    cap = 0;
    dev = -1;
  }
};
Arena g_arena;
struct Carve {   // offsets first (so that one reserve() covers the call), pointers after
  size_t total = 0;
  size_t add(size_t bytes) {
    const size_t o = total;
    total += (bytes + 255) & ~size_t(255);
    return o;
  }
};
constexpr int EXACT_BLOCKS = 148 * 2, EXACT_THREADS = 32;
constexpr size_t EXACT_SCRATCH = sizeof(double) * 2 * mrdgen::MAXE * (size_t)EXACT_BLOCKS * EXACT_THREADS;   // 182 MB
}  // namespace

int mrd_meshgen_release(void) {
  std::lock_guard<std::mutex> g(g_arena.mu);
  g_arena.release();
  return MRD_OK;
}

int mrd_meshgen_test_quality(int64_t n_triangle, const double *xy_dev, const int32_t *tri_dev, double R, double B, double *r_dev,
                             double *beta_dev, double *cc_dev, uint8_t *bad_dev, int64_t *n_bad, void *stream) {
  if (n_triangle < 0 || (n_triangle > 0 && (!xy_dev || !tri_dev || !r_dev || !beta_dev || !cc_dev || !bad_dev)))
    return gen_fail(MRD_EINVAL, "null argument");
  if (!(R > 0.0) || !(B > 0.0)) return gen_fail(MRD_EINVAL, "R and B must be positive");
  cudaStream_t s = (cudaStream_t)stream;
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(256);
  if (e != cudaSuccess) return cuda_fail("test_quality", e);
  unsigned long long *cnt = (unsigned long long *)g_arena.base;
  cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  if (n_triangle > 0)
    mrdgen::test_quality_kernel<<<(unsigned)((n_triangle + 255) / 256), 256, 0, s>>>(n_triangle, (const double2 *)xy_dev, tri_dev, R, B, r_dev, beta_dev,
                                                                                     (double2 *)cc_dev, bad_dev, cnt, mrdgen::SizeGrid{nullptr, 0, 0, 0, 0, 0, 0});
  e = cudaMemcpyAsync(g_arena.pinned, cnt, sizeof *cnt, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("test_quality", e);
  if (n_bad) *n_bad = (int64_t)g_arena.pinned[0];
  return MRD_OK;
}

static int predicate_impl(int which, int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  if (n < 0 || (n > 0 && (!xy_dev || !idx_dev || !sign_dev))) return gen_fail(MRD_EINVAL, "null argument");
  if (n > 0x7FFFFFF0ll) return gen_fail(MRD_EINVAL, "too many tests for 32-bit work lists");
  cudaStream_t s = (cudaStream_t)stream;
  Carve c;
  const size_t o_cnt = c.add(sizeof(unsigned long long)), o_work = c.add(sizeof(int32_t) * (size_t)(n > 0 ? n : 1));
  const size_t o_scr = which == 1 ? c.add(EXACT_SCRATCH) : 0;
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(c.total);
  if (e != cudaSuccess) return cuda_fail("predicate", e);
  unsigned long long *cnt = (unsigned long long *)(g_arena.base + o_cnt);
  int32_t *work = (int32_t *)(g_arena.base + o_work);
  double *scratch = (double *)(g_arena.base + o_scr);
  cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  if (n > 0) {
    const unsigned nb = (unsigned)((n + 255) / 256);
    if (which == 0) {
      mrdgen::orient_filter_kernel<<<nb, 256, 0, s>>>(n, (const double2 *)xy_dev, idx_dev, sign_dev, work, cnt);
      mrdgen::orient_exact_kernel<<<EXACT_BLOCKS, 128, 0, s>>>(cnt, work, (const double2 *)xy_dev, idx_dev, sign_dev);
    } else {
      mrdgen::incircle_filter_kernel<<<nb, 256, 0, s>>>(n, (const double2 *)xy_dev, idx_dev, sign_dev, work, cnt);
      mrdgen::incircle_exact_kernel<<<EXACT_BLOCKS, EXACT_THREADS, 0, s>>>(cnt, work, (const double2 *)xy_dev, idx_dev, sign_dev, scratch);
    }
  }
  e = cudaMemcpyAsync(g_arena.pinned, cnt, sizeof *cnt, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("predicate", e);
  if (n_exact) *n_exact = (int64_t)g_arena.pinned[0];
  return MRD_OK;
}

int mrd_meshgen_orient2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  return predicate_impl(0, n, xy_dev, idx_dev, sign_dev, n_exact, stream);
}
int mrd_meshgen_incircle2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream) {
  return predicate_impl(1, n, xy_dev, idx_dev, sign_dev, n_exact, stream);
}

namespace {
// device address of g_static_scratch on the CURRENT device, taken once per device (with that device current)
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[STATIC_MAX_DEVICES] = {};
int static_scratch_of(unsigned char **out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail("orient2d_static: cudaGetDevice", e);
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return gen_fail(MRD_EINVAL, "orient2d_static: device number beyond 63");
  std::lock_guard<std::mutex> g(g_static_mu);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess || !p) return cuda_fail("orient2d_static: cudaGetSymbolAddress", e);
    g_static_ptr[dev] = (unsigned char *)p;
  }
  *out = g_static_ptr[dev];
  return MRD_OK;
}
}  // namespace

int mrd_meshgen_orient2d_static(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact_dev,
                                void *stream) {
  if (n < 0 || (n > 0 && (!xy_dev || !idx_dev || !sign_dev))) return gen_fail(MRD_EINVAL, "null argument");
  if (n > (int64_t)MRD_STATIC_MAX_TESTS)
    return gen_fail(MRD_EINVAL, "orient2d_static: " + std::to_string(n) + " tests exceed the static scratch (at most " +
                                    std::to_string((int64_t)MRD_STATIC_MAX_TESTS) + " per call; use mrd_meshgen_orient2d)");
  unsigned char *base = nullptr;
  const int rc = static_scratch_of(&base);
  if (rc != MRD_OK) return rc;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long *cnt = (unsigned long long *)base;
  int32_t *work = (int32_t *)(base + 256);
  // the array keeps the last call's contents: the counter must start at zero (the work list is only read below the counter)
  cudaError_t e = cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  if (e == cudaSuccess && n > 0) {
    mrdgen::orient_filter_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(n, (const double2 *)xy_dev, idx_dev, sign_dev, work, cnt);
    mrdgen::orient_exact_kernel<<<EXACT_BLOCKS, 128, 0, s>>>(cnt, work, (const double2 *)xy_dev, idx_dev, sign_dev);
    e = cudaPeekAtLastError();
  }
  if (e == cudaSuccess && n_exact_dev) e = cudaMemcpyAsync(n_exact_dev, cnt, sizeof(int64_t), cudaMemcpyDeviceToDevice, s);
  if (e != cudaSuccess) return cuda_fail("orient2d_static", e);
  return MRD_OK;   // enqueued; no synchronisation
}

namespace {
// work space of build_edges for n = 3 * triangles entries
struct EdgeWork {
  size_t o_k0, o_k1, o_v0, o_v1, o_head, o_incl, o_err, o_tmp, tmp_sort, tmp_scan;
  void plan(Carve &c, int64_t n, cudaStream_t s) {
    tmp_sort = tmp_scan = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, tmp_sort, (unsigned long long *)nullptr, (unsigned long long *)nullptr, (int32_t *)nullptr,
                                    (int32_t *)nullptr, n, 0, 64, s);
    cub::DeviceScan::InclusiveSum(nullptr, tmp_scan, (int32_t *)nullptr, (int32_t *)nullptr, n, s);
    o_k0 = c.add(sizeof(unsigned long long) * n);
    o_k1 = c.add(sizeof(unsigned long long) * n);
    o_v0 = c.add(sizeof(int32_t) * n);
    o_v1 = c.add(sizeof(int32_t) * n);
    o_head = c.add(sizeof(int32_t) * n);
    o_incl = c.add(sizeof(int32_t) * n);
    o_err = c.add(sizeof(int));
    o_tmp = c.add(std::max(tmp_sort, tmp_scan));
  }
};
// te, et from tv (arena reserved and locked by the caller); synchronises s
int build_edges_run(const EdgeWork &w, int64_t n_triangle, int bits, const int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev, int64_t *n_edge, cudaStream_t s) {
  const int64_t n = 3 * n_triangle;
  char *b = g_arena.base;
  unsigned long long *k0 = (unsigned long long *)(b + w.o_k0), *k1 = (unsigned long long *)(b + w.o_k1);
  int32_t *v0 = (int32_t *)(b + w.o_v0), *v1 = (int32_t *)(b + w.o_v1), *head = (int32_t *)(b + w.o_head), *incl = (int32_t *)(b + w.o_incl);
  int *err = (int *)(b + w.o_err);
  const unsigned nb = (unsigned)((n + 255) / 256);
  size_t tmp_sort = w.tmp_sort, tmp_scan = w.tmp_scan;
  cudaMemsetAsync(err, 0, sizeof(int), s);
  cudaMemsetAsync(et_dev, 0xFF, sizeof(int32_t) * 2 * (size_t)n, s);   // -1: no second triangle
  mrdgen::edge_keys_kernel<<<nb, 256, 0, s>>>(n, tv_dev, bits, k0, v0);
  // (only the 2 * bits significant bits are sorted: fewer radix passes when the caller knows how many vertices there are)
  cub::DeviceRadixSort::SortPairs(b + w.o_tmp, tmp_sort, k0, k1, v0, v1, n, 0, std::min(2 * bits, 64), s);
  mrdgen::edge_heads_kernel<<<nb, 256, 0, s>>>(n, k1, head);
  cub::DeviceScan::InclusiveSum(b + w.o_tmp, tmp_scan, head, incl, n, s);
  mrdgen::edge_fill_kernel<<<nb, 256, 0, s>>>(n, k1, v1, incl, te_dev, et_dev, err);
  int32_t *h = (int32_t *)g_arena.pinned;
  cudaMemcpyAsync(h, err, sizeof(int), cudaMemcpyDeviceToHost, s);
  cudaMemcpyAsync(h + 1, incl + (n - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s);
  cudaError_t e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("build_edges", e);
  if (h[0]) return gen_fail(MRD_EINVAL, "build_edges: an edge belongs to more than two triangles");
  *n_edge = h[1];
  return MRD_OK;
}

// work space of the flip loop for up to nt triangles and ne edges
struct FlipWork {
  size_t o_cnt, o_state, o_lock, o_mark, o_l0, o_l1, o_work, o_scr, o_loop;
  void plan(Carve &c, size_t nt, size_t ne, bool with_scratch) {
    o_cnt = c.add(sizeof(mrdgen::FlipCounters));
    o_loop = c.add(sizeof(mrdgen::FlipLoopState));
    o_state = c.add(ne);
    o_lock = c.add(sizeof(unsigned long long) * nt);
    o_mark = c.add(sizeof(int32_t) * ne);
    o_l0 = c.add(sizeof(int32_t) * ne);
    o_l1 = c.add(sizeof(int32_t) * ne);
    o_work = c.add(sizeof(int32_t) * ne);
    o_scr = with_scratch ? c.add(EXACT_SCRATCH) : 0;
  }
};
// flips (tv, te, et) to the Delaunay triangulation (arena reserved and locked by the caller); synchronises s every iteration
// diagnostics of the flip loops since the last mrd_meshgen_flip_stats(reset): cooperative launches, iterations run inside them,
// iterations handed back to the host path because a test needed the long expansions, iterations run by the host path
int64_t g_flip_stats[4] = {0, 0, 0, 0};
constexpr int64_t FLIP_LOOP_MAX = 1 << 16;                           // candidate sets up to this size go through the cooperative loop
int g_flip_loop_cached[64] = {};
int flip_loop_blocks() {                                          // resident blocks of flip_loop_kernel on the current device (0: not available)
  int *cached = g_flip_loop_cached;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 0;
  if (cached[dev] == 0) {
    int coop = 0, per_sm = 0, sms = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (!coop || cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, mrdgen::flip_loop_kernel, 256, 0) != cudaSuccess || per_sm < 1) cached[dev] = -1;
    else cached[dev] = per_sm * sms;
  }
  return cached[dev] > 0 ? cached[dev] : 0;
}
// `init` (refinement only): the caller has cleared state / lock / mark, put the first candidates into the list at w.o_l0 (their
// number in device memory, n_upper an upper bound of it) and wants touched slots recorded
struct FlipInit {
  const unsigned long long *n_dev;
  int64_t n_upper;
  mrdgen::Touch touch;
};
int flip_run(const FlipWork &w, size_t o_scratch, int64_t n_triangle, int64_t n_edge, const double2 *xy, int32_t *tv_dev, int32_t *te_dev,
             int32_t *et_dev, int64_t *flips_out, int64_t *iters_out, int64_t *exact_out, cudaStream_t s, const FlipInit *init = nullptr) {
  using mrdgen::FlipCounters;
  const size_t nt = (size_t)std::max<int64_t>(n_triangle, 1), ne = (size_t)n_edge;
  char *b = g_arena.base;
  FlipCounters *cnt = (FlipCounters *)(b + w.o_cnt);
  int8_t *state = (int8_t *)(b + w.o_state);
  unsigned long long *lock = (unsigned long long *)(b + w.o_lock);
  int32_t *mark = (int32_t *)(b + w.o_mark), *list[2] = {(int32_t *)(b + w.o_l0), (int32_t *)(b + w.o_l1)}, *work = (int32_t *)(b + w.o_work);
  double *scratch = (double *)(b + o_scratch);
  static_assert(sizeof(FlipCounters) <= 16 * sizeof(unsigned long long), "pinned block too small");
  const FlipCounters *h = (const FlipCounters *)g_arena.pinned;
  int64_t flips = 0, iters = 0, exact = 0;
  if (!init) {
    cudaMemsetAsync(state, 0, ne, s);
    cudaMemsetAsync(lock, 0, sizeof(unsigned long long) * nt, s);
    cudaMemsetAsync(mark, 0, sizeof(int32_t) * ne, s);
  }
  int64_t n = init ? init->n_upper : n_edge;
  const int32_t *cand = init ? list[0] : nullptr;                // first iteration: every edge, unless the caller knows better
  const unsigned long long *n_dev = init ? init->n_dev : nullptr;
  const mrdgen::Touch touch = init ? init->touch : mrdgen::Touch{nullptr, nullptr, nullptr, nullptr, nullptr};
  mrdgen::FlipLoopState *loop_dev = (mrdgen::FlipLoopState *)(b + w.o_loop);
  static_assert(sizeof(mrdgen::FlipLoopState) <= 16 * sizeof(unsigned long long), "pinned block too small");
  bool host_once = false;                                         // the cooperative loop handed one iteration back
  for (int32_t iter = 1;; ++iter) {
    if (iter > 100000) return gen_fail(MRD_EINVAL, "delaunay_flip: no convergence (is the input a valid triangulation?)");
    if (cand && n > 0 && n <= FLIP_LOOP_MAX && !host_once) {
      // small candidate set: the rest of the loop in one cooperative launch (flip_loop_kernel)
      const int blocks = std::min<int64_t>((n + 255) / 256, flip_loop_blocks());
      if (blocks > 0) {
        cudaMemsetAsync(loop_dev, 0, sizeof(mrdgen::FlipLoopState), s);
        int64_t n0 = n;
        int32_t iter0 = iter;
        int max_iters = 64;
        int32_t *l0 = list[0], *l1 = list[1];
        void *args[] = {&n0, (void *)&n_dev, &iter0, &max_iters, &l0, &l1, (void *)&xy, &tv_dev, &te_dev, &et_dev, &state, &lock, &mark, &loop_dev, (void *)&touch};
        cudaError_t e = cudaLaunchCooperativeKernel((const void *)mrdgen::flip_loop_kernel, dim3(blocks), dim3(256), args, 0, s);
        if (e != cudaSuccess) {
          // the device cannot hold the grid right now (another context shares it, MPS limits, ...): nothing has run, so the
          // launch-by-launch path does this and every later iteration of the process
          cudaGetLastError();
          int dev = 0;
          if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < 64) g_flip_loop_cached[dev] = -1;
          host_once = true;
          --iter;
          continue;
        }
        e = cudaMemcpyAsync(g_arena.pinned, loop_dev, sizeof(mrdgen::FlipLoopState), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail("delaunay_flip (cooperative loop)", e);
        const mrdgen::FlipLoopState *hl = (const mrdgen::FlipLoopState *)g_arena.pinned;
        g_flip_stats[0] += 1;
        g_flip_stats[1] += hl->done_iters;
        g_flip_stats[2] += hl->abort ? 1 : 0;
        iters += hl->done_iters;
        flips += (int64_t)hl->n_flip;
        exact += (int64_t)hl->n_exact;
        if (hl->converged) break;
        iter += hl->done_iters;                                   // resume at the iteration the loop stopped at
        cand = list[(iter & 1) ^ 1];
        n = (int64_t)hl->n_cur;
        n_dev = nullptr;
        host_once = hl->abort != 0;                               // that iteration needs the long expansions: host path once
        --iter;                                                   // (the for statement adds it back)
        continue;
      }
    }
    host_once = false;
    g_flip_stats[3] += 1;
    const unsigned long long stamp = (unsigned long long)iter << 32;
    int32_t *next = list[iter & 1];
    const unsigned nb = (unsigned)((n + 255) / 256);
    cudaMemsetAsync(cnt, 0, sizeof(FlipCounters), s);
    if (n > 0) mrdgen::check_edge_kernel<<<nb, 256, 0, s>>>(n, cand, xy, tv_dev, te_dev, et_dev, state, lock, stamp, work, cnt, n_dev);
    mrdgen::check_edge_exact_kernel<<<EXACT_BLOCKS, EXACT_THREADS, 0, s>>>(work, xy, tv_dev, te_dev, et_dev, state, lock, stamp, cnt, scratch);
    if (n > 0) mrdgen::flip_kernel<<<nb, 256, 0, s>>>(n, cand, tv_dev, te_dev, et_dev, state, lock, stamp, iter, mark, next, cnt, n_dev, touch);
    cudaError_t e = cudaMemcpyAsync(g_arena.pinned, cnt, sizeof(FlipCounters), cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail("delaunay_flip", e);
    iters++;
    flips += (int64_t)h->n_flip;
    exact += (int64_t)h->n_exact;
    if (h->n_bad == 0) break;                                    // every edge is locally Delaunay
    cand = next;
    n = (int64_t)h->n_next;
    n_dev = nullptr;
  }
  if (flips_out) *flips_out = flips;
  if (iters_out) *iters_out = iters;
  if (exact_out) *exact_out = exact;
  return MRD_OK;
}
}  // namespace

int mrd_meshgen_flip_stats(int64_t stats[4], int reset) {
  std::lock_guard<std::mutex> g(g_arena.mu);
  if (stats)
    for (int k = 0; k < 4; ++k) stats[k] = g_flip_stats[k];
  if (reset)
    for (int k = 0; k < 4; ++k) g_flip_stats[k] = 0;
  return MRD_OK;
}

int mrd_meshgen_build_edges(int64_t n_triangle, const int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev, int64_t *n_edge, void *stream) {
  if (n_triangle < 0 || !n_edge || (n_triangle > 0 && (!tv_dev || !te_dev || !et_dev))) return gen_fail(MRD_EINVAL, "null argument");
  if (3 * n_triangle > 0x7FFFFFF0ll) return gen_fail(MRD_EINVAL, "too many triangles for 32-bit edge numbers");
  *n_edge = 0;
  if (n_triangle == 0) return MRD_OK;
  cudaStream_t s = (cudaStream_t)stream;
  Carve c;
  EdgeWork w;
  w.plan(c, 3 * n_triangle, s);
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(c.total);
  if (e != cudaSuccess) return cuda_fail("build_edges", e);
  return build_edges_run(w, n_triangle, 32, tv_dev, te_dev, et_dev, n_edge, s);
}

int mrd_meshgen_delaunay_flip(int64_t n_triangle, int64_t n_edge, const double *xy_dev, int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev,
                              int64_t *n_flips, int64_t *n_iterations, int64_t *n_exact, void *stream) {
  if (n_triangle < 0 || n_edge < 0 || ((n_triangle > 0 || n_edge > 0) && (!xy_dev || !tv_dev || !te_dev || !et_dev)))
    return gen_fail(MRD_EINVAL, "null argument");
  if (n_edge > 0x7FFFFFF0ll) return gen_fail(MRD_EINVAL, "too many edges");
  if (n_flips) *n_flips = 0;
  if (n_iterations) *n_iterations = 0;
  if (n_exact) *n_exact = 0;
  if (n_edge == 0) return MRD_OK;
  cudaStream_t s = (cudaStream_t)stream;
  Carve c;
  FlipWork w;
  w.plan(c, (size_t)std::max<int64_t>(n_triangle, 1), (size_t)n_edge, true);
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(c.total);
  if (e != cudaSuccess) return cuda_fail("delaunay_flip", e);
  // a triangulation with a clockwise triangle is not valid, and flips on it need not terminate: refuse it
  unsigned long long *bad = (unsigned long long *)(g_arena.base + w.o_cnt);
  cudaMemsetAsync(bad, 0, sizeof *bad, s);
  if (n_triangle > 0)
    mrdgen::validate_kernel<<<(unsigned)((n_triangle + 255) / 256), 256, 0, s>>>(n_triangle, 0x7FFFFFFF, (const double2 *)xy_dev, tv_dev, bad);
  e = cudaMemcpyAsync(g_arena.pinned, bad, sizeof *bad, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("delaunay_flip", e);
  if (g_arena.pinned[0] != 0)
    return gen_fail(MRD_EINVAL, "delaunay_flip: " + std::to_string(g_arena.pinned[0]) + " triangles of the input are clockwise or degenerate");
  cudaMemsetAsync(bad, 0, sizeof *bad, s);
  if (n_triangle > 0) mrdgen::validate_sides_kernel<<<(unsigned)((n_triangle + 255) / 256), 256, 0, s>>>(n_triangle, n_edge, te_dev, et_dev, bad);
  if (n_edge > 0) mrdgen::validate_edges_kernel<<<(unsigned)((n_edge + 255) / 256), 256, 0, s>>>(n_edge, n_triangle, tv_dev, te_dev, et_dev, bad);
  e = cudaMemcpyAsync(g_arena.pinned, bad, sizeof *bad, cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("delaunay_flip", e);
  if (g_arena.pinned[0] != 0)
    return gen_fail(MRD_EINVAL, "delaunay_flip: the edge tables do not describe a triangulation (" + std::to_string(g_arena.pinned[0]) +
                    " entries: triangleEdges and edgeTriangles disagree, or the two triangles of an edge lie on the same side of it)");
  return flip_run(w, w.o_scr, n_triangle, n_edge, (const double2 *)xy_dev, tv_dev, te_dev, et_dev, n_flips, n_iterations, n_exact, s);
}

int mrd_meshgen_refine(double R, double B, uint32_t seed, int64_t first_iteration, int64_t max_iterations, const double *box,
                       const double *size_dev, const double *size_box, int64_t size_nx, int64_t size_ny, int64_t cap_vertex,
                       int64_t cap_triangle, int64_t cap_edge, int64_t *n_vertex, int64_t *n_triangle, int64_t *n_edge, double *xy_dev,
                       int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev, int64_t *n_iterations, int64_t *n_bad_left, void *stream) {
  if (!n_vertex || !n_triangle || !n_edge || !xy_dev || !tv_dev || !te_dev || !et_dev) return gen_fail(MRD_EINVAL, "null argument");
  if (!(R > 0.0) || !(B > 0.0)) return gen_fail(MRD_EINVAL, "R and B must be positive");
  if (box && !(box[2] > box[0] && box[3] > box[1])) return gen_fail(MRD_EINVAL, "refine: box must be (x0, y0, x1, y1) with x1 > x0, y1 > y0");
  mrdgen::SizeGrid size_grid{nullptr, 0, 0, 0, 0, 0, 0};
  if (size_dev) {
    if (!size_box || !(size_box[2] > size_box[0] && size_box[3] > size_box[1]) || size_nx < 2 || size_ny < 2 || size_nx > 1 << 20 || size_ny > 1 << 20)
      return gen_fail(MRD_EINVAL, "refine: the size grid needs its rectangle (x0, y0, x1, y1) and at least 2 x 2 points");
    size_grid = mrdgen::SizeGrid{size_dev, (int)size_nx, (int)size_ny, size_box[0], size_box[1], ((double)size_nx - 1.0) / (size_box[2] - size_box[0]),
                                 ((double)size_ny - 1.0) / (size_box[3] - size_box[1])};
  }
  int64_t nv = *n_vertex, nt = *n_triangle, ne = *n_edge;
  if (nv < 3 || nt < 1 || ne < 3 || nv > cap_vertex || nt > cap_triangle || ne > cap_edge || first_iteration < 0 || max_iterations < 0)
    return gen_fail(MRD_EINVAL, "refine: sizes out of range");
  if (cap_edge > 0x7FFFFFF0ll / 2 || 3 * cap_triangle > 0x7FFFFFF0ll) return gen_fail(MRD_EINVAL, "refine: capacity beyond 32-bit numbering");
  if (cap_edge < 3 * cap_triangle) return gen_fail(MRD_EINVAL, "refine: et must hold 3 * cap_triangle pairs (mrd_meshgen_build_edges writes that many)");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t ct = (size_t)cap_triangle, ce = (size_t)cap_edge;
  Carve c;
  EdgeWork ew;
  ew.plan(c, 3 * cap_triangle, s);
  FlipWork fw;
  fw.plan(c, ct, ce, false);
  const size_t o_scr = c.add(EXACT_SCRATCH);
  const size_t o_cnt = c.add(sizeof(unsigned long long)), o_err = c.add(sizeof(int)), o_nsel = c.add(sizeof(int32_t));
  const size_t o_r = c.add(sizeof(double) * ct), o_beta = c.add(sizeof(double) * ct), o_cc = c.add(sizeof(double2) * ct), o_bad = c.add(ct);
  const size_t o_cand = c.add(sizeof(int32_t) * ct), o_kind = c.add(ct), o_pt = c.add(sizeof(double2) * ct);
  const size_t o_tins = c.add(sizeof(int32_t) * ct), o_eins = c.add(sizeof(int32_t) * ct), o_claim = c.add(sizeof(unsigned long long) * ct);
  const size_t o_sel = c.add(sizeof(int32_t) * ct), o_seg = c.add(sizeof(int32_t) * ct), o_rank = c.add(sizeof(int32_t) * ct), o_srank = c.add(sizeof(int32_t) * ct);
  const size_t o_touch_t = c.add(ct), o_touch_e = c.add(ce), o_slot_t = c.add(sizeof(int32_t) * ct), o_slot_e = c.add(sizeof(int32_t) * ce);
  const size_t o_tri_map = c.add(sizeof(int32_t) * ct), o_edge_map = c.add(sizeof(int32_t) * ce), o_tmp_te = c.add(sizeof(int32_t) * 3 * ct);
  const size_t o_tmp_et = c.add(sizeof(int2) * ce), o_jpos = c.add(3 * ct), o_ninit = c.add(sizeof(unsigned long long));
  const int64_t pool_cap = (int64_t)std::min<size_t>(4 * ct, (size_t)1 << 28);   // ints; a cavity takes 1 + its size
  const size_t o_cav_pool = c.add(sizeof(int32_t) * (size_t)pool_cap), o_cav_off = c.add(sizeof(int32_t) * ct), o_pool_n = c.add(sizeof(unsigned long long));
  const size_t o_near = c.add((size_t)cap_vertex);
  const size_t o_cav_store = c.add(sizeof(int32_t) * (size_t)mrdgen::CAVITY_STORE * (mrdgen::CAVITY_MAX + 1));
  const size_t o_cwork = c.add(sizeof(int32_t) * ct), o_cwork2 = c.add(sizeof(int32_t) * ct), o_cwn = c.add(2 * sizeof(unsigned long long));
  const size_t cm = std::max(ct, (size_t)cap_vertex);               // the sort buffers serve triangles and vertices
  const size_t o_klo0 = c.add(sizeof(unsigned long long) * cm), o_klo1 = c.add(sizeof(unsigned long long) * cm);
  const size_t o_khi0 = c.add(sizeof(unsigned) * ct), o_khi1 = c.add(sizeof(unsigned) * ct);
  const size_t o_i0 = c.add(sizeof(int32_t) * cm), o_i1 = c.add(sizeof(int32_t) * cm), o_tv2 = c.add(sizeof(int32_t) * 3 * ct);
  const size_t o_xy2 = c.add(sizeof(double2) * (size_t)cap_vertex), o_num = c.add(sizeof(int32_t) * (size_t)cap_vertex);   // (cap_vertex <= cap_triangle is not required)
  size_t tmp_sel = 0, tmp_scan = 0, tmp_s64 = 0, tmp_s32 = 0;
  cub::DeviceSelect::Flagged(nullptr, tmp_sel, thrust::counting_iterator<int32_t>(0), (const uint8_t *)nullptr, (int32_t *)nullptr, (int32_t *)nullptr, (int64_t)ce, s);
  cub::DeviceScan::ExclusiveSum(nullptr, tmp_scan, (int32_t *)nullptr, (int32_t *)nullptr, (int64_t)ct, s);
  cub::DeviceRadixSort::SortPairs(nullptr, tmp_s64, (unsigned long long *)nullptr, (unsigned long long *)nullptr, (int32_t *)nullptr, (int32_t *)nullptr, (int64_t)cm, 0, 64, s);
  cub::DeviceRadixSort::SortPairs(nullptr, tmp_s32, (unsigned *)nullptr, (unsigned *)nullptr, (int32_t *)nullptr, (int32_t *)nullptr, (int64_t)ct, 0, 32, s);
  constexpr int64_t MERGE_MAX = 1 << 16;                              // touched sets up to this size go through a merge sort
  size_t tmp_m3 = 0, tmp_m1 = 0;
  cub::DeviceMergeSort::SortPairs(nullptr, tmp_m3, (mrdgen::TriKey *)nullptr, (int32_t *)nullptr, MERGE_MAX, mrdgen::TriKeyLess(), s);
  cub::DeviceMergeSort::SortPairs(nullptr, tmp_m1, (unsigned long long *)nullptr, (int32_t *)nullptr, MERGE_MAX, mrdgen::U64Less(), s);
  const size_t tmp_all = std::max(std::max(std::max(tmp_sel, tmp_scan), std::max(tmp_s64, tmp_s32)), std::max(tmp_m3, tmp_m1));
  const size_t o_tmp = c.add(tmp_all);
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(c.total);
  if (e != cudaSuccess) return cuda_fail("refine", e);
  char *b = g_arena.base;
  unsigned long long *cnt = (unsigned long long *)(b + o_cnt), *claim = (unsigned long long *)(b + o_claim);
  int *err = (int *)(b + o_err);
  int32_t *d_nsel = (int32_t *)(b + o_nsel);
  double *r = (double *)(b + o_r), *beta = (double *)(b + o_beta), *scratch = (double *)(b + o_scr);
  double2 *cc = (double2 *)(b + o_cc), *pt = (double2 *)(b + o_pt), *xy = (double2 *)xy_dev;
  uint8_t *bad = (uint8_t *)(b + o_bad);
  int8_t *kind = (int8_t *)(b + o_kind);
  int32_t *cand = (int32_t *)(b + o_cand), *tins = (int32_t *)(b + o_tins), *eins = (int32_t *)(b + o_eins);
  int32_t *sel = (int32_t *)(b + o_sel), *seg = (int32_t *)(b + o_seg), *rank = (int32_t *)(b + o_rank), *srank = (int32_t *)(b + o_srank);
  unsigned long long *klo0 = (unsigned long long *)(b + o_klo0), *klo1 = (unsigned long long *)(b + o_klo1);
  unsigned *khi0 = (unsigned *)(b + o_khi0), *khi1 = (unsigned *)(b + o_khi1);
  int32_t *i0 = (int32_t *)(b + o_i0), *i1 = (int32_t *)(b + o_i1), *tv2 = (int32_t *)(b + o_tv2), *number = (int32_t *)(b + o_num);
  double2 *xy2 = (double2 *)(b + o_xy2);
  uint8_t *touch_t = (uint8_t *)(b + o_touch_t), *touch_e = (uint8_t *)(b + o_touch_e);
  int32_t *slot_t = (int32_t *)(b + o_slot_t), *slot_e = (int32_t *)(b + o_slot_e), *tri_map = (int32_t *)(b + o_tri_map);
  int32_t *edge_map = (int32_t *)(b + o_edge_map), *tmp_te = (int32_t *)(b + o_tmp_te);
  int2 *tmp_et = (int2 *)(b + o_tmp_et);
  int8_t *jpos = (int8_t *)(b + o_jpos);
  unsigned long long *n_init = (unsigned long long *)(b + o_ninit);
  int32_t *cav_store = (int32_t *)(b + o_cav_store), *cav_pool = (int32_t *)(b + o_cav_pool), *cav_off = (int32_t *)(b + o_cav_off);
  unsigned long long *pool_n = (unsigned long long *)(b + o_pool_n);
  uint8_t *near_seg = (uint8_t *)(b + o_near);
  int32_t *cwork = (int32_t *)(b + o_cwork), *cwork2 = (int32_t *)(b + o_cwork2);
  unsigned long long *cwork_n = (unsigned long long *)(b + o_cwn);
  void *tmp = b + o_tmp;
  volatile unsigned long long *hp = g_arena.pinned;
  auto sync = [&](const char *what) -> int {
    cudaError_t e2 = cudaStreamSynchronize(s);
    if (e2 == cudaSuccess) e2 = cudaGetLastError();
    return e2 == cudaSuccess ? MRD_OK : cuda_fail(what, e2);
  };
  // 4.1.4 / M12 / M14: (vertices along the Morton curve of the box,) triangles in canonical order, edges rebuilt
  auto resort = [&](int bits) -> int {
    size_t tb;
    const unsigned nbt = (unsigned)((nt + 255) / 256);
    if (box) {
      const unsigned nbv = (unsigned)((nv + 255) / 256);
      mrdgen::morton_keys_kernel<<<nbv, 256, 0, s>>>(nv, xy, box[0], box[1], 2097152.0 / (box[2] - box[0]), 2097152.0 / (box[3] - box[1]), klo0, i0);
      tb = tmp_s64;
      cub::DeviceRadixSort::SortPairs(tmp, tb, klo0, klo1, i0, i1, nv, 0, 42, s);   // stable: ties keep their order
      mrdgen::vertex_permute_kernel<<<nbv, 256, 0, s>>>(nv, i1, xy, xy2, number);
      cudaMemcpyAsync(xy, xy2, sizeof(double2) * (size_t)nv, cudaMemcpyDeviceToDevice, s);
      mrdgen::relabel_kernel<<<(unsigned)((3 * nt + 255) / 256), 256, 0, s>>>(3 * nt, number, tv_dev);
    }
    mrdgen::canonical_keys_kernel<<<nbt, 256, 0, s>>>(nt, tv_dev, bits, klo0, i0);
    tb = tmp_s64;
    cub::DeviceRadixSort::SortPairs(tmp, tb, klo0, klo1, i0, i1, nt, 0, 2 * bits, s);
    mrdgen::gather_first_kernel<<<nbt, 256, 0, s>>>(nt, tv_dev, i1, khi0);
    tb = tmp_s32;
    cub::DeviceRadixSort::SortPairs(tmp, tb, khi0, khi1, i1, i0, nt, 0, bits, s);
    mrdgen::gather_rows_kernel<<<nbt, 256, 0, s>>>(nt, tv_dev, i0, tv2);
    cudaMemcpyAsync(tv_dev, tv2, sizeof(int32_t) * 3 * (size_t)nt, cudaMemcpyDeviceToDevice, s);
    int64_t ne_built = 0;
    const int r2 = build_edges_run(ew, nt, bits, tv_dev, te_dev, et_dev, &ne_built, s);
    if (r2 != MRD_OK) return r2;
    if (ne_built != ne) return gen_fail(MRD_EINVAL, "refine: edge count changed under renumbering (internal error)");
    return MRD_OK;
  };
  int64_t done = 0, left = 0;
  int rc = MRD_OK;
  cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  mrdgen::validate_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, s>>>(nt, nv, xy, tv_dev, cnt);
  cudaMemcpyAsync((void *)hp, cnt, sizeof *cnt, cudaMemcpyDeviceToHost, s);
  if ((rc = sync("refine: input check")) != MRD_OK) return rc;
  if (hp[0] != 0)
    return gen_fail(MRD_EINVAL, "refine: " + std::to_string((unsigned long long)hp[0]) + " triangles of the input are clockwise, degenerate or name vertices out of range");
  cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
  mrdgen::validate_sides_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, s>>>(nt, ne, te_dev, et_dev, cnt);
  mrdgen::validate_edges_kernel<<<(unsigned)((ne + 255) / 256), 256, 0, s>>>(ne, nt, tv_dev, te_dev, et_dev, cnt);
  cudaMemcpyAsync((void *)hp, cnt, sizeof *cnt, cudaMemcpyDeviceToHost, s);
  if ((rc = sync("refine: input check")) != MRD_OK) return rc;
  if (hp[0] != 0)
    return gen_fail(MRD_EINVAL, "refine: the edge tables do not describe a triangulation (" + std::to_string((unsigned long long)hp[0]) +
                    " entries: triangleEdges and edgeTriangles disagree, or the two triangles of an edge lie on the same side of it)");
  for (int64_t it = 0;; ++it) {
    // 2.4.1: bad triangles and their circumcentres
    cudaMemsetAsync(cnt, 0, sizeof *cnt, s);
    mrdgen::test_quality_kernel<<<(unsigned)((nt + 255) / 256), 256, 0, s>>>(nt, xy, tv_dev, R, B, r, beta, cc, bad, cnt, size_grid);
    cudaMemcpyAsync((void *)hp, cnt, sizeof *cnt, cudaMemcpyDeviceToHost, s);
    if ((rc = sync("refine: test_quality")) != MRD_OK) return rc;
    const int64_t nc = (int64_t)hp[0];
    left = nc;
    if (nc == 0 || it >= max_iterations) break;
    // candidates in ascending order of their bad triangle; 2.4.2-2.4.3
    size_t tb = tmp_sel;
    cub::DeviceSelect::Flagged(tmp, tb, thrust::counting_iterator<int32_t>(0), (const uint8_t *)bad, cand, d_nsel, nt, s);
    cudaMemsetAsync(err, 0, sizeof(int), s);
    cudaMemsetAsync(near_seg, 0, (size_t)nv, s);
    mrdgen::near_segment_kernel<<<(unsigned)((ne + 255) / 256), 256, 0, s>>>(ne, et_dev, tv_dev, near_seg);
    mrdgen::candidate_kernel<<<(unsigned)((nc + 127) / 128), 128, 0, s>>>(nc, cand, cc, nt + 16, xy, tv_dev, te_dev, et_dev, kind, pt, tins, eins, err, near_seg);
    // 4.1.1: cavities, claims, selection
    cudaMemsetAsync(claim, 0, sizeof(unsigned long long) * (size_t)nt, s);
    const unsigned itn = (unsigned)(first_iteration + it);
    const unsigned nbc = (unsigned)((nc + 127) / 128);
    cudaMemsetAsync(cwork_n, 0, 2 * sizeof(unsigned long long), s);
    cudaMemsetAsync(pool_n, 0, sizeof(unsigned long long), s);
    mrdgen::cavity_kernel<1><<<nbc, 128, 0, s>>>(nc, cand, kind, pt, tins, eins, xy, tv_dev, te_dev, et_dev, claim, seed, itn, sel, seg, cwork, cwork_n,
                                                 cav_pool, pool_n, pool_cap, cav_off, nt);
    mrdgen::cavity_exact_kernel<1><<<EXACT_BLOCKS, EXACT_THREADS, 0, s>>>(cwork_n, cwork, cand, kind, pt, tins, eins, xy, tv_dev, te_dev, et_dev, claim, seed, itn, sel, seg, scratch, cav_store, nt);
    mrdgen::cavity_kernel<2><<<nbc, 128, 0, s>>>(nc, cand, kind, pt, tins, eins, xy, tv_dev, te_dev, et_dev, claim, seed, itn, sel, seg, cwork2, cwork_n + 1,
                                                 cav_pool, pool_n, pool_cap, cav_off, nt);
    mrdgen::cavity_exact_kernel<2><<<EXACT_BLOCKS, EXACT_THREADS, 0, s>>>(cwork_n, cwork, cand, kind, pt, tins, eins, xy, tv_dev, te_dev, et_dev, claim, seed, itn, sel, seg, scratch, cav_store, nt);
    tb = tmp_scan;
    cub::DeviceScan::ExclusiveSum(tmp, tb, sel, rank, nc, s);
    tb = tmp_scan;
    cub::DeviceScan::ExclusiveSum(tmp, tb, seg, srank, nc, s);
    int32_t *h32 = (int32_t *)hp;
    cudaMemcpyAsync(h32 + 0, err, sizeof(int), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(h32 + 1, rank + (nc - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(h32 + 2, sel + (nc - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(h32 + 3, srank + (nc - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    cudaMemcpyAsync(h32 + 4, seg + (nc - 1), sizeof(int32_t), cudaMemcpyDeviceToHost, s);
    if ((rc = sync("refine: candidates")) != MRD_OK) return rc;
    if (h32[0]) return gen_fail(MRD_EINVAL, "refine: a point-location walk did not end (the input is not a Delaunay triangulation)");
    const int64_t nsel = (int64_t)h32[1] + h32[2], nseg = (int64_t)h32[3] + h32[4];
    if (nsel == 0) return gen_fail(MRD_EINVAL, "refine: bad triangles remain but no vertex can be inserted (every circumcentre falls on a vertex, or the input was not a Delaunay triangulation)");
    const int64_t nv2 = nv + nsel, nt2 = nt + 2 * nsel - nseg, ne2 = ne + 3 * nsel - nseg;
    if (nv2 > cap_vertex || nt2 > cap_triangle || ne2 > cap_edge) {
      rc = gen_fail(MRD_ENOMEM, "refine: capacity of the mesh arrays reached (the mesh is valid and Delaunay; call again with larger arrays)");
      break;
    }
    // 2.4.4: insert; 2.4.6: flips
    const bool in_place = box == nullptr;                          // reading M15: no re-sort inside the loop
    mrdgen::Touch touch{nullptr, nullptr, nullptr, nullptr, nullptr};
    FlipInit init{nullptr, 0, touch};
    if (in_place) {
      cudaMemsetAsync(touch_t, 0, (size_t)nt2, s);
      cudaMemsetAsync(touch_e, 0, (size_t)ne2, s);
      cudaMemsetAsync(b + fw.o_state, 0, (size_t)ne2, s);
      cudaMemsetAsync(b + fw.o_lock, 0, sizeof(unsigned long long) * (size_t)nt2, s);
      cudaMemsetAsync(b + fw.o_mark, 0, sizeof(int32_t) * (size_t)ne2, s);
      cudaMemsetAsync(n_init, 0, sizeof(unsigned long long), s);
      touch = mrdgen::Touch{touch_t, touch_e, (int32_t *)(b + fw.o_mark), (int32_t *)(b + fw.o_l0), n_init};
      init = FlipInit{n_init, 8 * nsel, touch};                    // at most 8 edges per inserted vertex
    }
    mrdgen::insert_kernel<<<(unsigned)((nc + 127) / 128), 128, 0, s>>>(nc, kind, pt, tins, eins, sel, rank, srank, (int32_t)nv, (int32_t)nt, (int32_t)ne, xy, tv_dev, te_dev, et_dev, touch);
    nv = nv2; nt = nt2; ne = ne2;
    if ((rc = flip_run(fw, o_scr, nt, ne, xy, tv_dev, te_dev, et_dev, nullptr, nullptr, nullptr, s, in_place ? &init : nullptr)) != MRD_OK) return rc;
    int bits = 1;
    while ((1ll << bits) < nv) ++bits;                               // width of a vertex number
    if (in_place) {
      // created triangles and edges into the freed and the new slots, in ascending order (M15)
      size_t tb = tmp_sel;
      cub::DeviceSelect::Flagged(tmp, tb, thrust::counting_iterator<int32_t>(0), (const uint8_t *)touch_t, slot_t, d_nsel, nt, s);
      tb = tmp_sel;
      cub::DeviceSelect::Flagged(tmp, tb, thrust::counting_iterator<int32_t>(0), (const uint8_t *)touch_e, slot_e, d_nsel + 1, ne, s);
      int32_t *h32b = (int32_t *)hp;
      cudaMemcpyAsync(h32b, d_nsel, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
      if ((rc = sync("refine: touched slots")) != MRD_OK) return rc;
      const int64_t ns = h32b[0], nse = h32b[1];
      const unsigned nbs = (unsigned)((ns + 255) / 256), nbs3 = (unsigned)((3 * ns + 255) / 256), nbe = (unsigned)((nse + 255) / 256);
      if (ns <= MERGE_MAX) {
        mrdgen::TriKey *tk = (mrdgen::TriKey *)klo0;               // (12 bytes per key: klo0 and klo1 are adjacent and 16 bytes per item together)
        mrdgen::touched_triples_kernel<<<nbs, 256, 0, s>>>(ns, slot_t, tv_dev, te_dev, tk, i0);
        tb = tmp_all;
        cub::DeviceMergeSort::SortPairs(tmp, tb, tk, i0, ns, mrdgen::TriKeyLess(), s);     // i0: order of the touched triangles
      } else {
        mrdgen::touched_keys_kernel<<<nbs, 256, 0, s>>>(ns, slot_t, tv_dev, te_dev, bits, klo0, i0);
        tb = tmp_s64;
        cub::DeviceRadixSort::SortPairs(tmp, tb, klo0, klo1, i0, i1, ns, 0, 2 * bits, s);
        mrdgen::touched_first_kernel<<<nbs, 256, 0, s>>>(ns, slot_t, tv_dev, i1, khi0);
        tb = tmp_s32;
        cub::DeviceRadixSort::SortPairs(tmp, tb, khi0, khi1, i1, i0, ns, 0, bits, s);      // i0: order of the touched triangles
      }
      mrdgen::tri_map_kernel<<<nbs, 256, 0, s>>>(ns, slot_t, i0, tv_dev, te_dev, tri_map, tv2, tmp_te);
      unsigned long long *ek0 = (unsigned long long *)(b + ew.o_k0), *ek1 = (unsigned long long *)(b + ew.o_k1);
      int32_t *ev0 = (int32_t *)(b + ew.o_v0), *ev1 = (int32_t *)(b + ew.o_v1);             // (the edge builder's buffers are idle here)
      mrdgen::touched_edge_keys_kernel<<<nbe, 256, 0, s>>>(nse, slot_e, tv_dev, te_dev, et_dev, bits, ek0, ev0);
      const int32_t *eorder = ev1;                                 // order of the touched edges
      if (nse <= MERGE_MAX) {
        tb = tmp_all;
        cub::DeviceMergeSort::SortPairs(tmp, tb, ek0, ev0, nse, mrdgen::U64Less(), s);
        eorder = ev0;
      } else {
        tb = ew.tmp_sort;
        cub::DeviceRadixSort::SortPairs(b + ew.o_tmp, tb, ek0, ek1, ev0, ev1, nse, 0, 2 * bits, s);
      }
      mrdgen::edge_map_kernel<<<nbe, 256, 0, s>>>(nse, slot_e, eorder, et_dev, edge_map, tmp_et);
      mrdgen::side_pos_kernel<<<nbs3, 256, 0, s>>>(ns, slot_t, i0, tmp_te, touch_e, et_dev, jpos);
      mrdgen::renumber_scatter_kernel<<<std::max(nbs, nbe), 256, 0, s>>>(ns, nse, slot_t, slot_e, tv2, tmp_te, tmp_et, jpos, touch_e, tri_map, edge_map,
                                                                        tv_dev, te_dev, et_dev);
      mrdgen::renumber_order_kernel<<<nbs3, 256, 0, s>>>(ns, slot_t, te_dev, et_dev);
    } else {
      if ((rc = resort(bits)) != MRD_OK) return rc;                // 4.1.4: vertices along the Morton curve, canonical triangles (M12, M14)
    }
    done++;
  }
  if (!box && done > 0) {                                          // one canonical re-sort after the last in-place iteration
    int bits = 1;
    while ((1ll << bits) < nv) ++bits;
    const int rc2 = resort(bits);
    if (rc2 != MRD_OK) return rc2;
  }
  *n_vertex = nv;
  *n_triangle = nt;
  *n_edge = ne;
  if (n_iterations) *n_iterations = done;
  if (n_bad_left) *n_bad_left = left;
  return rc;
}

int mrd_meshgen_find_triangle(int64_t n_point, const double *p_dev, const int32_t *t0_dev, int64_t n_triangle, const double *xy_dev,
                              const int32_t *tv_dev, const int32_t *te_dev, const int32_t *et_dev, int32_t *t_dev, int8_t *code_dev,
                              void *stream) {
  if (n_point < 0 || n_triangle < 0 || (n_point > 0 && (!p_dev || !t0_dev || !xy_dev || !tv_dev || !te_dev || !et_dev || !t_dev || !code_dev)))
    return gen_fail(MRD_EINVAL, "null argument");
  if (n_point == 0) return MRD_OK;
  if (n_triangle == 0) return gen_fail(MRD_EINVAL, "find_triangle: empty triangulation");
  cudaStream_t s = (cudaStream_t)stream;
  std::lock_guard<std::mutex> g(g_arena.mu);
  cudaError_t e = g_arena.reserve(256);
  if (e != cudaSuccess) return cuda_fail("find_triangle", e);
  int *err = (int *)g_arena.base;
  cudaMemsetAsync(err, 0, sizeof(int), s);
  mrdgen::find_triangle_kernel<<<(unsigned)((n_point + 127) / 128), 128, 0, s>>>(n_point, (const double2 *)p_dev, t0_dev, n_triangle + 16,
                                                                                   (const double2 *)xy_dev, tv_dev, te_dev, et_dev, t_dev, code_dev, err);
  e = cudaMemcpyAsync(g_arena.pinned, err, sizeof(int), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail("find_triangle", e);
  if (*(const int *)g_arena.pinned) return gen_fail(MRD_EINVAL, "find_triangle: a walk did not end (not a Delaunay triangulation, or a start triangle out of range)");
  return MRD_OK;
}

}  // extern "C"
