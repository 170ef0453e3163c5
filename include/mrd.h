/* mrd.h -- C-ABI of the B200-native residual-distribution hydrodynamics sweep.
 *
 * What it computes: the per-time-step sweep over all triangles of an unstructured 2D mesh of the
 * multidimensional upwind (residual distribution) method of arXiv:1705.02028 ("PAPER.md"):
 * Roe-parameter-vector linearisation (eq. 39), inflow matrices K_i^(+/-) (eq. 37-42,
 * App. A), triangle residual (eq. 36), N / LDA / blended B distribution (eq. 48-53), per-vertex
 * accumulation and the two-stage Runge-Kutta update (eq. 60-65), global CFL time step (eq. 44-45),
 * boundary conditions of paragraph 3.5 (L580-L602).  Readings of passages where the paper is silent or
 * garbled are C1-C22 of DESIGN.md.
 *
 * Conventions
 *  - Every function returns MRD_OK (0) or a negative code; mrd_last_error() gives a thread-local
 *    message for the last non-zero return on the calling thread.
 *  - "host" / "device" is stated per pointer.  Device pointers must belong to the CUDA device that
 *    was current when the mesh was created.  `stream` is a cudaStream_t passed as void* (NULL = the
 *    legacy default stream); the library enqueues on it and only synchronises where stated.
 *  - Ownership: the library copies the mesh arrays at create time and owns every device and host
 *    buffer it allocates (cudaMalloc inside mrd_mesh_create, released by mrd_mesh_destroy).  State
 *    buffers passed to set/get are caller-owned and are only touched inside the call (on `stream`).
 *  - State layout at the boundary: W[4][nv], structure of arrays (rho, rho*u, rho*v, e) (eq. 6-11,
 *    L212-L233), USER vertex numbering, element type double (precision 0) or float (precision 1).
 *    The internal (Morton) numbering never leaks, except through the mrd_layout_* test accessors.
 *  - There is no CPU fallback: without a CUDA device mrd_mesh_create fails with MRD_ECUDA.
 */
#ifndef MRD_H
#define MRD_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  MRD_OK = 0,
  MRD_EINVAL = -1,       /* bad argument, index out of range, degenerate triangle, bad wall edge */
  MRD_ENOMEM = -2,       /* host or device allocation failed                                    */
  MRD_ECUDA = -3,        /* CUDA runtime error (string in mrd_last_error)                        */
  MRD_ENONPHYSICAL = -4  /* rho <= 0, p <= 0 or linearised c^2 <= 0 met; state = last good step  */
};
enum { MRD_SCHEME_N = 0, MRD_SCHEME_LDA = 1, MRD_SCHEME_B = 2,      /* eq. 48-49 / 50-51 / 52-53 */
       MRD_SCHEME_BMAX = 3, MRD_SCHEME_BMIN = 4,                     /* B with all Theta_kk = their max / min (L503) */
       MRD_SCHEME_BX = 5 };  /* scalar blend from the shock sensor of eq. 54-56 (L505-L517; readings C23-C26 of DESIGN.md):
                                one more pass over the vertices per stage for |v|_max - |v|_min; on a partitioned mesh
                                the caller reduces that range over all parts (mrd_range_get / mrd_range_set) */
enum { MRD_FP64 = 0, MRD_FP32 = 1 };

typedef struct mrd_mesh mrd_mesh;     /* opaque: mesh layout + device state + stepper */
typedef struct mrd_layout mrd_layout; /* opaque: host-only result of the mesh-layout stage */

typedef struct {
  double gamma;       /* ratio of specific heats, > 1 (eq. 10)                                  */
  double cfl;         /* dt = cfl * (bound of eq. 44), > 0                                       */
  int32_t scheme;     /* MRD_SCHEME_N | _LDA | _B | _BMAX | _BMIN | _BX                                */
  int32_t time_order; /* 1 = single stage eq. 43 (L437); 2 = RK2 eq. 60-61 (L539-L553)                 */
  int32_t precision;  /* MRD_FP64 | MRD_FP32: arithmetic AND storage type of the sweep                 */
  int32_t reorder;    /* 1 = renumber vertices/triangles along a Morton curve (L669-L675); 0 = keep    */
  double period_x;    /* > 0: periodic in x with this period, coordinates in [0, period); 0 = bounded  */
  double period_y;    /* same for y (L584: periodicity is "handled by the mesh")                       */
  int32_t tile;       /* triangles (= threads) per tile of the fused tile kernels: 0 = default (256), or 64, 128, 256; -1 = the
                         unfused kernels (one thread per triangle through global memory, kept for comparison).  Results
                         depend on it through summation order only                                              */
  int32_t lumping;    /* 0 = global lumping (all tests of the paper, L576); 1 = selective lumping with the Galerkin
                         mass matrix (eq. 66-67), stage 2 of time_order 2 only                        */
  double domain_size; /* MRD_SCHEME_BX: "L, the domain size" of eq. 56 (L515; reading C25).  0 = take it from this mesh
                         (larger side of its bounding box, the period where periodic); > 0 = use this value -- a part of
                         a domain decomposition passes the WHOLE mesh's L (mrd_partition_domain_size)            */
} mrd_params;

/* ------------------------------------------------------------------------------------------------
 * Mesh-layout stage (host only, no CUDA).  Makes every triangle counter-clockwise
 * (swapping its 2nd and 3rd vertex when needed), unwraps periodic triangles by minimum image,
 * computes Morton keys (L669-L675) of vertices and triangle centroids, the two renumberings, the
 * vertex -> incident (triangle, local node) CSR in ascending order, the triangle geometry of eq. 35
 * (L397-L399) and the dual volumes V_i = sum |T|/3 (L441, reading C5).
 *   xy   host [nv][2] double   vertexCoordinates  (L656-L663)
 *   tri  host [nt][3] int32    triangleVertices, any orientation
 *   vertex_flag host [nv] uint8 or NULL: 1 = frozen ghost vertex that keeps its initial state (L582);
 *               2 = halo vertex of a partition (see mrd_partition_create)
 *   wall_edge   host [ne][2] int32 or NULL: vertex pairs of edges on reflecting walls (L586-L602);
 *               each must belong to exactly one triangle
 * Errors: MRD_EINVAL (null/empty mesh, index out of range, repeated vertex in a triangle, zero-area
 * triangle, vertex without triangle, bad/duplicate wall edge), MRD_ENOMEM.
 * ---------------------------------------------------------------------------------------------- */
int mrd_layout_create(mrd_layout **out, const mrd_params *p, int64_t n_vertex, const double *xy,
                      int64_t n_triangle, const int32_t *tri, const uint8_t *vertex_flag,
                      int64_t n_wall_edge, const int32_t *wall_edge);
void mrd_layout_destroy(mrd_layout *l);
/* Sizes: n[0]=nv, n[1]=nt, n[2]=n_wall_edge, n[3]=n_frozen, n[4]=n_tiles, n[5]=n_tile_slots (host out). */
int mrd_layout_sizes(const mrd_layout *l, int64_t n[6]);
/* Test accessors (host out; any pointer may be NULL):
 *   vperm[nv]: user index of internal vertex k        tperm[nt]: user index of internal triangle k
 *   tri_int[nt][3]: internal connectivity (internal vertex ids, CCW)
 *   csr_off[nv+1], csr_ent[3 nt]: incidence, entries = internal_triangle*3 + local_node, ascending
 *   area[nt], vol[nv]: |T| and V_i in INTERNAL numbering */
int mrd_layout_get(const mrd_layout *l, int32_t *vperm, int32_t *tperm, int32_t *tri_int,
                   int32_t *csr_off, int32_t *csr_ent, double *area, double *vol);

/* ------------------------------------------------------------------------------------------------
 * Mesh object = layout stage + upload to the current CUDA device + all device workspace.
 * Arguments as mrd_layout_create.  Additional errors: MRD_ECUDA (no device / CUDA failure).
 * ---------------------------------------------------------------------------------------------- */
int mrd_mesh_create(mrd_mesh **out, const mrd_params *p, int64_t n_vertex, const double *xy,
                    int64_t n_triangle, const int32_t *tri, const uint8_t *vertex_flag,
                    int64_t n_wall_edge, const int32_t *wall_edge);
void mrd_mesh_destroy(mrd_mesh *m);
/* Device bytes held by the mesh (host out). */
int mrd_mesh_device_bytes(const mrd_mesh *m, int64_t *bytes);

/* Set the state W^n and t = 0; also records the values kept by frozen vertices (L582).
 *   W  DEVICE [4][nv] SoA, user numbering, double or float per params.precision.
 * Enqueued on `stream`; synchronises the stream before returning (positivity of the state is
 * checked: MRD_ENONPHYSICAL if some rho <= 0 or p <= 0). */
int mrd_set_state(mrd_mesh *m, const void *W_dev, void *stream);
/* Same with W in HOST memory (pageable or pinned); the copy is part of the call. */
int mrd_set_state_host(mrd_mesh *m, const void *W_host, void *stream);
/* Read the current state into W_out (DEVICE [4][nv] SoA, user numbering). Enqueued; not synchronised. */
int mrd_get_state(mrd_mesh *m, void *W_out_dev, void *stream);
/* Same into HOST memory; synchronises the stream before returning. */
int mrd_get_state_host(mrd_mesh *m, void *W_out_host, void *stream);

/* Advance in time: repeat the step of eq. 43 (time_order 1) or eq. 60-61 (time_order 2), each with
 * dt from eq. 44-45 computed on the device from W^n, until `max_steps` steps are done or, when
 * t_end > 0, t reaches t_end (the last dt is clipped to land on it, reading C13).
 * All kernels are enqueued on `stream`; the call synchronises the stream before returning and then
 * writes the host scalars (any may be NULL): steps_done, t (time reached), dt_last.
 * MRD_ENONPHYSICAL: the step that met it is discarded and the state left at the last good step. */
int mrd_step(mrd_mesh *m, int64_t max_steps, double t_end, void *stream, int64_t *steps_done,
             double *t, double *dt_last);
/* As mrd_step without the final synchronisation and without host outputs (for timing loops and
 * overlap); t_end is not supported here.  Errors surface at the next synchronising call. */
int mrd_step_async(mrd_mesh *m, int64_t n_steps, void *stream);
/* Synchronise `stream` and fetch the counters kept on the device (host out, any may be NULL). */
int mrd_sync(mrd_mesh *m, void *stream, int64_t *steps_total, double *t, double *dt_last);

/* Diagnostics of the current state: totals[k] = sum_i V_i W_k,i (conservation,
 * L455), min rho, min p. Synchronises the stream. Deterministic (fixed reduction order). */
int mrd_get_diagnostics(mrd_mesh *m, double totals[4], double *min_rho, double *min_p, void *stream);

/* Per-triangle stage-1 quantities at the CURRENT state, no update (parity of SURVEY 8a S2-S6 against
 * the oracle): HOST out, USER triangle numbering, local node order = the order given in `tri`
 * after the orientation fix; any pointer may be NULL.
 *   phiT[nt][4] (eq. 36)  phiN[nt][3][4] (eq. 48)  phiLDA[nt][3][4] (eq. 50)  phiB[nt][3][4]
 *   (eq. 52; = phiN / phiLDA for scheme N / LDA)  sT[nt] (eq. 45 times l_max).  Always double. */
int mrd_dump_stage1(mrd_mesh *m, double *phiT, double *phiN, double *phiLDA, double *phiB, double *sT,
                    void *stream);

/* As mrd_dump_stage1 for a SAMPLE of triangles (full-size meshes): tri_user[n_sample] HOST user triangle ids;
 * outputs are HOST arrays indexed by sample: phiT[n][4], phiN/phiLDA/phiB[n][3][4], sT[n]; any may be NULL. */
int mrd_dump_stage1_sample(mrd_mesh *m, int64_t n_sample, const int64_t *tri_user, double *phiT, double *phiN,
                           double *phiLDA, double *phiB, double *sT, void *stream);

/* Micro-benchmarks of the device the roofline is quoted against (host out, any may be NULL):
 * dependent-chain-free DFMA and FFMA loops (TFLOP/s, 2 flops per FMA) and a device-to-device copy
 * (GB/s, read + write bytes). Synchronises. */
int mrd_measure_peaks(double *fp64_tflops, double *fp32_tflops, double *copy_gbs, void *stream);

/* One time step with a CUDA event after every kernel launch (on `stream`): ms[k] = device time of the
 * kernel(s) in slot k of this step, 0 for kernels the configuration does not launch. Synchronises.
 * Used by bench.py for the live per-kernel durations of the roofline object. */
enum {
  MRD_PROF_TRI1 = 0,          /* triangle kernel, stage 1 (S2-S6)                 */
  MRD_PROF_GATHER_DT = 1,     /* vertex gather + CFL minimum (S7, S8 first half)  */
  MRD_PROF_WALL1 = 2,         /* wall terms, stage 1 (S11)                        */
  MRD_PROF_UPDATE = 3,        /* vertex update W* (S8) or W^{n+1} (S12)           */
  MRD_PROF_TRI2 = 4,          /* triangle kernel, stage 2 (S9)                    */
  MRD_PROF_WALL2 = 5,         /* wall terms, stage 2                              */
  MRD_PROF_GATHER_UPDATE = 6, /* vertex gather + update W^{n+1} (S10)             */
  MRD_PROF_CTL = 7,           /* step control (dt, t, counters)                   */
  MRD_PROFILE_SLOTS = 8
};
int mrd_step_profile(mrd_mesh *m, void *stream, float ms[MRD_PROFILE_SLOTS]);

/* ------------------------------------------------------------------------------------------------
 * Domain decomposition for several GPUs (the paper ran on one device and names no scheme, so
 * this is this library's own: owner-computes over contiguous ranges of the vertices' Morton order,
 * L669-L675).  Part `part` of `n_part` OWNS the vertices of its range, holds every triangle incident to
 * an owned vertex (triangles cut by the partition are held and recomputed by each side: no residual is
 * exchanged) and, as HALO vertices, the other vertices of those triangles.  One exchange of vertex states
 * per stage (after eq. 60 and after eq. 61 / 43) and one min-reduction of a double per step (eq. 44)
 * keep every part's copy equal to the single-device run up to summation order.
 *
 * mrd_partition_create (host only, no CUDA): arguments as mrd_layout_create plus the periods; the global
 * mesh is given in full to every part.  Errors: MRD_EINVAL (as the layout stage; vertex_flag other than
 * 0/1; n_part < 1; part out of range; a part without vertices), MRD_ENOMEM.
 * mrd_partition_sizes: n[0] = local vertices (owned first, then halo; each group in ascending global id),
 *   n[1] = owned vertices, n[2] = local triangles (ascending global id), n[3] = local wall edges,
 *   n[4] = neighbour parts, n[5] = vertices sent per exchange, n[6] = vertices received per exchange,
 *   n[7] = global vertices.
 * mrd_partition_get(name, dst host, bytes = exact size of the array; MRD_EINVAL otherwise):
 *   "vertex_global" int32[n0]    global id of each local vertex
 *   "xy"            double[n0][2]
 *   "tri"           int32[n2][3] local vertex ids, node order of the global triangle
 *   "tri_global"    int32[n2]
 *   "vertex_flag"   uint8[n0]    0 free, 1 frozen (L582), 2 halo  -> pass to mrd_mesh_create
 *   "wall_edge"     int32[n3][2] local ids (wall edges with an owned end)
 *   "neighbour"     int32[n4]    ascending part ids
 *   "send_off"      int32[n4+1], "send_idx" int32[n5]: owned local vertices whose state neighbour k needs,
 *   "recv_off"      int32[n4+1], "recv_idx" int32[n6]: halo local vertices owned by neighbour k; both lists
 *                   ascending in global id per neighbour, so that send list of a for b == recv list of b from a
 *   "owner"         int32[n7]    owning part of every global vertex (empty, 0 bytes, for mrd_partition_create_local)
 * ---------------------------------------------------------------------------------------------- */
typedef struct mrd_partition mrd_partition;
int mrd_partition_create(mrd_partition **out, int64_t n_vertex, const double *xy, int64_t n_triangle,
                         const int32_t *tri, const uint8_t *vertex_flag, int64_t n_wall_edge,
                         const int32_t *wall_edge, double period_x, double period_y, int32_t n_part, int32_t part);
/* As mrd_partition_create with the owning part of every vertex given by the caller (owner: host int32[n_vertex], values in
 * [0, n_part)) instead of the Morton ranges: any decomposition into connected pieces works the same way. */
int mrd_partition_create_owned(mrd_partition **out, int64_t n_vertex, const double *xy, int64_t n_triangle,
                               const int32_t *tri, const uint8_t *vertex_flag, int64_t n_wall_edge,
                               const int32_t *wall_edge, double period_x, double period_y, int32_t n_part, int32_t part,
                               const int32_t *owner);
/* The same part assembled from LOCAL pieces, for meshes whose arrays should never exist in full on one host (the start-up of an
 * N-GPU run then costs each rank its own share only).  The caller passes the vertices and triangles it knows -- at least every
 * triangle incident to a vertex owned by `part`, with all three vertices of each -- and for each vertex its global id and
 * owning part (all host arrays, copied):
 *   vertex_global int32[n_local_vertex]   global vertex ids (unique, any order), < n_vertex_global
 *   owner         int32[n_local_vertex]   owning part of each of these vertices
 *   xy            double[n_local_vertex][2];  vertex_flag uint8[n_local_vertex] or NULL (0 free, 1 frozen)
 *   tri           int32[n_local_triangle][3]  indices INTO the arrays above;  tri_global int32[n_local_triangle] global triangle ids
 *   wall_edge     int32[n_wall_edge][2] or NULL, indices into the arrays above
 *   domain_size   L of eq. 56 of the whole mesh (reading C25; only MRD_SCHEME_BX uses it)
 * Triangles without a vertex of `part` and vertices used by no kept triangle are dropped.  The result is what
 * mrd_partition_create_owned gives for the whole mesh with the same owners (same local numbering, same exchange lists:
 * they are sorted by global id), except that "owner" (a whole-mesh array) is empty.  Errors as mrd_partition_create. */
int mrd_partition_create_local(mrd_partition **out, int64_t n_vertex_global, double domain_size, int64_t n_local_vertex,
                               const int32_t *vertex_global, const int32_t *owner, const double *xy, const uint8_t *vertex_flag,
                               int64_t n_local_triangle, const int32_t *tri, const int32_t *tri_global, int64_t n_wall_edge,
                               const int32_t *wall_edge, int32_t n_part, int32_t part);
void mrd_partition_destroy(mrd_partition *p);
int mrd_partition_sizes(const mrd_partition *p, int64_t n[8]);
/* L of eq. 56 (reading C25) of the WHOLE mesh the partition was made from (host out): goes into the
 * mrd_params.domain_size of every part's mesh, so that the Bx sensor is the same on all parts and on one device. */
int mrd_partition_domain_size(const mrd_partition *p, double *L);
int mrd_partition_get(const mrd_partition *p, const char *name, void *dst, int64_t bytes);

/* Halo lists of a mesh created from a partition (vertex_flag 2 = halo: such a vertex keeps its value in
 * the updates like a frozen one, is left out of the minimum of eq. 44 and of the totals of
 * mrd_get_diagnostics, and gets its value from mrd_halo_unpack).  send_idx / recv_idx: HOST int32 lists
 * of USER (= partition-local) vertex ids, copied; recv_idx must name halo vertices only (MRD_EINVAL). */
int mrd_halo_set(mrd_mesh *m, int64_t n_send, const int32_t *send_idx, int64_t n_recv, const int32_t *recv_idx);

/* One time step in phases, for a caller that exchanges between them (all enqueued on `stream`; none
 * synchronises except begin/end).  Sequence per step, the same on every part:
 *   mrd_phase(RESIDUAL1)   stage-1 triangle pass, wall terms, local min of 2 V_i / sum s_T (eq. 44-45)
 *   mrd_dt_get -> min-reduce the two doubles over all parts -> mrd_dt_set
 *   mrd_phase(UPDATE1)     eq. 60 (time_order 2) or eq. 43 (time_order 1) on the owned vertices
 *   mrd_halo_pack -> exchange -> mrd_halo_unpack
 *   time_order 2 only: mrd_phase(STAGE2) (stage-2 triangle pass, eq. 61 on the owned vertices), then
 *   mrd_halo_pack -> exchange -> mrd_halo_unpack
 *   mrd_status_get -> max-reduce the double over all parts -> mrd_status_set
 *   mrd_phase(END)         advance t, count the step -- or discard it on EVERY part if any part met rho <= 0, p <= 0 or
 *                          c^2 <= 0 anywhere in it
 * mrd_phase_begin settles earlier asynchronous work, arms the stepper and sets t_end (<= 0: none; every part
 * must pass the same); mrd_phase_end synchronises and reports like mrd_step (steps_done counts the steps since
 * mrd_phase_begin).  With the status reduction every part commits or discards the same steps, so (steps, t, error code)
 * are identical on all parts and the state is left at the last good step everywhere (MRD_ENONPHYSICAL), as in mrd_step. */
enum { MRD_PHASE_RESIDUAL1 = 0, MRD_PHASE_UPDATE1 = 1, MRD_PHASE_STAGE2 = 2, MRD_PHASE_END = 3 };
int mrd_phase_begin(mrd_mesh *m, double t_end, void *stream);
int mrd_phase(mrd_mesh *m, int32_t phase, void *stream);
int mrd_phase_end(mrd_mesh *m, void *stream, int64_t *steps_done, double *t, double *dt_last);
/* d DEVICE double[2]: d[0] = local min_i 2 V_i / sum s_T over non-halo vertices, d[1] = -1 if this part met a
 * non-physical state, else 0.  After the min-reduction, mrd_dt_set installs both. */
int mrd_dt_get(mrd_mesh *m, double *d_dev, void *stream);
int mrd_dt_set(mrd_mesh *m, const double *d_dev, void *stream);
/* d DEVICE double[1]: 1 if this part met a non-physical state in the step in flight, else 0.  Call both after the last
 * exchange of the step and before mrd_phase(END); between them, max-reduce the double over all parts. */
int mrd_status_get(mrd_mesh *m, double *d_dev, void *stream);
int mrd_status_set(mrd_mesh *m, const double *d_dev, void *stream);
/* buf DEVICE [n_send][4] / [n_recv][4] (double or float per precision), rows in list order: the conserved
 * state just written by the preceding UPDATE1 / STAGE2 phase.  Unpack also derives what the triangle kernels
 * read (Z, and dW/dt of eq. 57 or |v| + c) exactly as the owner did, so halo copies are bitwise the owner's. */
int mrd_halo_pack(mrd_mesh *m, void *buf_dev, void *stream);
/* MRD_SCHEME_BX in phases: the sensor of eq. 56 needs |v|_max - |v|_min over the WHOLE mesh (reading C24).
 * mrd_range_get: d DEVICE double[2] = (|v|_max, -|v|_min) over this part's vertices (halo copies included: they are
 * some part's vertices) of the state that stage `stage` reads -- stage 1: W^n, call after mrd_phase_begin and after
 * every mrd_phase(END); stage 2: W*, call after the halo unpack that follows mrd_phase(UPDATE1).  After a
 * max-reduction of both doubles over all parts, mrd_range_set installs the result for that stage. */
int mrd_range_get(mrd_mesh *m, int32_t stage, double *d_dev, void *stream);
int mrd_range_set(mrd_mesh *m, int32_t stage, const double *d_dev, void *stream);
int mrd_halo_unpack(mrd_mesh *m, const void *buf_dev, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Mesh generation, first slice (section 2.4, and 4.1.3, L665-L667): the kernels that open
 * every iteration of the parallel Delaunay refinement, and the exact predicates the rest of it rests on.  Bounded meshes
 * (no periodic unwrap).  All arrays are DEVICE arrays of the current device; the calls synchronise `stream`.
 *
 * mrd_meshgen_test_quality: for every triangle (a, b, c) = tri[t] of the counter-clockwise mesh
 *   r[t]     circumradius, eq. 2 (L146): l_a l_b l_c / (2 det), det the determinant of eq. 3
 *   beta[t]  r / shortest edge (L120: 2 beta = 1 / sin(smallest angle))
 *   cc[t]    circumcentre, where the refinement inserts the new vertex (L150); double[nt][2]
 *   bad[t]   1 if r > R (too big) or beta > B (low quality) (L150), or det <= 0 (not counter-clockwise); uint8
 *   n_bad    HOST out (may be NULL): number of flagged triangles
 *   xy double[nv][2], tri int32[nt][3].  Every operation is a single IEEE round-to-nearest operation in a fixed order: the
 *   results are reproducible bit for bit (oracle/meshgen.py evaluates the same sequence).
 * mrd_meshgen_orient2d / _incircle2d: the SIGN (+1, 0, -1; int8) of the determinants of eq. 3 (L160: positive when a, b, c are
 *   counter-clockwise) and eq. 5 (L198: positive when d lies inside the circle through the counter-clockwise a, b, c), EXACT
 *   for any double coordinates: a floating-point filter with a rigorous error bound, then exact expansion arithmetic for the
 *   tests it cannot decide (L166, L206: "we need the test to give the exact result").  idx int32[n][3] / [n][4]: vertex
 *   numbers of (a, b, c[, d]) of each test; n_exact HOST out (may be NULL): how many tests needed the exact path.
 * Errors: MRD_EINVAL (null pointer, non-positive R or B), MRD_ENOMEM, MRD_ECUDA.
 * ---------------------------------------------------------------------------------------------- */
int mrd_meshgen_test_quality(int64_t n_triangle, const double *xy_dev, const int32_t *tri_dev, double R, double B,
                             double *r_dev, double *beta_dev, double *cc_dev, uint8_t *bad_dev, int64_t *n_bad, void *stream);
int mrd_meshgen_orient2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream);
int mrd_meshgen_incircle2d(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact, void *stream);

/* mrd_meshgen_orient2d_static: mrd_meshgen_orient2d for callers that must not allocate (code under CUDA graph capture, tight
 *   serving loops, harnesses that forbid cudaMalloc).  Same kernels, same result (the exact sign of eq. 3 for every row of
 *   idx), but the scratch -- the list of tests the filter cannot decide and its length -- lives in a file-scope
 *   `static __device__` array of the library: 4 MB + 256 B on every GPU that loads the library, held until the process exits.
 *   The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it ENQUEUES its work on `stream` and
 *   returns without synchronising (errors of the kernels themselves surface at the caller's next synchronisation).
 *   Limit: n <= 1 048 576 tests per call; a larger n is rejected with MRD_EINVAL and a message that says so.
 *   n_exact_dev: DEVICE out (int64, may be NULL): how many tests needed the exact path.
 *   All calls on one device share the array, which keeps the contents of the last call (the call clears the one word that
 *   must start at zero): two calls that overlap on the GPU (different streams, or graphs launched concurrently) RACE --
 *   order them on one stream or with events.  The device address of the array is taken once per device
 *   (cudaGetSymbolAddress, with that device current); devices 0-63.
 * Errors: MRD_EINVAL (null pointer, n beyond the limit, device number beyond 63), MRD_ECUDA. */
int mrd_meshgen_orient2d_static(int64_t n, const double *xy_dev, const int32_t *idx_dev, int8_t *sign_dev, int64_t *n_exact_dev,
                                void *stream);

/* ------------------------------------------------------------------------------------------------
 * Mesh generation, second slice: the mesh data structure of section 4.1.2 (L656-L663), the Delaunay triangulator of
 * section 2.4.6 (L186-L208) / 4.1.5 (L677-L681), and the search for the triangle that contains a new vertex (section 2.4.2,
 * L152-L168).  Bounded meshes; all arrays DEVICE arrays of the current device; the calls synchronise `stream`.
 *
 * Data structure (the paper's four arrays): xy double[nv][2] (vertexCoordinates), tv int32[nt][3] (triangleVertices,
 * counter-clockwise), te int32[nt][3] (triangleEdges), et int32[ne][2] (edgeTriangles).  Conventions the paper leaves open:
 * edge k of a triangle is the one OPPOSITE its local vertex k (it joins local vertices k+1 and k+2); a boundary edge (a
 * segment, L663) has -1 as its second triangle.
 *
 * mrd_meshgen_build_edges: te and et from tv.  Edges are numbered in ascending order of (smaller vertex, larger vertex); et
 *   lists the two neighbours in ascending triangle order.  et_dev must hold 3 * n_triangle pairs (the upper bound); *n_edge
 *   (HOST out) receives the number of edges.  MRD_EINVAL if an edge belongs to more than two triangles.
 * mrd_meshgen_delaunay_flip: transforms the valid triangulation (tv, te, et), IN PLACE, into the Delaunay triangulation of its
 *   vertices by edge flips ("start with any valid triangulation, and perform edge flips until all edges are locally Delaunay",
 *   L112).  Per iteration (section 4.1.5): the exact INCIRCLE2D test of eq. 5 on every edge whose containing quadrilateral
 *   changed (all edges in the first iteration) lists the edges that are not Delaunay; of those, an independent set -- no two in
 *   the same triangle; the higher edge number wins a contested triangle -- is flipped in parallel; edgeTriangles of the edges
 *   that change sides is repaired in the same pass.  A flipped edge keeps its number and its two triangles: with a opposite E
 *   in t1 = (a, b, c) and d opposite E in t2 = (d, c, b), t1 becomes (a, b, d) and t2 (a, d, c).  Edges with INCIRCLE2D = 0
 *   (four cocircular vertices) are left alone.  The result is unique as a set of triangles when no four vertices are
 *   cocircular (L96), and deterministic (bitwise the same arrays on every run) in any case.
 *   HOST outs (may be NULL): n_flips, n_iterations, n_exact (INCIRCLE2D tests that needed the exact path).
 *   MRD_EINVAL when a triangle of the input is clockwise or degenerate (exact ORIENT2D <= 0), when te and et disagree, or when
 *   the two triangles of an edge run along it in the same direction (they lie on the same side: an overlap): not a valid
 *   triangulation, and flips on it need not end or keep the structure.  (What is not checked: overlaps of triangles that share
 *   no edge.)
 * mrd_meshgen_find_triangle: for every point p[i] (double[n][2]) the triangle that contains it, by walking from t0[i] across
 *   the first edge -- tried in the order (a, b), (b, c), (c, a) -- that has p strictly on its outer side (exact ORIENT2D,
 *   eq. 3).  t[i] >= 0: found, with code[i] = 0 strictly inside, 1 + k on edge k of t, 4 + k on local vertex k (L168);
 *   t[i] = -1 - t_last: the walk left the triangulation through a boundary edge of t_last.  The walk terminates on Delaunay
 *   triangulations; MRD_EINVAL if a walk exceeds n_triangle + 16 steps (not a Delaunay triangulation).
 * Work space: the mrd_meshgen_* calls keep one device block (grown on demand) and a small pinned host block between calls,
 *   because allocating them costs more than the kernels; calls are serialised by a lock.  Size: 182 MB for the scratch of the
 *   exact predicates, plus about 40 bytes per edge for build_edges / delaunay_flip, plus -- for mrd_meshgen_refine -- about 0.9 KB
 *   per vertex of CAPACITY (sort buffers, candidate records, cavity pool, renumbering maps: 1.8 GB for cap_vertex = 2.1 M).
 *   mrd_meshgen_release frees both blocks (they come back on the next call).
 * Errors: MRD_EINVAL (null pointer, inconsistent structure), MRD_ENOMEM, MRD_ECUDA.
 * ---------------------------------------------------------------------------------------------- */
int mrd_meshgen_release(void);
/* Diagnostics of the flip loops (mrd_meshgen_delaunay_flip and the flips inside mrd_meshgen_refine) of this process since the last
 * reset.  Candidate sets of at most 65 536 edges run check -> flip -> check ... in ONE cooperative launch with grid-wide
 * barriers; that launch can evaluate INCIRCLE2D exactly only when the six translations of the test are exact, and hands an
 * iteration that meets another test back to the kernels with the long expansions.  stats (HOST out, may be NULL):
 * [0] cooperative launches, [1] iterations run inside them, [2] iterations handed back, [3] iterations run launch by launch. */
int mrd_meshgen_flip_stats(int64_t stats[4], int reset);
int mrd_meshgen_build_edges(int64_t n_triangle, const int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev, int64_t *n_edge,
                            void *stream);
int mrd_meshgen_delaunay_flip(int64_t n_triangle, int64_t n_edge, const double *xy_dev, int32_t *tv_dev, int32_t *te_dev,
                              int32_t *et_dev, int64_t *n_flips, int64_t *n_iterations, int64_t *n_exact, void *stream);
int mrd_meshgen_find_triangle(int64_t n_point, const double *p_dev, const int32_t *t0_dev, int64_t n_triangle,
                              const double *xy_dev, const int32_t *tv_dev, const int32_t *te_dev, const int32_t *et_dev,
                              int32_t *t_dev, int8_t *code_dev, void *stream);

/* ------------------------------------------------------------------------------------------------
 * Mesh generation, third slice: Delaunay refinement of a bounded domain (section 2.3-2.4) with the parallel insertion
 * set of section 4.1.1 (L634-L654).  The boundary edges of the input triangulation are the segments (L128-L140).
 *
 * mrd_meshgen_refine: repeats, at most max_iterations times and until no triangle is bad,
 *   1. TestQuality (eq. 2): every triangle with circumradius r > R or r / shortest edge > B is bad; its circumcentre is a
 *      candidate vertex (2.4.1).  The size bound may vary in space (section 2.3.1): with size_dev (DEVICE, double
 *      [size_ny][size_nx], row-major, all > 0: factors at the points of a regular grid over the rectangle size_box =
 *      (x0, y0, x1, y1), HOST) the bound is R * f(circumcentre), f the bilinear interpolant of the grid (the nearest rim value
 *      outside the rectangle), evaluated one IEEE operation at a time: fx = min(max((x - x0) * ((nx - 1) / (x1 - x0)), 0),
 *      nx - 1), i = min(floor(fx), nx - 2), tx = fx - i (likewise y); f = (g[j][i] (1 - tx) + g[j][i+1] tx) (1 - ty) +
 *      (g[j+1][i] (1 - tx) + g[j+1][i+1] tx) ty.  size_dev = NULL: f = 1.  Termination needs f >= some M > 0 (L126);
 *   2. the triangle containing the candidate, by the walk of mrd_meshgen_find_triangle from the bad triangle (2.4.2).  A
 *      candidate outside the triangulation becomes the midpoint of the segment the walk left through; one on a segment the
 *      midpoint of that segment; one that coincides with a vertex is dropped;
 *   3. encroachment (2.4.3, eq. 4 in plain IEEE arithmetic): against the segments of all triangles that have a vertex of the
 *      insertion triangle(s) as a vertex; a candidate that encroaches becomes the midpoint of the encroached segment with
 *      the lowest edge number;
 *   4. the cavity of every candidate -- the triangles whose circumcircles contain it (exact INCIRCLE2D), reached from the
 *      insertion triangle(s) through shared edges -- claims its triangles with the candidate's priority i(v) (atomicMax, L648);
 *      a candidate is selected when it holds all of them (4.1.1).  i(v) = mix32(seed, iteration, bad triangle) * 2^32 + bad
 *      triangle; mix32(x): x ^= x >> 15, x *= 2246822519, x ^= x >> 13, x *= 3266489917, x ^= x >> 16 on
 *      x = t * 2654435761 + iteration * 40503 + seed (mod 2^32).  seed = MRD_MESHGEN_PRIORITY_REGULAR selects the paper's
 *      "regular integer assignment" i(v) = bad triangle instead (L654, Fig. 8: many more iterations on a Morton-ordered mesh;
 *      for comparison only).  A cavity may be of any size (a start mesh of slivers has cavities of most of its triangles): up to
 *      64 triangles are kept in a per-thread list, a larger cavity is walked along its outline without a list, which relies on
 *      the input being a Delaunay triangulation (its cavities are trees; a walk that does not close makes the candidate wait);
 *   5. the selected vertices are inserted (2.4.4: a triangle split in three, the two triangles at an edge split in two each, the
 *      one triangle at a segment split in two), numbered -- like their new triangles and edges -- in ascending order of
 *      their bad triangle;
 *   6. flips restore the Delaunay property (2.4.6);
 *   7. numbering.  With `box` = (x0, y0, x1, y1) (HOST, the rectangle the domain lies in) every iteration ends with the
 *      re-sort of 4.1.4: the vertices are renumbered in ascending Morton value -- 21 bits per coordinate,
 *      i = min(2^21 - 1, floor((x - x0) * (2^21 / (x1 - x0)))), x in the even bit places, ties keep their order -- and xy, tv
 *      follow; then the triangles are renumbered canonically (each rotated to its smallest vertex, sorted by vertex triple:
 *      along the same curve) and te, et rebuilt as by mrd_meshgen_build_edges.
 *      With box = NULL the vertices keep their numbers (input vertices first, inserted ones in order of insertion) and the
 *      iterations renumber IN PLACE: a triangle or edge that survives an iteration keeps its number (and rotation); the
 *      numbers of those that did not, and the new numbers at the end, go to the triangles / edges the iteration created,
 *      in ascending order of their vertex triple / pair of end points.  ONE canonical re-sort (as above, without the
 *      vertices) follows the last iteration of the call, whatever ended it.
 *   Every step is deterministic and independent of the order in which threads run: the result is, array for array, the one
 *   of oracle/meshgen.py: refine.
 *   In: a Delaunay triangulation (xy, tv, te, et) with *n_vertex, *n_triangle, *n_edge entries in device arrays with room
 *   for cap_vertex / cap_triangle / cap_edge (cap_edge >= 3 * cap_triangle); first_iteration: the iteration number the
 *   priorities start from.  Out: the refined mesh in the same arrays, the three counts, *n_iterations (iterations that
 *   inserted vertices), *n_bad_left (bad triangles remaining: 0 when finished).  HOST pointers for all counts.
 *   Guarantees on completion (section 2.3): no triangle with r > R or beta > B, hence no angle below arcsin(1 / 2B); Delaunay;
 *   no encroached segment.  Termination is guaranteed for B >= sqrt(2) and domains without small angles (L126).
 *   MRD_ENOMEM when the next insertion would exceed a capacity (the arrays then hold a valid Delaunay mesh, partly
 *   refined); MRD_EINVAL for an input with a clockwise or degenerate triangle or a vertex number out of range, or edge tables
 *   that do not describe a triangulation (as for mrd_meshgen_delaunay_flip; all checked first), or one that is not a Delaunay
 *   triangulation (a walk that does not end).
 * ---------------------------------------------------------------------------------------------- */
#define MRD_MESHGEN_PRIORITY_REGULAR 0xFFFFFFFFu
int mrd_meshgen_refine(double R, double B, uint32_t seed, int64_t first_iteration, int64_t max_iterations, const double *box,
                       const double *size_dev, const double *size_box, int64_t size_nx, int64_t size_ny, int64_t cap_vertex,
                       int64_t cap_triangle, int64_t cap_edge, int64_t *n_vertex, int64_t *n_triangle, int64_t *n_edge,
                       double *xy_dev, int32_t *tv_dev, int32_t *te_dev, int32_t *et_dev, int64_t *n_iterations,
                       int64_t *n_bad_left, void *stream);

/* Kernel launch counter: number of the library's own kernel launches since the mesh was created. */
int mrd_launch_count(const mrd_mesh *m, int64_t *launches);

const char *mrd_last_error(void);
const char *mrd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MRD_H */
