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
       MRD_SCHEME_BMAX = 3, MRD_SCHEME_BMIN = 4 };                   /* B with all Theta_kk = their max / min (L503) */
enum { MRD_FP64 = 0, MRD_FP32 = 1 };

typedef struct mrd_mesh mrd_mesh;     /* opaque: mesh layout + device state + stepper */
typedef struct mrd_layout mrd_layout; /* opaque: host-only result of the mesh-layout stage */

typedef struct {
  double gamma;       /* ratio of specific heats, > 1 (eq. 10)                                  */
  double cfl;         /* dt = cfl * (bound of eq. 44), > 0                                       */
  int32_t scheme;     /* MRD_SCHEME_N | _LDA | _B | _BMAX | _BMIN                                      */
  int32_t time_order; /* 1 = single stage eq. 43 (L437); 2 = RK2 eq. 60-61 (L539-L553)                 */
  int32_t precision;  /* MRD_FP64 | MRD_FP32: arithmetic AND storage type of the sweep                 */
  int32_t reorder;    /* 1 = renumber vertices/triangles along a Morton curve (L669-L675); 0 = keep    */
  double period_x;    /* > 0: periodic in x with this period, coordinates in [0, period); 0 = bounded  */
  double period_y;    /* same for y (L584: periodicity is "handled by the mesh")                       */
  int32_t tile;       /* triangles per thread block of the fused tile kernels: 0 = default (128), or 64, 128; -1 = the unfused kernels (one thread per triangle through
                         global memory, kept for comparison). Results depend on it through summation order
                         only                                                                          */
  int32_t lumping;    /* 0 = global lumping (all tests of the paper, L576); 1 = selective lumping with the Galerkin
                         mass matrix (eq. 66-67), stage 2 of time_order 2 only                        */
} mrd_params;

/* ------------------------------------------------------------------------------------------------
 * Mesh-layout stage (host only, no CUDA).  Makes every triangle counter-clockwise
 * (swapping its 2nd and 3rd vertex when needed), unwraps periodic triangles by minimum image,
 * computes Morton keys (L669-L675) of vertices and triangle centroids, the two renumberings, the
 * vertex -> incident (triangle, local node) CSR in ascending order, the triangle geometry of eq. 35
 * (L397-L399) and the dual volumes V_i = sum |T|/3 (L441, reading C5).
 *   xy   host [nv][2] double   vertexCoordinates  (L656-L663)
 *   tri  host [nt][3] int32    triangleVertices, any orientation
 *   vertex_flag host [nv] uint8 or NULL: 1 = frozen ghost vertex that keeps its initial state (L582)
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

/* Kernel launch counter: number of the library's own kernel launches since the mesh was created. */
int mrd_launch_count(const mrd_mesh *m, int64_t *launches);

const char *mrd_last_error(void);
const char *mrd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MRD_H */
