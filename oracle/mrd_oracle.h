/* mrd_oracle.h -- C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, step-by-step fp64 implementation of the residual-distribution sweep of
 * arXiv:1705.02028 ("PAPER.md"), written from the paper alone.  It shares no code, header,
 * table or helper with the CUDA path under paper_1705_02028_b200/ and must never be imported,
 * linked or called by it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may use it.
 *
 * All arrays are host memory.  State layout: W[4][nv] (SoA: rho, rho*u, rho*v, e), user numbering.
 */
#ifndef MRD_ORACLE_H
#define MRD_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_mesh orc_mesh;

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_ENONPHYSICAL = -4 };
enum { ORC_SCHEME_N = 0, ORC_SCHEME_LDA = 1, ORC_SCHEME_B = 2, ORC_SCHEME_BMAX = 3, ORC_SCHEME_BMIN = 4 /* L503 */,
       ORC_SCHEME_BX = 5 /* shock-sensor blend, eq. 54-56 L505-L517 */ };

/* Mesh + parameters (PAPER.md L656-L663 mesh arrays; L576 scheme choices; eq. 44 CFL). */
int orc_mesh_create(orc_mesh **out, double gamma, double cfl, int scheme, int time_order,
                    double period_x, double period_y,
                    int64_t n_vertex, const double *xy,          /* [nv][2] */
                    int64_t n_triangle, const int32_t *tri,      /* [nt][3], any orientation */
                    const uint8_t *vertex_flag,                  /* [nv] or NULL; 1 = frozen (L582) */
                    int64_t n_wall_edge, const int32_t *wall_edge /* [ne][2] or NULL (L586) */);
void orc_mesh_destroy(orc_mesh *m);
int orc_set_lumping(orc_mesh *m, int lumping);   /* 0 = global (L576, default), 1 = selective lumping eq. 66-67 */
int orc_set_num_threads(orc_mesh *m, int n);     /* OpenMP threads for the triangle loop (timing only) */
int orc_set_state(orc_mesh *m, const double *W);  /* also records the frozen-vertex values */
int orc_get_state(const orc_mesh *m, double *W);
/* Advance until max_steps steps are done or t reaches t_end (t_end <= 0: ignored). */
int orc_step(orc_mesh *m, int64_t max_steps, double t_end, int64_t *steps_done, double *t, double *dt_last);
int orc_get_diagnostics(const orc_mesh *m, double totals[4], double *min_rho, double *min_p);
/* Geometry as the oracle computed it (for layout tests): area[nt], vol[nv]. */
int orc_get_geometry(const orc_mesh *m, double *area, double *vol);
/* Per-triangle dump of stage 1 at the CURRENT state (no update): phiT[nt][4], phiN/phiLDA/phiB[nt][3][4]
 * (local node order = the order given in `tri`, after any orientation fix), sT[nt]. NULL = skip. */
int orc_dump_stage1(orc_mesh *m, double *phiT, double *phiN, double *phiLDA, double *phiB, double *sT);

/* ---- fine-grained entry points used by the pins in tests/ ---- */
/* App. A: K = l/2*(A nx + B ny) by eq. A2 and K+/- by eq. A10-A25 at the state (u,v,h), unit normal (nx,ny),
 * edge length len. Row-major 4x4 each. */
void orc_euler_matrices(double gamma, double u, double v, double h, double nx, double ny, double len,
                        double K[16], double Kp[16], double Km[16]);
/* Eq. A10-A25 with caller-chosen l_1, l_2, l_3 (L1350: l_k = lambda_k recovers K). */
void orc_euler_matrices_l(double gamma, double u, double v, double h, double nx, double ny,
                          double l1, double l2, double l3, double K[16]);
/* Eq. A7 and the corrected eq. A8 (reading C7): R and R^-1 for a unit normal. */
void orc_eigenvectors(double gamma, double u, double v, double h, double nx, double ny,
                      double R[16], double Rinv[16], double lambda[4]);
/* One triangle, stage 1 (O2-O7): W[3][4] vertex states, xy[3][2] CCW coordinates.
 * Outputs: phiT[4], phiN[3][4], phiLDA[3][4], phiB[3][4], theta[4], sT, Nhat[16], sumKm[16]. Any may be NULL. */
int orc_triangle_stage1(double gamma, const double *W, const double *xy,
                        double *phiT, double *phiN, double *phiLDA, double *phiB, double *theta,
                        double *sT, double *Nhat, double *sumKm);
/* One triangle, stage 2 (O9): Wn[3][4], Ws[3][4] (= W*), dt, stored phiT_n[4], phiN_n[3][4].
 * Outputs PhiT[4], PhiN[3][4], PhiLDA[3][4], PhiB[3][4]. */
int orc_triangle_stage2(double gamma, const double *Wn, const double *Ws, const double *xy, double dt,
                        const double *phiT_n, const double *phiN_n,
                        double *PhiT, double *PhiN, double *PhiLDA, double *PhiB);
/* Lumping used by the NEXT calls of orc_triangle_stage2 on this thread (0 global, 1 selective). */
void orc_triangle_stage2_lumping(int lumping);
/* Wall correction of eq. 68-71 for one edge a->b with OUTWARD unit normal n: out Phi_a[4], Phi_b[4]. */
void orc_wall_edge(double gamma, const double *Wa, const double *Wb, double nx, double ny, double len,
                   double *Phi_a, double *Phi_b);
/* Operation counts of one stage-1 / stage-2 triangle evaluation with a counting scalar type:
 * counts[6] = add/sub, mul, div, sqrt, abs, compare(max/min). */
int orc_count_ops(double gamma, const double *W, const double *xy, int stage, int scheme, int64_t counts[6]);

const char *orc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
