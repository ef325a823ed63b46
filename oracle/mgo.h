/* mgo.h -- CPU ORACLE for the variable-density pressure-Poisson multigrid V-cycle.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code,
 * header, table or helper with the CUDA path (paper_2605_30082_b200/csrc, include/mg.h).
 *
 * What it computes (citations: BJ = BASELINE.json north_star/configs, P:NNN = PAPER.md
 * line, Rn / Cn = SURVEY.md 8(c) readings and canonical arithmetic, restated in DESIGN.md):
 *
 *   A p = f,  (A p)_c = (1/h^2) * sum_{6 faces} beta_face * (p_nb - p_c)        [BJ; R1]
 *   the discrete form of  div( (1/rho) grad p ) = div(u*)/dt  implied by P:33-36 eq. 1-2,
 *   cell-centred on a uniform Cartesian finite-volume grid, dense (i,j,k) arrays
 *   with x fastest (R3), density per cell by volume-fraction mixing.
 *   beta_face = 1/rho_face with rho_face the harmonic mean of the two cell densities
 *             = (0.5/rho_a) + (0.5/rho_b)                                       [BJ; R4, C2]
 *   per axis: periodic (wrap) or homogeneous Neumann (wall-face beta = 0)       [R5]
 *   per side (mgo_create6): also Dirichlet walls, p = 0 on the wall face        [R24]
 *   solved by geometric multigrid V(nu1,nu2) cycles: red-black Gauss-Seidel, residual,
 *   8-child-mean restriction, cell-centred trilinear prolongation + correction,
 *   coarse faces = mean of the 4 coincident fine faces, 4^3-ish coarsest level
 *   relaxed with a fixed number of sweeps                                       [BJ; R7-R15]
 *
 * It is an iteration, so the oracle follows the algorithm step by step in the order
 * and with the expression trees C1-C9 (no blocking, fusion or reordering).  Every level
 * stores explicit minus-face arrays bx,by,bz (bx[i,j,k] = face between (i-1,j,k) and
 * (i,j,k); entry 0 of a non-periodic axis is the minus wall) and plus-wall arrays wx,wy,wz;
 * the neighbour value beyond any wall is 0.0 (C2).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form eigenvalues of sine/cosine
 * modes, symmetry / zero row+column sums, the layered-medium prefix-sum solution,
 * second-order convergence on a manufactured solution, a dense direct solve at 8^3,
 * smoother and transfer invariants, config 1's known solution.
 * The coarse-face rule C3 is pinned value by value against numpy slices of the finer level's
 * faces on a fully 3-D random density (test_coarse_faces_brute_force_3d); the coarsest-level
 * sweep count against a one-level hierarchy (test_coarsest_level_runs_exactly_coarse_sweeps_sweeps).
 * F- and W-cycles (R23): recursion over the pinned single steps bit for bit, visit counts, dense
 * 16^3 solve (test_oracle_cycles.py).  Dirichlet walls (R24): closed-form eigenmodes of all side
 * pairs, wall values and sides, coarse walls by brute force, layered medium with a Dirichlet top,
 * dense non-singular solve, ghost weights, second-order convergence (test_oracle_bc6.py).
 * MG-preconditioned CG (R22): adjoint identity, symmetry of M, dense solve (test_oracle_pcg.py).
 * Projection steps (R21): linear fields, Gauss theorem, div(u_new)/dt = f - A p (test_oracle_projection.py).
 * mgo_solve's control (R15): r_0 and hist[0] from the incoming p != 0, every hist[k] replayed through
 * apply, stop at the first k below rtol r_0, statuses for max_cycles = 0 and r_0 = 0
 * (test_solve_measures_r0_from_the_incoming_p).
 * PARITY UNPINNED (CHOICES among readings on which the paper is silent, not functions: what
 * the code computes under each choice is pinned): that R8 is the 4-face mean,
 * that R13's default is 32 sweeps, that R11 is the 8-child mean among the "full-weighting"
 * readings, R18 (sphere position in the input recipe), R21's staggering convention, R22's
 * symmetric coarsest solve, R24's reading of "continuous" planes as p = 0 on the wall face.
 *
 * All pointers are HOST pointers to dense fp64 arrays, idx = i + nx*(j + ny*k).
 */
#ifndef MGO_H
#define MGO_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mgo_solver mgo_solver;

enum { MGO_OK = 0, MGO_NOT_CONVERGED = 1, MGO_EINVAL = -1, MGO_ENOMEM = -2,
       MGO_EINCOMPATIBLE = -4, MGO_EDIVERGED = -5 };

/* bc[axis]: 0 periodic, 1 homogeneous Neumann.  Density defaults to rho == 1. */
int  mgo_create(int nx, int ny, int nz, double h, const int bc[3], mgo_solver **out);
/* R24 (the paper's box has a no-slip base, two symmetry planes and "continuous"
 * outflow planes): one boundary type per side, order x-, x+, y-, y+, z-, z+.
 * PERIODIC must be given for both sides of an axis.  NEUMANN: no flux through the wall (face
 * coefficient 0).  DIRICHLET: p = 0 on the wall face: the ghost value is -p_c, ghost density the
 * cell's, i.e. a wall face of coefficient 2 (a_c + a_c) whose neighbour value is 0; coarse walls
 * are the mean of the four finer wall faces (C3); the prolongation ghost is -e_boundary.  With a
 * Dirichlet wall the system is non-singular: mgo_solve checks no compatibility and removes no
 * mean.  mgo_solve_pcg / mgo_precondition / mgo_restrict_adj / mgo_project_* return MGO_EINVAL
 * on such a solver (they are defined for periodic and Neumann sides). */
enum { MGO_BC_PERIODIC = 0, MGO_BC_NEUMANN = 1, MGO_BC_DIRICHLET = 2 };
int  mgo_create6(int nx, int ny, int nz, double h, const int bc6[6], mgo_solver **out);
void mgo_destroy(mgo_solver *s);
int  mgo_set_cycle(mgo_solver *s, int nu1, int nu2, int coarse_sweeps);
/* R23: cycle index.  V (default): one visit of the coarse problem per level;
 * W: two, the second continuing from the first one's correction; F: an F visit, then a V visit.
 * mgo_vcycle / mgo_solve run this cycle. */
enum { MGO_CYCLE_V = 0, MGO_CYCLE_F = 1, MGO_CYCLE_W = 2 };
int  mgo_set_cycle_type(mgo_solver *s, int type);
int  mgo_set_density(mgo_solver *s, const double *rho);

int  mgo_vcycle(mgo_solver *s, const double *rhs, double *p);
int  mgo_residual(mgo_solver *s, const double *rhs, const double *p, double *r_or_null,
                  double *norm2);
int  mgo_solve(mgo_solver *s, const double *rhs, double *p, double rtol, int max_cycles,
               int *cycles_out, double *relres_out, double *hist_or_null);

/* ---- MG-preconditioned CG (R22 and C12-C14 are stated in mgo.c).
 * Needs nu1 == nu2 (MGO_EINVAL otherwise).  hist[k] = ||r_k||_2 of the recurrence residual. */
int  mgo_solve_pcg(mgo_solver *s, const double *rhs, double *p, double rtol, int max_iter,
                   int *iters_out, double *relres_out, double *hist_or_null);
/* z = M r: one SYMMETRIC cycle from z = 0 (black->red post-smoothing, restriction (1/8) P^T) */
int  mgo_precondition(mgo_solver *s, const double *r, double *z);
/* fc = (1/8) P^T r; r on `level`, fc on level+1 */
int  mgo_restrict_adj(const mgo_solver *s, int level, const double *r, double *fc);

/* ---- projection steps either side of the solve (staggering and the
 * expression trees C10, C11 are stated in mgo.c) ----
 * f = div(u*)/dt from the staggered velocity (u,v,w on the minus faces of each cell) */
int  mgo_project_rhs(const mgo_solver *s, const double *u, const double *v, const double *w,
                     double dt, double *f);
/* u -= dt * beta_face * grad p, in place, with the level-0 face coefficients */
int  mgo_project_correct(const mgo_solver *s, const double *p, double dt, double *u, double *v,
                         double *w);

/* ---- step-level entry points (used by the pins and by step-by-step parity) ---- */
int  mgo_num_levels(const mgo_solver *s);
int  mgo_level_dims(const mgo_solver *s, int level, int dims[3], double *h_level);
/* copies the minus-face coefficient arrays of `level` (each nx*ny*nz of that level) */
/* plus-wall face coefficients of level `level`: wx[ny*nz], wy[nx*nz], wz[nx*ny] (0 on a periodic axis) */
int  mgo_get_walls(const mgo_solver *s, int level, double *wx, double *wy, double *wz);
int  mgo_get_faces(const mgo_solver *s, int level, double *bx, double *by, double *bz);
/* out = A_level p */
int  mgo_apply(const mgo_solver *s, int level, const double *p, double *out);
/* one half-sweep on cells with (i+j+k)&1 == colour, in place (C4, C5) */
int  mgo_smooth_half(const mgo_solver *s, int level, int colour, const double *f, double *p);
/* r = f - A_level p (C6) */
int  mgo_residual_level(const mgo_solver *s, int level, const double *f, const double *p, double *r);
/* fc = 8-child mean of r (C7); r on `level`, fc on level+1 */
int  mgo_restrict(const mgo_solver *s, int level, const double *r, double *fc);
/* p += P e (C8); p on `level`, e on level+1 */
int  mgo_prolong_add(const mgo_solver *s, int level, const double *e, double *p);
/* number of OpenMP threads the loops use (1 if built without OpenMP) */
int  mgo_threads(void);
void mgo_set_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
