/* mg.h -- C ABI of libmg: B200 (sm_100a) geometric-multigrid solver for the
 * variable-density pressure Poisson equation of a two-phase VOF projection method,
 *
 *      div( (1/rho) grad p ) = div(u*) / dt                 (fp64, one GPU)
 *
 * i.e. the pressure step implied by the incompressible Navier-Stokes equations the
 * paper solves with FS3D (eq. 1-2) on a uniform Cartesian finite-volume
 * mesh, with cell density from volume-fraction mixing (PAPER.md:47-52,
 * eq. 5) and "the Multigrid" as the solver.  The paper gives no
 * further detail; the operation is fixed by BASELINE.json `north_star` and the readings
 * R1-R24 / expression trees C1-C14 listed in DESIGN.md §3.
 * The call list is north_star's: mg_create(nx,ny,nz,h,bc), mg_set_density(rho),
 * mg_vcycle, mg_residual, mg_solve(rhs,p,rtol,max_cycles).
 *
 * Discrete problem.  Cell-centred unknowns on nx*ny*nz cells of size h; dense arrays,
 * x fastest, idx = i + nx*(j + ny*k), no ghost layers, no padding.
 *      (A p)_c = (1/h^2) * sum over the 6 faces of  beta_face * (p_nb - p_c)
 *      beta_face = 1/rho_face, rho_face = harmonic mean of the two cell densities
 * Per axis the boundary is periodic (wrap) or homogeneous Neumann (wall-face beta = 0);
 * mg_create6 takes one type per side and adds Dirichlet walls (p = 0 on the wall face).
 * Without a Dirichlet wall A is singular (constants): rhs must be mean-free and mg_solve
 * returns the zero-mean p.
 * One V(nu1,nu2) cycle = nu1 red-black Gauss-Seidel sweeps (red = even i+j+k first),
 * residual, 8-child-mean restriction, recursion on the coarse grid from a zero guess,
 * cell-centred trilinear prolongation + correction, nu2 sweeps.  Coarse levels carry
 * face coefficients that are the mean of the 4 finer faces lying on each coarse face;
 * the coarsest level (reached when halving would make a dimension odd or <= 2, 4^3
 * for all BASELINE configs) is relaxed with `coarse_sweeps` sweeps.
 *
 * Conventions.  All functions return an int status: MG_OK (0), MG_NOT_CONVERGED (1) or
 * a negative error.  No exception crosses the ABI.  A handle is not thread-safe.
 * Pointers named *_dev are DEVICE pointers (cudaMalloc / torch tensor .data_ptr()) to
 * fp64 data on the device that was current at mg_create, aligned to 16 bytes (the kernels
 * move cell pairs; a misaligned pointer is rejected with MG_EINVAL); *_host are HOST pointers.
 * The library never frees or keeps caller buffers beyond what each call states.  Work
 * is enqueued on the handle's stream (mg_set_stream); calls that return a host value
 * synchronise that stream, the others are asynchronous.
 */
#ifndef MG_H
#define MG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_solver mg_handle;

enum {
    MG_OK = 0,
    MG_NOT_CONVERGED = 1,   /* mg_solve hit max_cycles; p holds the last iterate          */
    MG_EINVAL = -1,         /* bad argument (size < 4, odd size, h <= 0, bad bc, rho <= 0) */
    MG_ENOMEM = -2,         /* device or host allocation failed / workspace too small      */
    MG_ECUDA = -3,          /* a CUDA call failed; see mg_last_cuda_error()                */
    MG_EINCOMPATIBLE = -4,  /* singular system and |mean(rhs)| > 1e-12 * ||rhs||_2/sqrt(N)  */
    MG_EDIVERGED = -5       /* a residual norm became non-finite                           */
};

enum { MG_BC_PERIODIC = 0, MG_BC_NEUMANN = 1, MG_BC_DIRICHLET = 2 /* mg_create6 only */ };

/* mg_set_option keys */
enum {
    MG_OPT_KERNELS = 1,     /* 0 = reference kernels (one launch per half-sweep / transfer),
                               1 = fused streaming kernels, TMA-staged sweeps (default)      */
    MG_OPT_GRAPH = 2,       /* 1 (default) = V-cycle replayed from a captured CUDA graph     */
    MG_OPT_COARSE_CTA = 3,  /* 1 (default) = levels <= 16^3 run in one persistent CTA       */
    MG_OPT_SWEEP_FUSE = 4,  /* sweeps fused per pass of the TMA kernel: 1; 2 (default) = two where it
                               pays (level 0 from 2^26 cells, streamed stored-face levels);
                               3 = two wherever the kernel runs */
    MG_OPT_TAIL_FUSION = 5, /* 1 (default) = residual+restriction fused behind the last pre-sweep
                               and, in mg_solve, sum r^2 behind the last post-sweep, on level 0;
                               2 = the restriction tail on the streamed stored-face levels too;
                               0 = separate passes */
    MG_OPT_PROLONG_FUSE = 7, /* 1 = prolongation + correction fused in front of the first post-sweep
                               of level 0 (mg_vcycle; one pass of the TMA kernel whose p plane is
                               staged as p + P e); 0 (default) = separate prolongation pass, which
                               measured faster */
    MG_OPT_FACE_STREAM_LOG2 = 6 /* stored-face levels (>= 1) with at least 2^value cells use the
                               TMA kernel, smaller ones two half-sweep launches per sweep
                               (default 24; 0 = every level the kernel can tile) */
};

/* mg_get_stat keys */
enum {
    MG_STAT_KERNEL_LAUNCHES = 1,  /* kernels of this library launched so far (graph nodes
                                     counted per replay)                                    */
    MG_STAT_WORKSPACE_BYTES = 2,  /* device bytes of the workspace (mg_workspace_bytes)     */
    MG_STAT_LAUNCHES_PER_VCYCLE = 3,
    MG_STAT_EXTRA_DEVICE_BYTES = 4 /* device bytes the handle holds OUTSIDE the workspace, taken with
                                     cudaMalloc on first use even by mg_create_in handles and freed by
                                     mg_destroy: 4 N doubles after the first mg_solve_pcg /
                                     mg_precondition, 3 N doubles after the first mg_solve_host; 0 before */
};

/* Bytes of device workspace a solver of this size needs (all levels, all scratch). */
size_t mg_workspace_bytes(int nx, int ny, int nz);

/* north_star mg_create(nx,ny,nz,h,bc) (grid R2, R3, hierarchy R7, boundaries R5).
 * Create a solver.  bc[axis] in {MG_BC_PERIODIC, MG_BC_NEUMANN} for x,y,z (both sides
 * of an axis share the type).  Builds the level list, allocates ALL storage once
 * (cf. the paper's memory-pool lesson) with cudaMalloc, sets rho == 1,
 * V(2,2), 32 coarsest sweeps, stream 0.
 * Errors: MG_EINVAL (nx,ny,nz < 4 or odd, h <= 0 or non-finite, bad bc), MG_ENOMEM, MG_ECUDA. */
int mg_create(int nx, int ny, int nz, double h, const int bc[3], mg_handle **out);

/* As mg_create, but all device storage is carved from caller memory `workspace_dev`
 * (>= mg_workspace_bytes(), 256-byte aligned; e.g. a torch uint8 tensor).  The caller
 * keeps ownership and must keep it alive until mg_destroy. */
int mg_create_in(int nx, int ny, int nz, double h, const int bc[3],
                 void *workspace_dev, size_t workspace_bytes, mg_handle **out);

/* One boundary type per SIDE (R24; the paper's box has a no-slip
 * base, two symmetry planes and "continuous" outflow planes): bc6 = {x-, x+, y-, y+,
 * z-, z+}, each MG_BC_PERIODIC (both sides of the axis), MG_BC_NEUMANN (no flux through the wall)
 * or MG_BC_DIRICHLET (p = 0 on the wall face: ghost value -p_c, i.e. a wall face of coefficient
 * 2 (a_c + a_c) whose neighbour value is 0; coarse walls are the mean of the four finer wall
 * faces; the prolongation ghost is -e_boundary).  With a Dirichlet wall the system is
 * non-singular: mg_solve checks no compatibility and removes no mean.  Such a solver runs the
 * same kernels as the others: the TMA sweep kernel on level 0 (ghost beyond a Dirichlet wall:
 * a = 3 a_c, p = 0, never updated) and on the large stored-face levels (plus-wall faces patched into
 * the staged face tiles), the streaming residual / restriction / prolongation kernels with the wall
 * logic compiled in, half-sweep launches on the small levels, the persistent coarse CTA; mg_project*, mg_solve_pcg and mg_precondition return MG_EINVAL (the
 * staggered velocity layout has no plus-wall face; the symmetric cycle is defined for periodic
 * and Neumann sides).  Without a Dirichlet side this is mg_create / mg_create_in.  Errors as mg_create. */
int mg_create6(int nx, int ny, int nz, double h, const int bc6[6], mg_handle **out);
int mg_create6_in(int nx, int ny, int nz, double h, const int bc6[6],
                  void *workspace_dev, size_t workspace_bytes, mg_handle **out);

/* Frees everything the library allocated (never caller buffers).  NULL is allowed. */
void mg_destroy(mg_handle *s);

/* All later work is enqueued on `cuda_stream` (a cudaStream_t; NULL = default stream). */
int mg_set_stream(mg_handle *s, void *cuda_stream);

/* V(nu1,nu2) and the number of sweeps on the coarsest level (defaults 2,2,32). */
int mg_set_cycle(mg_handle *s, int nu1, int nu2, int coarse_sweeps);

/* Cycle index (R23; the paper only names "the Multigrid",
 * PAPER.md:216).  MG_CYCLE_V (default): every level visits its coarse problem once.
 * MG_CYCLE_W: twice, the second visit continuing from the correction of the first.
 * MG_CYCLE_F: an F-cycle visit followed by a V-cycle visit.  The coarsest level (R13) is
 * visited once per visit of the level above it.  mg_vcycle, mg_solve and mg_project run this
 * cycle; changing it re-captures the graph.  MG_EINVAL for any other value. */
enum { MG_CYCLE_V = 0, MG_CYCLE_F = 1, MG_CYCLE_W = 2 };
int mg_set_cycle_type(mg_handle *s, int type);

int mg_set_option(mg_handle *s, int key, int value);
int mg_get_stat(const mg_handle *s, int key, long long *value_host);

/* Step A0 (north_star "face coefficients from harmonic-averaged cell density";
 * density by volume-fraction mixing, eq. 5; readings R4, R8, C2, C3 of DESIGN.md).
 * Density field: rho_dev = N doubles, read-only, may be freed once the stream has
 * passed this call.  The library derives and owns a = 0.5/rho (level 0) and the face
 * coefficients of every coarser level.  Synchronises the stream (validity check).
 * MG_EINVAL if any rho is <= 0 or non-finite (coefficients are then unspecified). */
int mg_set_density(mg_handle *s, const double *rho_dev);

/* Steps A1-A6, A8 (north_star "geometric multigrid V-cycle ... red-black Gauss-Seidel
 * smoothing, residual, full-weighting restriction, trilinear prolongation and correction"; "the
 * Multigrid"; readings R9-R14, R23, C4-C8).  One cycle of the set type (V by default)
 * in place on p_dev for right-hand side rhs_dev (N doubles each), replayed from a CUDA graph.
 * No mean removal, no norm.  Asynchronous on the stream.  MG_EINVAL for NULL or misaligned pointers. */
int mg_vcycle(mg_handle *s, const double *rhs_dev, double *p_dev);

/* Steps A2, A7 (north_star "residual", "residual-norm reductions"; R10, R15, C6, C9).
 * r = rhs - A p.  Writes r to r_dev (N doubles, caller-owned) if non-NULL, and sqrt(sum r^2) to
 * *norm2_host if non-NULL (then the stream is synchronised; the sum is a fixed two-stage tree,
 * no atomics). */
int mg_residual(mg_handle *s, const double *rhs_dev, const double *p_dev,
                double *r_dev, double *norm2_host);

/* Step A7 + control (north_star mg_solve(rhs,p,rtol,max_cycles); R6, R15).
 * Cycles until ||rhs - A p||_2 <= rtol * ||rhs - A p_0||_2 or max_cycles.
 * p_dev: in = initial guess, out = iterate with its arithmetic mean removed.
 * hist_host (NULL or >= max_cycles+1 doubles) receives ||r_k||_2, k = 0..cycles.
 * Returns MG_OK, MG_NOT_CONVERGED, MG_EINCOMPATIBLE (p untouched), MG_EDIVERGED.
 * A residual that rises in the first cycle is normal and not an error. */
int mg_solve(mg_handle *s, const double *rhs_dev, double *p_dev, double rtol, int max_cycles,
             int *cycles_host, double *relres_host, double *hist_host);

/* MG-preconditioned conjugate gradients (R22, C12-C14; the paper
 * only names "the Multigrid").  Preconditioner z = M r = ONE symmetric cycle from
 * z = 0: nu1 red->black sweeps, residual, restriction (1/8) P^T (the adjoint of the trilinear
 * prolongation), coarse correction, prolongation, nu2 = nu1 black->red sweeps; on the coarsest
 * level coarse_sweeps sweeps in each order.  mg_solve_pcg: r = f - A p, z = M r, d = z, then per
 * iteration q = A d, alpha = r.z / d.q, p += alpha d, r -= alpha q, stop when ||r|| <= rtol ||r_0||
 * (r of the recurrence), z = M r, beta = r.z' / r.z, d = z + beta d.  Arguments, return values and
 * hist_host[0..iterations] as mg_solve; four more level-0 arrays (4 N doubles, NOT part of the
 * workspace or of mg_workspace_bytes; see MG_STAT_EXTRA_DEVICE_BYTES) are allocated with cudaMalloc on first use.
 * MG_EINVAL if nu1 != nu2 or the solver has a Dirichlet side.  On the paper's workloads this
 * iteration needs more work than mg_solve; it is here for completeness. */
int mg_solve_pcg(mg_handle *s, const double *rhs_dev, double *p_dev, double rtol, int max_iter,
                 int *iters_host, double *relres_host, double *hist_host);
/* z_dev = M r_dev (one symmetric cycle from zero).  Asynchronous on the stream. */
int mg_precondition(mg_handle *s, const double *r_dev, double *z_dev);

/* End-to-end variant on HOST buffers (N doubles each; pinned memory makes the copies
 * asynchronous): copies rhs_host and, if non-NULL, rho_host to the device (then also
 * runs mg_set_density), solves from the initial guess p = 0, copies the zero-mean
 * solution to p_host (output only).  Device staging buffers (3 N doubles) are owned by
 * the handle and allocated on first use.  Same return codes as mg_solve. */
int mg_solve_host(mg_handle *s, const double *rho_host, const double *rhs_host, double *p_host,
                  double rtol, int max_cycles, int *cycles_host, double *relres_host,
                  double *hist_host);

/* ---- projection steps either side of the solve (eq. 1-2).
 * Staggered velocity: u_dev[i,j,k] is the component on the MINUS x-face of cell (i,j,k) (the
 * face between cells (i-1,j,k) and (i,j,k)), v_dev on the minus y-face, w_dev on the minus
 * z-face; N doubles each, x fastest; a cell's plus face is the next cell's minus face (wrap).
 * On a Neumann axis the wrap face is the wall and the caller keeps the velocity there at 0.
 *
 * mg_project_rhs:     f = ((u[i+1]-u[i]) + (v[j+1]-v[j]) + (w[k+1]-w[k])) / (h dt)
 * mg_project_correct: u[i] -= (dt/h) beta_x[i] (p[i]-p[i-1]), likewise v, w, with the level-0
 *                     face coefficients of the current density (wall faces: beta = 0).
 * mg_project:         rhs -> mg_solve (p_dev: in = initial guess) -> correct; rhs_dev is N
 *                     doubles of caller-owned scratch that receives the right-hand side.
 * After mg_project the discrete divergence of (u,v,w) equals dt x the final residual.
 * All asynchronous on the stream except mg_project (mg_solve synchronises).
 * Errors: MG_EINVAL (NULL pointer, dt <= 0 or non-finite); mg_project also mg_solve's codes
 * (on a negative status the velocity is left untouched). */
int mg_project_rhs(mg_handle *s, const double *u_dev, const double *v_dev, const double *w_dev,
                   double dt, double *f_dev);
int mg_project_correct(mg_handle *s, const double *p_dev, double dt, double *u_dev, double *v_dev,
                       double *w_dev);
int mg_project(mg_handle *s, double *u_dev, double *v_dev, double *w_dev, double dt, double *p_dev,
               double *rhs_dev, double rtol, int max_cycles, int *cycles_host, double *relres_host);

/* ---- residual norm for callers that must not allocate (steps A2 + A7 on level 0; R10, R15, C2, C4, C6, C9).
 * Some hosts of this library cannot call cudaMalloc at the point where they want a residual
 * norm: a flow solver that, like the paper's (section 4.2), gave all device memory to
 * its own pool at start-up has nothing left to allocate from, and a convergence monitor hooked
 * into a running time loop must avoid the device-wide synchronisation cudaMalloc and cudaFree
 * imply.  Every other call here needs a handle, and creating one allocates (mg_create the whole
 * hierarchy; mg_create_in still pinned host memory).  This one call takes no handle and calls no
 * cudaMalloc, cudaFree, cudaMallocHost or any other allocating routine; it only launches two
 * kernels on `cuda_stream` (a cudaStream_t, NULL = default stream) and returns without waiting.
 *
 *   *norm2_dev = sqrt( sum over all cells of (rhs - A p)^2 ),  A built from rho as mg_set_density
 *   does (a = 0.5/rho, face = a_c + a_nb, Neumann wall face = 0) with cell size h.
 *
 * Inputs rho_dev, rhs_dev, p_dev: nx*ny*nz doubles each on the CURRENT device, read-only, layout
 * as everywhere in this header; rho must be finite and > 0 (not checked here).  Output norm2_dev:
 * one double on the same device, written by the second kernel.  bc[axis] is MG_BC_PERIODIC or
 * MG_BC_NEUMANN.  The value differs from mg_residual's norm only in how the partial sums are
 * grouped (tests/test_zz_no_alloc.py holds the two to relative 1e-10).
 *
 * Scratch.  The per-block partial sums live in a fixed array compiled into the library (128 KB;
 * every GPU that loads libmg holds it until the process ends), sized for at most
 * MG_STATIC_MAX_CELLS = 2^27 cells (512^3, the paper's load per device).  A larger grid is
 * refused with MG_EINVAL and mg_last_cuda_error() then says so; use mg_residual on a handle
 * there.  All calls on one GPU share that array: calls whose kernels can overlap on the GPU
 * (different streams without an ordering between them, several host threads) race on it and
 * return garbage, so keep them on one stream or order them with events.  The array keeps the
 * partial sums of the previous call; each call first overwrites every slot it later reads, so
 * nothing has to be cleared and no call sees another's leftovers.
 *
 * First call on each device.  It looks up the device address of that array
 * (cudaGetSymbolAddress, with this device current) and remembers it; later calls skip this.
 * Make this first call during start-up, before any stream capture begins.
 * Errors: MG_EINVAL (bad sizes as mg_create, bad bc, NULL pointer, too many cells), MG_ECUDA. */
#define MG_STATIC_MAX_CELLS 134217728LL
int mg_residual_norm_static(int nx, int ny, int nz, double h, const int bc[3],
                            const double *rho_dev, const double *rhs_dev, const double *p_dev,
                            double *norm2_dev, void *cuda_stream);

const char *mg_strerror(int status);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char *mg_last_cuda_error(void);

/* ---- introspection and single steps of the cycle (same kernels the cycle uses;
 *      meant for step-by-step verification and for embedding in other cycles) ---- */
int mg_num_levels(const mg_handle *s);
int mg_level_dims(const mg_handle *s, int level, int dims[3], double *h_level_host);
/* Copies the minus-face coefficients of `level` into caller device arrays (level cells
 * each): bx[i,j,k] = face between (i-1,j,k) and (i,j,k), etc.; wall faces are 0. */
int mg_level_faces(mg_handle *s, int level, double *bx_dev, double *by_dev, double *bz_dev);
/* One Gauss-Seidel half-sweep on the cells with (i+j+k)&1 == colour, in place. */
int mg_level_smooth_half(mg_handle *s, int level, int colour, const double *f_dev, double *p_dev);
/* `sweeps` full red-black sweeps with the kernels selected by MG_OPT_KERNELS. */
int mg_level_smooth(mg_handle *s, int level, int sweeps, const double *f_dev, double *p_dev);
/* r = f - A_level p */
int mg_level_residual(mg_handle *s, int level, const double *f_dev, const double *p_dev,
                      double *r_dev);
/* fc = 8-child mean of (f - A_level p): fused residual + restriction, level -> level+1 */
int mg_level_residual_restrict(mg_handle *s, int level, const double *f_dev,
                               const double *p_dev, double *fc_dev);
/* `sweeps` (>= 1) sweeps in place on p, then fc = 8-child mean of (f - A_level p): the last
 * pre-sweep of the cycle with steps A2+A3 fused behind it (level 0: one pass of the TMA kernel) */
int mg_level_smooth_restrict(mg_handle *s, int level, int sweeps, const double *f_dev, double *p_dev,
                             double *fc_dev);
/* `sweeps` (>= 1) level-0 sweeps in place on p, then sqrt(sum (f - A p)^2) to *norm2_host: the
 * last post-sweep of mg_solve's cycle with step A7 fused behind it.  Synchronises the stream. */
int mg_level_smooth_norm(mg_handle *s, int sweeps, const double *f_dev, double *p_dev, double *norm2_host);
/* p += trilinear prolongation of e (e on level+1, p on level) */
/* p <- `sweeps` (>= 1) sweeps of (p + P e): prolongation, correction and the first sweep in one
 * pass where the TMA kernel runs (level 0), otherwise mg_level_prolong_add + mg_level_smooth */
int mg_level_prolong_smooth(mg_handle *s, int level, int sweeps, const double *e_dev, const double *f_dev,
                            double *p_dev);
/* fc = (1/8) P^T r (C14), level -> level + 1 */
int mg_level_restrict_adj(mg_handle *s, int level, const double *r_dev, double *fc_dev);
int mg_level_prolong_add(mg_handle *s, int level, const double *e_dev, double *p_dev);

/* Verification aid (C5: p = fma(-h2, f, S) * (1.0 / D) with the correctly rounded reciprocal).  The
 * TMA sweep kernels form 1.0 / D with a branch-free instruction sequence when every a = 0.5/rho
 * lies in [2^-900, 2^900] (mg_set_density checks), else with the library reciprocal.  This call
 * evaluates both on n caller values: fast_dev[i] = branch-free sequence, lib_dev[i] = library
 * reciprocal of d_dev[i]; all device arrays of n doubles; asynchronous on `cuda_stream`.  A test
 * holds both to the host's 1.0 / d bit for bit over the admitted range (tests/test_gpu_rcp.py). */
int mg_test_rcp(const double *d_dev, size_t n, double *fast_dev, double *lib_dev, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* MG_H */
