/*
 * mg.h -- C ABI of libmg_b200: the B200 (sm_100a) geometric-multigrid pressure solve and the
 * explicit stencil residuals of arxiv/paper_2401_06755 (NN4PDEs multiphase flow).
 *
 * "P:NNN" cites a line of the paper text.  Readings of silent / garbled passages
 * ("reading Cn") are listed in DESIGN.md.
 *
 * Conventions (all entry points)
 * ------------------------------
 *  - Every field is a dense array of nx*ny*nz values, x fastest: idx = i + nx*(j + ny*k),
 *    cell-centred, WITHOUT halo (the paper's outputs are unpadded).  Halos
 *    carrying the boundary conditions exist only inside the kernels.
 *  - Pointers named d_* are DEVICE pointers, 16-byte aligned, owned by the caller; the
 *    library never frees or reallocates them.  Pointers named h_* are HOST pointers.
 *    The element type is float (MG_F32) or double (MG_F64) as selected at creation.
 *  - All work is enqueued on the CUDA stream given at creation (a cudaStream_t passed as
 *    void*; NULL = the legacy default stream).  Only mg_solve*, *_host and mg_vcycle_timed
 *    synchronise with the host.
 *  - Return value: 0 = MG_OK, < 0 = error (nothing useful was computed; mg_last_error()
 *    describes it), > 0 = non-fatal status of mg_solve.  No exception or abort crosses
 *    the boundary.  There is no CPU fallback: without a CUDA device every compute call
 *    returns MG_ECUDA.
 */
#ifndef MG_B200_H
#define MG_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mg_solver mg_solver; /* opaque; owned by the library, freed by mg_destroy */

typedef enum { MG_F32 = 0, MG_F64 = 1 } mg_dtype;

/* Boundary condition of one face = the factor s of the halo rule ghost = s * mirror
 * (reading C3; Fig. 2 caption P:276); applied at every multigrid level. */
typedef enum {
    MG_BC_NEUMANN = 0,       /* s = +1: zero normal derivative, "copying the nearest nodal value" */
    MG_BC_DIRICHLET = 1,     /* s = -1: zero value ON the cell face (interpolation rule of Fig. 2)  */
    MG_BC_DIRICHLET_HALO = 2 /* s =  0: halo node set to the value 0 (literal P:256)                        */
} mg_bc;

typedef struct { int nx, ny, nz; double hx, hy, hz; } mg_grid;

/* V-cycle parameters (the paper gives none: P:43, P:47, P:105 name "Jacobi smoothing" only;
 * defaults are BASELINE.json config 1): nu_pre, nu_post weighted-Jacobi sweeps, coarse_sweeps
 * sweeps on the coarsest level from a zero guess, omega the damping.
 * sweeps_per_pass: how many dependent stencil stages (sweeps, the prolongation + sweep, the residual +
 * restriction) one kernel launch may carry on a level, 1 .. 4 (wave_kernel.cuh); other values are refused
 * with MG_EINVAL; a level on which that many stages do not fit the machine at once gets fewer per launch.
 * Results do not depend on it beyond rounding order.  mixed_precision (MG_F32 only): mg_solve keeps the
 * iterate and the fine-grid residual in fp64 around fp32 V-cycles (reading C6/C8).
 * cycles_per_defect (mixed precision only): V-cycles applied to one correction equation A e = r before the next fp64 defect is
 * formed -- the first from a zero guess, the others continue the iteration on e with the same r, so in exact arithmetic the
 * iterates are those of plain cycles; the residual (stopping test, history) is then evaluated every cycles_per_defect cycles
 * only, which is what saves the time (the fp64 defect and the fp64 update cost 40 % of a cycle).  Default 1: every cycle.
 * 0 = adaptive: a tolerance-driven solve starts with one cycle per defect and then takes, round by round, as many cycles as the
 * contraction observed in the last round says are still needed to reach tol, at most 8 and no more than keep the round's
 * contraction above 1e-5 (what fp32 resolves of a correction), rounded down to 1, 2, 4 or 8; a fixed-count solve (tol = 0)
 * takes 4 (then 2, 1 for what is left).
 * mg_get_history_cycles tells after how many cycles each history entry was taken. */
typedef struct {
    int nu_pre, nu_post, coarse_sweeps, sweeps_per_pass;
    double omega;
    int mixed_precision;
    int cycles_per_defect;   /* 1 .. 8, default 1; 0 = adaptive */
} mg_params;

enum {
    MG_OK = 0,
    MG_NOT_CONVERGED = 1, /* mg_solve stopped on max_cycles */
    MG_STAGNATED = 2,     /* residual ratio > 0.95 for 3 consecutive cycles, or non-finite */
    MG_EINVAL = -1,       /* NULL or out-of-range argument */
    MG_ESHAPE = -2,       /* a dimension not divisible by 2^(levels-1), coarsest dimension < 2, or more than 2^31 - 1 points */
    MG_ECUDA = -3,        /* a CUDA call failed (no device, launch error, ...) */
    MG_EALLOC = -4        /* device or host allocation failed */
};

/* Create a solver for A p = b with A the 27-point trilinear-FE discretisation of -div(k grad)
 * (Eqs. 8, 11-13; readings C1, C2) on `grid`, with `levels` grids
 * coarsened 2:1 (n_{l+1} = n_l/2, h_{l+1} = 2 h_l, operator rediscretised, reading C5) and the
 * boundary factors bc[6] = {x-, x+, y-, y+, z-, z+}.  The solver owns its level hierarchy,
 * scratch, CUDA graph and pinned host words.  Coefficient starts as k = 1 (constant).  Size: nx ny nz <= 2^31 - 1 (MG_ESHAPE
 * otherwise); 2048 x 1024 x 512 (2^30 points, 4 GiB per fp32 field) is the largest grid under test (tests/test_gpu_maxsize.py). */
int mg_create(mg_solver** out, const mg_grid* grid, int levels, const int bc[6], int dtype, void* cuda_stream);
void mg_destroy(mg_solver* s);

int mg_set_params(mg_solver* s, const mg_params* p); /* defaults: 2, 2, 50, 1, 2/3, 1 */
int mg_get_params(const mg_solver* s, mg_params* p);

/* Coefficient k (a7).  d_k: nx*ny*nz values of k > 0, or NULL for constant k = 1.  The field is
 * copied; coarse levels get the arithmetic mean of the 8 children (reading C5). */
int mg_set_coefficient(mg_solver* s, const void* d_k);
/* k = 1 / (rho_l a + rho_g (1 - a)), Eqs. 2 and 19, with a = alpha limited to [0, 1] (reading C7: the paper does not
 * clip, but an undershoot of alpha below -rho_g / (rho_l - rho_g) = -0.001 would make the density negative and the operator
 * indefinite; the explicit stages form rho and mu the same way). */
int mg_set_coefficient_from_vof(mg_solver* s, const void* d_alpha, double rho_l, double rho_g);

/* a1: y = A x on the fine level.  d_y must not alias d_x. */
int mg_apply_operator(mg_solver* s, const void* d_x, void* d_y);
/* a2: `sweeps` weighted-Jacobi sweeps x <- x + omega (b - A x) / D, in place (two-buffer
 * inside; every point of a sweep uses the previous sweep's x).  Reading C4. */
int mg_smooth(mg_solver* s, void* d_x, const void* d_b, int sweeps);
/* r = b - A x on the fine level. */
int mg_residual(mg_solver* s, const void* d_x, const void* d_b, void* d_r);
/* a3..a6: one V(nu_pre, nu_post) cycle in place (Fig. 5; reading C6). */
int mg_vcycle(mg_solver* s, void* d_x, const void* d_b);
/* a6: V-cycles until ||b - A x||_2 / ||b||_2 < tol or max_cycles (the paper runs a fixed 20,
 * P:429).  d_x holds the initial guess on entry and the solution on exit.  cycles_out /
 * relres_out may be NULL.  Returns MG_OK, MG_NOT_CONVERGED or MG_STAGNATED. */
int mg_solve(mg_solver* s, void* d_x, const void* d_b, double tol, int max_cycles, int* cycles_out,
             double* relres_out);
/* V-cycle-preconditioned conjugate gradients (SURVEY 8(f) "next 1"; NOT in the paper, which runs plain cycles):
 * textbook PCG for the SPD system A p = b with one V(nu, nu) cycle from a zero guess as preconditioner; it converges in
 * ~12 iterations where the plain cycle stalls under a 1000:1 coefficient jump.  Needs nu_pre == nu_post >= 1 (symmetric
 * cycle) and a uniform grid with nx % 4 == 0, else MG_EINVAL.  The CG vectors are fp64 for either dtype.  Same argument
 * conventions, stopping rule (||b - A x||_2 / ||b||_2 < tol, recursively updated residual) and return values as mg_solve;
 * iters_out = iterations = V-cycles after the first; mg_get_history gives the residual after every iteration. */
int mg_pcg_solve(mg_solver* s, void* d_x, const void* d_b, double tol, int max_iter, int* iters_out, double* relres_out);
/* Same with HOST buffers: copies h_b and the guess h_x to the device, solves, copies x back. */
int mg_solve_host(mg_solver* s, void* h_x, const void* h_b, double tol, int max_cycles, int* cycles_out,
                  double* relres_out);
/* Same from a ZERO initial guess (the pressure correction of a time step starts from zero): h_x is output only
 * and is not read; the guess is set on the device, so the call moves one field in (h_b) and one out (h_x).  The iterates
 * are those of mg_solve_host called with h_x = 0, bit for bit. */
int mg_solve_host_zero(mg_solver* s, void* h_x, const void* h_b, double tol, int max_cycles, int* cycles_out,
                       double* relres_out);
/* Relative residual after every cycle of the last mg_solve (up to n entries); returns count. */
int mg_get_history(const mg_solver* s, double* h_history, int n);
/* The number of V-cycles (mg_pcg_solve: iterations) completed when each of those entries was taken: 1, 2, 3, ... unless
 * cycles_per_defect != 1 (up to n entries; returns count, the same as mg_get_history). */
int mg_get_history_cycles(const mg_solver* s, int* h_cycles, int n);

/* Measurement helpers.  mg_level_info: points of level l (returns < 0 if l is out of range).
 * mg_vcycle_timed: one V-cycle with CUDA events around every level's down leg and up leg;
 * h_ms_down / h_ms_up receive `levels` floats each (the coarsest level's time is in down). */
long long mg_level_info(const mg_solver* s, int level, int* nx, int* ny, int* nz);
int mg_vcycle_timed(mg_solver* s, void* d_x, const void* d_b, float* h_ms_down, float* h_ms_up);
/* Number of kernel launches the library has enqueued on behalf of this solver so far. */
long long mg_launch_count(const mg_solver* s);
/* 0: every level with separate one-sweep kernels (reference path); 1 (default): fused kernels,
 * single-CTA coarse tail and CUDA-graph replay. */
int mg_set_fused(mg_solver* s, int fused);

/* ------------------------------------------------------------------------------------------
 * Explicit stencil residuals feeding the solve (a8-a10).  Stateless; scratch comes from the
 * stream-ordered pool of `cuda_stream`.  Halos of C, of the velocities and of every derived
 * field are zero-derivative copies (reading C9-iv).
 * ------------------------------------------------------------------------------------------ */

/* a8: compressive-advection VoF residual, Eqs. 16, 26/27, 29, 33, 35-42 (P:179-181, 264-288,
 * 301, 327-401; reading C9 steps 1-12).  d_sC_out (may be NULL) receives the nodal residual
 * s~_C / m_l; d_Cnew_out (may be NULL) receives C - dt * sC, Eq. 55. */
int vof_residual(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v,
                 const void* d_w, double dt, void* d_sC_out, void* d_Cnew_out, void* cuda_stream);
/* SURVEY 8(f) "next 4", the part of the higher-order scheme the paper prints in full: the same residual with the oscillation
 * detectors S^x, S^y, S^z chosen by `detector`: 3 = Eq. 33 (three points per direction, = vof_residual), 5 = Eq. 34 (the
 * minimum of the three products of consecutive differences over i-2 .. i+2; halo of C by reflection).  Other values: MG_EINVAL. */
int vof_residual_ex(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                    int detector, void* d_sC_out, void* d_Cnew_out, void* cuda_stream);
/* The same residual for callers that must not allocate (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): no cudaMalloc / cudaMallocAsync / cudaFree and no allocating library routine is called.  The four intermediate fields
 * (adv, k^x, k^y, k^z) live in a static device array of VOF_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until
 * the process exits; inputs and outputs are the caller's, as in vof_residual_ex, and the results are bit-identical to it.
 * Limit: 4 * roundup(nx ny nz * sizeof(element), 256) <= VOF_NOALLOC_SCRATCH_BYTES, i.e. up to 524288 points in fp32 (64 x 64 x 128)
 * and 262144 in fp64 (64^3); larger grids are refused with MG_EINVAL and a message that names both sizes (use vof_residual_ex).
 * Every call on a device shares that one array: calls that overlap on the GPU (different streams, or graphs replayed concurrently)
 * race on it -- keep them on one stream or order them with events.  The array keeps the last call's contents; nothing in it has
 * to start at zero (every field is fully written before it is read), so no clearing is needed between calls. */
#define VOF_NOALLOC_SCRATCH_BYTES (8u << 20)
int vof_residual_noalloc(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w, double dt,
                         int detector, void* d_sC_out, void* d_Cnew_out, void* cuda_stream);

/* a9: momentum advection-diffusion residual and predictor, Eqs. 18, 30-32, 45-46 (P:198-220,
 * 309-319, 433-441; reading C9 "Momentum").  d_qh[3] = half-level (u, v, w), d_qn[3] = level-n
 * (u, v, w); d_qt[3] receives q~ = q_n - dt s~/rho, d_qhn[3] (may be NULL) (q_n + q~)/2.
 * Outputs must not alias inputs. */
int mom_predictor(const mg_grid* grid, int dtype, const void* d_C, const void* const d_qh[3],
                  const void* const d_qn[3], double rho_l, double rho_g, double mu_l, double mu_g, double dt,
                  void* const d_qt[3], void* const d_qhn[3], void* cuda_stream);

/* SURVEY 8(f) "next 3": the same predictor with free-slip walls.  vbc[6 c + f] is the halo code (an mg_bc) of velocity
 * component c = u, v, w on face f: at a wall the component NORMAL to it is odd about the face (MG_BC_DIRICHLET: zero normal
 * velocity on the wall, the interpolation rule of Fig. 2), the tangential ones and everything on an open face are copied
 * (MG_BC_NEUMANN).  The halo of a component enters its gradient and its diffusion; derived fields keep copy halos.
 * vbc = NULL: all copies (= mom_predictor). */
int mom_predictor_bc(const mg_grid* grid, int dtype, const void* d_C, const void* const d_qh[3], const void* const d_qn[3],
                     const int vbc[18], double rho_l, double rho_g, double mu_l, double mu_g, double dt, void* const d_qt[3],
                     void* const d_qhn[3], void* cuda_stream);
/* SURVEY 8(f) "next 3": the terms of Eq. 18 that the advection-diffusion residual leaves out, applied to the predicted
 * velocity (Eq. 45 is linear in the source):
 *   q~_c <- q~_c - (dt / rho) ( f(p_hs + p~_nh; w_c) + f(F_c; w_m) ),   F = -(s + s_t) as written by hydrostatic_rhs_force,
 * and, if d_qhn != NULL, q_half' = (q_n + q~)/2 (Eq. 46).  Halos: p_hs zero derivative on the sides, zero value on the top face and
 * the extrapolation ghost mirror + hz g rho below the bottom (dp_hs/dz = -rho g); p~_nh the factors pbc of its solver; F
 * copies.  d_phs, d_pnh, d_force may be NULL (term absent).  d_qt is updated in place. */
int mom_forcing(const mg_grid* grid, int dtype, const void* d_C, const void* d_phs, const void* d_pnh, const int pbc[6], double g,
                const void* const d_force[3], double rho_l, double rho_g, double dt, void* const d_qt[3], const void* const d_qn[3],
                void* const d_qhn[3], void* cuda_stream);

/* a10: b = -(1/dt) (f(u; w_x) + f(v; w_y) + f(w; w_z)), nodal FE filters of Eq. 11
 * (structure of Eq. 53; reading C10). */
int pressure_rhs(const mg_grid* grid, int dtype, const void* d_u, const void* d_v, const void* d_w, double dt,
                 void* d_b, void* cuda_stream);
/* the same with the velocity halo codes vbc of mom_predictor_bc (NULL: copies) */
int pressure_rhs_bc(const mg_grid* grid, int dtype, const void* d_u, const void* d_v, const void* d_w, const int vbc[18], double dt,
                    void* d_b, void* cuda_stream);
/* SURVEY 8(f) "next 2", the paper's own stage-3 right-hand side, Eqs. 52-53: density on the right, constant-
 * coefficient Laplacian:  b = -(1/dt) sum_d f(rho q_d; w_d) + (1/dt) sum_d q_d f(rho; w_d),  rho = rho_l C + rho_g (1 - C). */
int pressure_rhs_paper(const mg_grid* grid, int dtype, const void* d_C, const void* d_u, const void* d_v, const void* d_w,
                       double rho_l, double rho_g, double dt, void* d_b, void* cuda_stream);
/* SURVEY 8(f) "next 3", stage 1: right-hand side of the hydrostatic and surface-tension pressure p_hs (Eqs. 20-23, 44;
 * P:226-246, 419-427):  n_t = grad C / (1e-7/hx + |grad C|), kappa = -(f(n_tu; w_x) + f(n_tv; w_y) + f(n_tw; w_z)),
 * s_t = sigma_t kappa grad C,  b = f(g rho; w_z) - (f(s_tu; w_x) + f(s_tv; w_y) + f(s_tw; w_z)), plus the contribution of the bottom
 * boundary condition dp_hs/dz = -rho g on the plane z = 0.  Solve A p_hs = b with a constant-coefficient solver and
 * bc = {N, N, N, N, N, D}.  Readings (Eq. 22 / 23 misprints; the signs of Eqs. 5, 43, 44) in DESIGN.md N3.  d_kappa_out may be NULL.
 * SIGN: d_kappa_out holds kappa = -div(n_t) and d_st_out s_t = sigma_t kappa grad C with that kappa (reading N3-b: the
 * continuum-surface-force convention, force towards the centre of curvature, p_hs higher inside a drop).  This is the
 * OPPOSITE sign of Eq. 5 as printed (kappa = +div n_t); b is numerically the b of Eq. 44 as printed either way. */
int hydrostatic_rhs(const mg_grid* grid, int dtype, const void* d_C, double rho_l, double rho_g, double g, double sigma_t,
                    void* d_b, void* d_kappa_out, void* cuda_stream);
/* the same, also writing the force field F = -(s + s_t) = (-s_tu, -s_tv, g rho - s_tw) (Eqs. 20-21) whose FE divergence is b before
 * the bottom-boundary fold; mom_forcing takes it.  d_force_out[3] may be NULL. */
int hydrostatic_rhs_force(const mg_grid* grid, int dtype, const void* d_C, double rho_l, double rho_g, double g, double sigma_t,
                          void* d_b, void* d_kappa_out, void* const d_force_out[3], void* cuda_stream);
/* a10: q <- q - dt k f(p; w_x|y|z), Eq. 54 with Eq. 48; halo of p by bc[6]. */
int project_velocity(const mg_grid* grid, const int bc[6], int dtype, const void* d_p, const void* d_k,
                     double dt, void* d_u, void* d_v, void* d_w, void* cuda_stream);

/* Config-5 time step on device buffers (stages 2-4 of P:403-505 under readings C9, C10):
 * two momentum predictor iterations, VoF residual + update, k = 1/rho(C^n), pressure RHS,
 * mg_solve(tol, max_cycles) from a zero guess into d_p, projection.  In place on d_C, d_u,
 * d_v, d_w.  The solver supplies grid, dtype, bc and stream. */
int flow_time_step(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l,
                   double rho_g, double mu_l, double mu_g, double dt, double tol, int max_cycles,
                   int* cycles_out, double* relres_out);

/* The same time step with the pressure equation solved by mg_pcg_solve(tol, max_iter) from a zero guess (SURVEY 8(f) "next 1":
 * V-cycle-preconditioned CG, not in the paper, whose plain cycles converge at 0.95 per cycle under the 1000:1 density jump);
 * needs nu_pre == nu_post >= 1 and a uniform grid with nx % 4 == 0 like mg_pcg_solve.  Everything else as flow_time_step. */
int flow_time_step_pcg(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l,
                       double rho_g, double mu_l, double mu_g, double dt, double tol, int max_iter,
                       int* iters_out, double* relres_out);

/* SURVEY 8(f) "next 3": the paper's FOUR-stage step on device fields, in place:
 *   stage 1: hydrostatic_rhs_force(C^n); A p_hs = b_hs with the constant-coefficient solver s_hs from p_hs = 0,
 *                        hs_cycles cycles (the paper's fixed 20) or until hs_tol;
 *   stage 2: two predictor iterations with free-slip wall halos (mom_predictor_bc) and the forcing terms of Eq. 18
 *                        (mom_forcing with p_hs, the incoming d_pnh and the force field);
 *   stage 3 (reading C10): b = -(1/dt) D.q~ (pressure_rhs_bc); A(1/rho) dp = b with s (mg_solve(tol, max_cycles));
 *                        q = q~ - dt k G dp; d_pnh += dp;
 *   stage 4: C <- C - dt s~_C(C^n, q^{n+1}).
 * walls[6]: 1 = free-slip wall, 0 = open face.  s_hs and s: same grid, dtype, device and stream, bc = {N,N,N,N,N,D}, s_hs
 * with a constant coefficient.  Returns the status of the stage-3 solve; cycles_out / relres_out refer to it. */
int flow_time_step_full(mg_solver* s_hs, mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_phs, void* d_pnh,
                        double rho_l, double rho_g, double mu_l, double mu_g, double g, double sigma_t, double dt, double tol,
                        int max_cycles, double hs_tol, int hs_cycles, const int walls[6], int* cycles_out, double* relres_out);
/* The same step with the stage-3 solver chosen by pressure_solver: 0 = mg_solve (plain cycles, the paper's; = flow_time_step_full),
 * 1 = mg_pcg_solve (tol, max_cycles iterations; its requirements apply).  Other values: MG_EINVAL. */
int flow_time_step_full_ex(mg_solver* s_hs, mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_phs, void* d_pnh,
                           double rho_l, double rho_g, double mu_l, double mu_g, double g, double sigma_t, double dt, double tol,
                           int max_cycles, double hs_tol, int hs_cycles, const int walls[6], int pressure_solver, int* cycles_out,
                           double* relres_out);

/* The same time step with the PAPER'S stage 3 (SURVEY 8(f) "next 2"): constant-coefficient Laplacian with the density on the
 * right (Eqs. 52-53), `cycles` V-cycles per solve from a zero guess (the paper's fixed 20), velocity correction Eq. 54,
 * the stage carried out `passes` times (twice).  d_p receives the accumulated p_nh; the solver's coefficient is reset
 * to constant; relres_out (may be NULL) the relative residual of the last solve. */
int flow_time_step_paper(mg_solver* s, void* d_C, void* d_u, void* d_v, void* d_w, void* d_p, double rho_l, double rho_g,
                         double mu_l, double mu_g, double dt, int cycles, int passes, double* relres_out);

/* Thread-local description of the last error; never freed by the caller. */
const char* mg_last_error(void);
/* Library / build identification, e.g. "libmg_b200 sm_100a". */
const char* mg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MG_B200_H */
