/*
 * oracle.c -- plain, slow, fp64 CPU oracle for the multigrid pressure solve and the
 * explicit stencil residuals of arxiv/paper_2401_06755 (NN4PDEs multiphase flow).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may build, load or call it.  It
 * shares no code, header, table or constant generator with the CUDA path under
 * paper_2401_06755_b200/csrc/, and neither includes the other.
 *
 * Every function is written as nested loops over (k, j, i) with an explicit ghost()
 * evaluation of halo values, in the order and notation of the paper.  "P:NNN" is a line
 * of /root/reference/PAPER.md.  Readings of silent / garbled passages are those of
 * DESIGN.md ("Readings").
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): Eq. 11's printed weights, the closed
 * form discrete eigenpair, 2nd-order manufactured solution, symmetry, constant null space,
 * literal Eq. 13 == collapsed difference form, dense direct solves on <= 8^3, Fourier-mode
 * Jacobi factors, transfer adjointness, hand-computed VoF cases, the hand-reduced 1-D momentum scheme
 * (both branches of min{k_max, k_abs} of Eqs. 30-32 under varying rho and mu), and -- for the step composition in
 * oracle/__init__.py -- the stages chained by hand, the potential-flow property of stage 4 (Eq. 16 advects with
 * u^{n+1}) and the second-order accuracy of the two predictor iterations (tests/test_oracle_step.py).
 * The limit of the volume fraction in the material mixtures (reading C7, mix01 below): closed-form k values, bit-identity of
 * every rho / mu consumer under limiting, and the scaling law that shows the surface-tension terms are NOT limited.
 * PARITY UNPINNED against the paper (no worked example exists in its text): the transfer
 * operators / coarse operator (Fig. 5 is an image), the momentum residual without the
 * missing Eq. 28, and vof_residual beyond its hand-computable special cases.
 *
 * Layout: dense, x fastest: idx = i + nx*(j + ny*k); no halo in arrays.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { int nx, ny, nz; double hx, hy, hz; } orc_grid;

/* boundary codes -> ghost factor s (reading C3):
 * 0 Neumann (copy, s=+1); 1 Dirichlet zero on the cell face (s=-1); 2 Dirichlet halo value 0 (s=0) */
static double bc_factor(int code) { return code == 0 ? 1.0 : (code == 1 ? -1.0 : 0.0); }

static const int BC_COPY[6] = {0, 0, 0, 0, 0, 0};

#define IDX(g, i, j, k) ((size_t)(i) + (size_t)(g)->nx * ((size_t)(j) + (size_t)(g)->ny * (size_t)(k)))

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Halo value of field f at a (possibly out-of-box) index: reflect about the face
 * (-1 -> 0, n -> n-1) and multiply the face factors; edges and corners reflect
 * successively so the factors multiply (Fig. 2). */
static double ghost(const double* f, const orc_grid* g, const int* bc, int i, int j, int k) {
    double s = 1.0;
    if (i < 0) { i = -1 - i; s *= bc_factor(bc[0]); } else if (i >= g->nx) { i = 2 * g->nx - 1 - i; s *= bc_factor(bc[1]); }
    if (j < 0) { j = -1 - j; s *= bc_factor(bc[2]); } else if (j >= g->ny) { j = 2 * g->ny - 1 - j; s *= bc_factor(bc[3]); }
    if (k < 0) { k = -1 - k; s *= bc_factor(bc[4]); } else if (k >= g->nz) { k = 2 * g->nz - 1 - k; s *= bc_factor(bc[5]); }
    return s * f[IDX(g, i, j, k)];
}

/* ------------------------------------------------------------------------------------
 * Filters (Eqs. 9-11).  All are NODAL, i.e. the
 * paper's integrated filter divided by m_l = dx dy dz (its own w_ml^-1).
 * 1-D factors of the trilinear element on a uniform line of spacing d:
 *   stiffness  K = (1/d) [-1, 2, -1],  consistent mass M = (d/6) [1, 4, 1],
 *   derivative D = (1/2) [-1, 0, 1]   (int N_i dN_j/dx).
 * w[(ii+1) + 3*(jj+1) + 9*(kk+1)], ii along x.
 * which: 0 w_lap = (KMM + MKM + MMK)/m_l     (-Laplacian, positive definite; reading C1)
 *        1 w_x, 2 w_y, 3 w_z                 (Eq. 11 / m_l)
 *        4 w_xx, 5 w_yy, 6 w_zz              (the three summands of w_lap)
 *        7 w_m / m_l                         (consistent mass, MMM / m_l)
 * ------------------------------------------------------------------------------------ */
void orc_filter(const orc_grid* g, int which, double* w) {
    const double h[3] = {g->hx, g->hy, g->hz};
    double K[3][3], M[3][3], D[3][3];
    for (int d = 0; d < 3; ++d) {
        K[d][0] = -1.0 / h[d]; K[d][1] = 2.0 / h[d]; K[d][2] = -1.0 / h[d];
        M[d][0] = h[d] / 6.0;  M[d][1] = 4.0 * h[d] / 6.0; M[d][2] = h[d] / 6.0;
        D[d][0] = -0.5;        D[d][1] = 0.0;        D[d][2] = 0.5;
    }
    const double ml = h[0] * h[1] * h[2];
    for (int kk = 0; kk < 3; ++kk)
        for (int jj = 0; jj < 3; ++jj)
            for (int ii = 0; ii < 3; ++ii) {
                const double xx = K[0][ii] * M[1][jj] * M[2][kk];
                const double yy = M[0][ii] * K[1][jj] * M[2][kk];
                const double zz = M[0][ii] * M[1][jj] * K[2][kk];
                double v = 0.0;
                switch (which) {
                    case 0: v = xx + yy + zz; break;
                    case 1: v = D[0][ii] * M[1][jj] * M[2][kk]; break;
                    case 2: v = M[0][ii] * D[1][jj] * M[2][kk]; break;
                    case 3: v = M[0][ii] * M[1][jj] * D[2][kk]; break;
                    case 4: v = xx; break;
                    case 5: v = yy; break;
                    case 6: v = zz; break;
                    case 7: v = M[0][ii] * M[1][jj] * M[2][kk]; break;
                }
                w[ii + 3 * jj + 9 * kk] = v / ml;
            }
}

/* f(C; w), Eq. 8: y_ijk = sum_{ii,jj,kk} w_{ii,jj,kk} C_{i+ii,j+jj,k+kk}, halo by ghost(). */
void orc_apply_filter(const orc_grid* g, const int* bc, const double* w, const double* C, double* y) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                double s = 0.0;
                for (int kk = -1; kk <= 1; ++kk)
                    for (int jj = -1; jj <= 1; ++jj)
                        for (int ii = -1; ii <= 1; ++ii)
                            s += w[(ii + 1) + 3 * (jj + 1) + 9 * (kk + 1)] * ghost(C, g, bc, i + ii, j + jj, k + kk);
                y[IDX(g, i, j, k)] = s;
            }
}

/* ------------------------------------------------------------------------------------
 * Operator y = A x (SURVEY/DESIGN C1, C2).
 *   kcoef == NULL : y = f(x; w_lap)                                    (Eq. 8 with w_lap)
 *   kcoef != NULL : y_i = sum_{j != i} (-w_ij) * 1/2 (k_i + k_j) (x_i - x_j)
 * the exact collapse of Eq. 13 because sum_j w_ij = 0.  Halo of x by the BC
 * factors, halo of k by copy.  w is any second-derivative filter (w_lap, w_xx...).
 * ------------------------------------------------------------------------------------ */
void orc_apply_diffusion(const orc_grid* g, const int* bc, const double* w, const double* kcoef,
                         const double* x, double* y) {
    if (!kcoef) { orc_apply_filter(g, bc, w, x, y); return; }
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                const double xi = x[IDX(g, i, j, k)], ki = kcoef[IDX(g, i, j, k)];
                double s = 0.0;
                for (int kk = -1; kk <= 1; ++kk)
                    for (int jj = -1; jj <= 1; ++jj)
                        for (int ii = -1; ii <= 1; ++ii) {
                            if (ii == 0 && jj == 0 && kk == 0) continue;
                            const double wij = w[(ii + 1) + 3 * (jj + 1) + 9 * (kk + 1)];
                            const double xj = ghost(x, g, bc, i + ii, j + jj, k + kk);
                            const double kj = ghost(kcoef, g, BC_COPY, i + ii, j + jj, k + kk);
                            s += (-wij) * 0.5 * (ki + kj) * (xi - xj);
                        }
                y[IDX(g, i, j, k)] = s;
            }
}

void orc_apply_operator(const orc_grid* g, const int* bc, const double* kcoef, const double* x, double* y) {
    double w[27];
    orc_filter(g, 0, w);
    orc_apply_diffusion(g, bc, w, kcoef, x, y);
}

/* Literal Eq. 13: 1/2 ( f(k.C; w) + k.f(C; w) - C.f(k; w) ), three stencils.
 * Halo of the product field k.C is ghost(k)*ghost(C).  Used only to pin the collapsed form. */
void orc_apply_operator_eq13(const orc_grid* g, const int* bc, const double* kcoef, const double* x, double* y) {
    double w[27];
    orc_filter(g, 0, w);
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                double fkc = 0.0, fc = 0.0, fk = 0.0;
                for (int kk = -1; kk <= 1; ++kk)
                    for (int jj = -1; jj <= 1; ++jj)
                        for (int ii = -1; ii <= 1; ++ii) {
                            const double wij = w[(ii + 1) + 3 * (jj + 1) + 9 * (kk + 1)];
                            const double xj = ghost(x, g, bc, i + ii, j + jj, k + kk);
                            const double kj = ghost(kcoef, g, BC_COPY, i + ii, j + jj, k + kk);
                            fkc += wij * (kj * xj); fc += wij * xj; fk += wij * kj;
                        }
                const size_t c = IDX(g, i, j, k);
                y[c] = 0.5 * (fkc + kcoef[c] * fc - x[c] * fk);
            }
}

/* Jacobi "diagonal" (reading C2-2): the centre coefficient of the conv-layer view,
 * D_i = sum_{j != i} (-w_ij) 1/2 (k_i + k_j) over all 26 positions, ghosts included;
 * constant coefficient: D = w_000. */
void orc_diagonal(const orc_grid* g, const double* kcoef, double* D) {
    double w[27];
    orc_filter(g, 0, w);
#pragma omp parallel for schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                if (!kcoef) { D[IDX(g, i, j, k)] = w[13]; continue; }
                const double ki = kcoef[IDX(g, i, j, k)];
                double s = 0.0;
                for (int kk = -1; kk <= 1; ++kk)
                    for (int jj = -1; jj <= 1; ++jj)
                        for (int ii = -1; ii <= 1; ++ii) {
                            if (ii == 0 && jj == 0 && kk == 0) continue;
                            const double kj = ghost(kcoef, g, BC_COPY, i + ii, j + jj, k + kk);
                            s += (-w[(ii + 1) + 3 * (jj + 1) + 9 * (kk + 1)]) * 0.5 * (ki + kj);
                        }
                D[IDX(g, i, j, k)] = s;
            }
}

/* ------------------------------------------------------------------------------------
 * Weighted Jacobi (reading C4): x' = x + omega (b - A x) / D, every
 * point from the OLD x (two buffers).  xnew must not alias x.
 * ------------------------------------------------------------------------------------ */
void orc_jacobi_sweep(const orc_grid* g, const int* bc, const double* kcoef, const double* x,
                      const double* b, double omega, double* xnew) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double* Ax = (double*)malloc(n * sizeof(double));
    double* D = (double*)malloc(n * sizeof(double));
    orc_apply_operator(g, bc, kcoef, x, Ax);
    orc_diagonal(g, kcoef, D);
    for (size_t c = 0; c < n; ++c) xnew[c] = x[c] + omega * (b[c] - Ax[c]) / D[c];
    free(Ax); free(D);
}

/* `sweeps` sweeps in place (ping-pong through a scratch copy). */
void orc_smooth(const orc_grid* g, const int* bc, const double* kcoef, double* x, const double* b,
                double omega, int sweeps) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double* t = (double*)malloc(n * sizeof(double));
    for (int s = 0; s < sweeps; ++s) {
        orc_jacobi_sweep(g, bc, kcoef, x, b, omega, t);
        memcpy(x, t, n * sizeof(double));
    }
    free(t);
}

void orc_residual(const orc_grid* g, const int* bc, const double* kcoef, const double* x,
                  const double* b, double* r) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    orc_apply_operator(g, bc, kcoef, x, r);
    for (size_t c = 0; c < n; ++c) r[c] = b[c] - r[c];
}

/* ------------------------------------------------------------------------------------
 * Transfers (Fig. 5 caption P:417; reading C5 -- the paper gives no weights):
 * restriction = mean of the 8 children (stride-2 2x2x2 filter, weights 1/8);
 * prolongation = piecewise constant (nearest-neighbour upsampling x2), added to x.
 * gc is the coarse grid: n/2 in each direction, spacing 2h.
 * ------------------------------------------------------------------------------------ */
void orc_coarse_grid(const orc_grid* gf, orc_grid* gc) {
    gc->nx = gf->nx / 2; gc->ny = gf->ny / 2; gc->nz = gf->nz / 2;
    gc->hx = 2.0 * gf->hx; gc->hy = 2.0 * gf->hy; gc->hz = 2.0 * gf->hz;
}

void orc_restrict(const orc_grid* gf, const double* rf, double* rc) {
    orc_grid gc; orc_coarse_grid(gf, &gc);
    for (int k = 0; k < gc.nz; ++k)
        for (int j = 0; j < gc.ny; ++j)
            for (int i = 0; i < gc.nx; ++i) {
                double s = 0.0;
                for (int dk = 0; dk < 2; ++dk)
                    for (int dj = 0; dj < 2; ++dj)
                        for (int di = 0; di < 2; ++di)
                            s += rf[IDX(gf, 2 * i + di, 2 * j + dj, 2 * k + dk)];
                rc[IDX(&gc, i, j, k)] = 0.125 * s;
            }
}

void orc_prolong_add(const orc_grid* gf, const double* xc, double* xf) {
    orc_grid gc; orc_coarse_grid(gf, &gc);
    for (int k = 0; k < gf->nz; ++k)
        for (int j = 0; j < gf->ny; ++j)
            for (int i = 0; i < gf->nx; ++i)
                xf[IDX(gf, i, j, k)] += xc[IDX(&gc, i / 2, j / 2, k / 2)];
}

/* Material property of the one-fluid model, Eqs. 2 and 19: a = a_l C + a_g (1 - C), with C limited to [0, 1]
 * first (reading C7, revised in round 2: the paper does not clip, and says of its scheme only that it "reduces the
 * likelihood" of C leaving [0, 1]; an undershoot C = -0.003 gives rho < 0 at rho_g / rho_l = 1e-3 and the pressure
 * operator loses definiteness).  Only the mixtures rho and mu see the limited value; gradients, curvature and the VoF scheme
 * use C as it is. */
static inline double mix01(double al, double ag, double C) {
    const double c = C < 0.0 ? 0.0 : (C > 1.0 ? 1.0 : C);
    return al * c + ag * (1.0 - c);
}

/* k = 1 / rho(alpha), Eqs. 2 and 19, alpha limited to [0, 1] (C7). */
void orc_k_from_vof(size_t n, const double* alpha, double rho_l, double rho_g, double* kcoef) {
    for (size_t c = 0; c < n; ++c) kcoef[c] = 1.0 / mix01(rho_l, rho_g, alpha[c]);
}

/* ------------------------------------------------------------------------------------
 * V-cycle (Fig. 5; reading C6).  Coarse operators are rediscretised with
 * spacing 2h and the same BC factors; coarse coefficient = arithmetic mean of the
 * 8 children.  The coarsest level runs `coarse_sweeps` Jacobi sweeps on the incoming guess.
 *   vcycle(l,x,b): if coarsest: n_c sweeps; return
 *                  nu1 sweeps; r = b - A x; b_c = R r; x_c = 0; vcycle(l+1,x_c,b_c);
 *                  x += P x_c; nu2 sweeps
 * ------------------------------------------------------------------------------------ */
void orc_vcycle(const orc_grid* g, const int* bc, const double* kcoef, int levels, int nu_pre, int nu_post,
                int coarse_sweeps, double omega, double* x, const double* b) {
    if (levels <= 1) { orc_smooth(g, bc, kcoef, x, b, omega, coarse_sweeps); return; }
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    orc_grid gc; orc_coarse_grid(g, &gc);
    const size_t nc = (size_t)gc.nx * gc.ny * gc.nz;
    double* r = (double*)malloc(n * sizeof(double));
    double* bcz = (double*)malloc(nc * sizeof(double));
    double* xc = (double*)calloc(nc, sizeof(double));
    double* kc = kcoef ? (double*)malloc(nc * sizeof(double)) : NULL;
    if (kcoef) orc_restrict(g, kcoef, kc);
    orc_smooth(g, bc, kcoef, x, b, omega, nu_pre);
    orc_residual(g, bc, kcoef, x, b, r);
    orc_restrict(g, r, bcz);
    orc_vcycle(&gc, bc, kc, levels - 1, nu_pre, nu_post, coarse_sweeps, omega, xc, bcz);
    orc_prolong_add(g, xc, x);
    orc_smooth(g, bc, kcoef, x, b, omega, nu_post);
    free(r); free(bcz); free(xc); free(kc);
}

double orc_norm2(size_t n, const double* v) {
    double s = 0.0;
    for (size_t c = 0; c < n; ++c) s += v[c] * v[c];
    return sqrt(s);
}

/* Repeat V-cycles until ||b - A x||_2 / ||b||_2 < tol (the paper runs a fixed 20; the
 * tolerance is BASELINE.json's).  history (may be NULL) receives the relative residual after
 * every cycle (max_cycles entries).  Returns the number of cycles run. */
int orc_solve(const orc_grid* g, const int* bc, const double* kcoef, int levels, int nu_pre, int nu_post,
              int coarse_sweeps, double omega, double* x, const double* b, double tol, int max_cycles,
              double* history, double* relres_out) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double* r = (double*)malloc(n * sizeof(double));
    const double nb = orc_norm2(n, b);
    double rel = 0.0;
    int c = 0;
    orc_residual(g, bc, kcoef, x, b, r);
    rel = nb > 0.0 ? orc_norm2(n, r) / nb : 0.0;
    while (c < max_cycles && !(rel < tol)) {
        orc_vcycle(g, bc, kcoef, levels, nu_pre, nu_post, coarse_sweeps, omega, x, b);
        orc_residual(g, bc, kcoef, x, b, r);
        rel = orc_norm2(n, r) / nb;
        if (history) history[c] = rel;
        ++c;
    }
    if (relres_out) *relres_out = rel;
    free(r);
    return c;
}

/* ------------------------------------------------------------------------------------
 * V-cycle-preconditioned conjugate gradients (SURVEY 8(f) "next 1").
 * NOT in the paper, which always runs plain cycles; it is the standard remedy for
 * the slow convergence of those cycles under a 1000:1 coefficient jump (SURVEY hard part 4).
 * Textbook preconditioned CG for the symmetric positive definite system A x = b, the
 * preconditioner z = M r being ONE V(nu, nu) cycle on A z = r from z = 0 (symmetric because
 * nu_pre = nu_post, the Jacobi smoother is symmetric and R = P^T / 8):
 *   r = b - A x;  z = M r;  p = z;  rz = <r, z>
 *   repeat:  q = A p;  alpha = rz / <p, q>;  x += alpha p;  r -= alpha q;
 *            stop if ||r||_2 / ||b||_2 < tol;
 *            z = M r;  rz' = <r, z>;  beta = rz' / rz;  p = z + beta p;  rz = rz'
 * history (may be NULL) receives the relative residual after every iteration.  Returns the
 * number of iterations (= V-cycles after the first).
 * ------------------------------------------------------------------------------------ */
static double dot(size_t n, const double* a, const double* b) {
    double s = 0.0;
    for (size_t c = 0; c < n; ++c) s += a[c] * b[c];
    return s;
}

int orc_pcg_solve(const orc_grid* g, const int* bc, const double* kcoef, int levels, int nu, int coarse_sweeps,
                  double omega, double* x, const double* b, double tol, int max_iter, double* history,
                  double* relres_out) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double* r = (double*)malloc(n * sizeof(double));
    double* z = (double*)malloc(n * sizeof(double));
    double* p = (double*)malloc(n * sizeof(double));
    double* q = (double*)malloc(n * sizeof(double));
    const double nb = orc_norm2(n, b);
    int it = 0;
    orc_residual(g, bc, kcoef, x, b, r);
    double rel = nb > 0.0 ? orc_norm2(n, r) / nb : 0.0;
    if (!(rel < tol) && max_iter > 0) {
        memset(z, 0, n * sizeof(double));
        orc_vcycle(g, bc, kcoef, levels, nu, nu, coarse_sweeps, omega, z, r);
        memcpy(p, z, n * sizeof(double));
        double rz = dot(n, r, z);
        while (it < max_iter) {
            orc_apply_operator(g, bc, kcoef, p, q);
            const double alpha = rz / dot(n, p, q);
            for (size_t c = 0; c < n; ++c) { x[c] += alpha * p[c]; r[c] -= alpha * q[c]; }
            rel = orc_norm2(n, r) / nb;
            if (history) history[it] = rel;
            ++it;
            if (rel < tol) break;
            memset(z, 0, n * sizeof(double));
            orc_vcycle(g, bc, kcoef, levels, nu, nu, coarse_sweeps, omega, z, r);
            const double rz_new = dot(n, r, z);
            const double beta = rz_new / rz;
            for (size_t c = 0; c < n; ++c) p[c] = z[c] + beta * p[c];
            rz = rz_new;
        }
    }
    if (relres_out) *relres_out = rel;
    free(r); free(z); free(p); free(q);
    return it;
}

/* ====================================================================================
 * Explicit stencil residuals that feed the pressure solve.
 * All derived fields are nodal (divided by m_l); halos of C, of the velocities and of every
 * derived field are zero-derivative copies (reading C9-iv).
 * ==================================================================================== */

/* Eqs. 26/27: first residual-based PG diffusion coefficient, p = 1 so
 * alpha_kabs = 1/(8*2^p) = 1/16, eps_k = 1e-7.  Uniform spacing uses
 * Eq. 27, otherwise Eq. 26 (reading C9-ii). */
static double k_abs_pg(const orc_grid* g, double a, double px, double py, double pz) {
    const double alpha_kabs = 1.0 / 16.0, eps_k = 1e-7;
    const double s = fabs(px) + fabs(py) + fabs(pz);
    if (g->hx == g->hy && g->hy == g->hz) return alpha_kabs * g->hx * fabs(a) / (eps_k + s / 3.0);
    return alpha_kabs * fabs(a) * (g->hx * fabs(px) + g->hy * fabs(py) + g->hz * fabs(pz)) / (eps_k + s * s / 3.0);
}

/* Gradient by the linear-FE filters (Eq. 11 / m_l) and the advection term q . grad(Psi). */
static void grad_and_adv_bc(const orc_grid* g, const int* bc, const double* psi, const double* u, const double* v, const double* w,
                            double* px, double* py, double* pz, double* adv) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wx[27], wy[27], wz[27];
    orc_filter(g, 1, wx); orc_filter(g, 2, wy); orc_filter(g, 3, wz);
    orc_apply_filter(g, bc, wx, psi, px);
    orc_apply_filter(g, bc, wy, psi, py);
    orc_apply_filter(g, bc, wz, psi, pz);
    for (size_t c = 0; c < n; ++c) adv[c] = u[c] * px[c] + v[c] * py[c] + w[c] * pz[c];
}
static void grad_and_adv(const orc_grid* g, const double* psi, const double* u, const double* v, const double* w,
                         double* px, double* py, double* pz, double* adv) {
    grad_and_adv_bc(g, BC_COPY, psi, u, v, w, px, py, pz, adv);
}

/* Eq. 29: a = alpha_a f(adv; w_m/m_l - E), alpha_a = 2. */
static void mixed_mass_residual(const orc_grid* g, const double* adv, double* a) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wm[27];
    orc_filter(g, 7, wm);
    wm[13] -= 1.0; /* minus the identity filter E */
    orc_apply_filter(g, BC_COPY, wm, adv, a);
    for (size_t c = 0; c < n; ++c) a[c] *= 2.0;
}

/* vof_residual (reading C9, steps 1-12): sC = nodal s~_C of Eq. 16;
 * Cnew (may be NULL) = C - dt sC, Eq. 55. */
/* detector = 3: Eq. 33 (linear 3 x 3 x 3 filters);  detector = 5: the 5-point oscillation detectors of Eq. 34, the
 * minimum of the three products of consecutive differences over i-2 .. i+2 ("a much more rigorous approach to detecting an
 * oscillation") -- SURVEY 8(f) next 4, the part of the higher-order scheme the paper prints in full.  Halo of C: copy,
 * i.e. reflection about the face for the second ghost layer as well (-1 -> 0, -2 -> 1). */
void orc_vof_residual_ex(const orc_grid* g, const double* C, const double* u, const double* v, const double* w,
                         double dt, int detector, double* sC, double* Cnew) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    const double Kp = 300.0, Km = 300.0;          /* K+, K-  */
    const double beta = 0.1, eps_x = 1e-4;        /* Eq. 36 */
    const double Kcal = 3.0;                      /* Eq. 39 */
    const double a_min = 1e-4, a_max = 0.05;      /* Eq. 42 */
    const double hmax = fmax(g->hx, fmax(g->hy, g->hz)), hmin = fmin(g->hx, fmin(g->hy, g->hz));
    const double k_min = a_min / dt * hmax * hmax, k_max = a_max / dt * hmin * hmin;
    const double hd[3] = {g->hx, g->hy, g->hz};
    double* Cx = (double*)malloc(n * sizeof(double)); double* Cy = (double*)malloc(n * sizeof(double));
    double* Cz = (double*)malloc(n * sizeof(double)); double* adv = (double*)malloc(n * sizeof(double));
    double* a = (double*)malloc(n * sizeof(double));
    double* kd[3]; double* diff = (double*)malloc(n * sizeof(double));
    for (int d = 0; d < 3; ++d) kd[d] = (double*)malloc(n * sizeof(double));

    grad_and_adv(g, C, u, v, w, Cx, Cy, Cz, adv);            /* steps 1-2 */
    mixed_mass_residual(g, adv, a);                          /* step 3 */
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                const size_t c = IDX(g, i, j, k);
                const double kabs = k_abs_pg(g, a[c], Cx[c], Cy[c], Cz[c]);          /* step 4 */
                /* step 5: Eq. 33 + override */
                const double C0 = C[c];
                double S[3];
                S[0] = (C0 - ghost(C, g, BC_COPY, i - 1, j, k)) * (ghost(C, g, BC_COPY, i + 1, j, k) - C0);
                S[1] = (C0 - ghost(C, g, BC_COPY, i, j - 1, k)) * (ghost(C, g, BC_COPY, i, j + 1, k) - C0);
                S[2] = (C0 - ghost(C, g, BC_COPY, i, j, k - 1)) * (ghost(C, g, BC_COPY, i, j, k + 1) - C0);
                if (detector == 5) {                                                 /* Eq. 34 */
                    const int di[3] = {1, 0, 0}, dj[3] = {0, 1, 0}, dk[3] = {0, 0, 1};
                    for (int d = 0; d < 3; ++d) {
                        double cv[5];
                        for (int m = -2; m <= 2; ++m) cv[m + 2] = ghost(C, g, BC_COPY, i + m * di[d], j + m * dj[d], k + m * dk[d]);
                        const double p0 = (cv[1] - cv[0]) * (cv[2] - cv[1]);
                        const double p1 = (cv[2] - cv[1]) * (cv[3] - cv[2]);
                        const double p2 = (cv[3] - cv[2]) * (cv[4] - cv[3]);
                        S[d] = fmin(p0, fmin(p1, p2));
                    }
                }
                if (C0 > 0.95 || C0 < 0.05) S[0] = S[1] = S[2] = -1.0;
                /* step 7: Eq. 37 */
                const double g2 = Cx[c] * Cx[c] + Cy[c] * Cy[c] + Cz[c] * Cz[c];
                const double gq = (u[c] * Cx[c] + v[c] * Cy[c] + w[c] * Cz[c]) / (eps_x + g2);
                const double us = gq * Cx[c], vs = gq * Cy[c], ws = gq * Cz[c];
                /* step 8: Eq. 36 */
                const double kneg = -beta * (u[c] * u[c] + v[c] * v[c] + w[c] * w[c]) /
                                    (eps_x + g2 * (fabs(us) + fabs(vs) + fabs(ws)) / 3.0);
                for (int d = 0; d < 3; ++d) {
                    const double wp = -fmax(-1.0, fmin(0.0, Kp * S[d]));             /* step 6: Eq. 35 */
                    const double wm = fmin(1.0, fmax(0.0, Km * S[d]));
                    const double kplus = Kcal * kabs;                                /* step 9: Eq. 39 */
                    const double kminus = kneg / hd[d];                              /* Eq. 38 */
                    const double kk = wp * kplus + wm * kminus;                      /* Eq. 40 */
                    kd[d][c] = fmax(-k_min, fmin(k_max, kk));                        /* step 10: Eq. 41 */
                }
            }
    for (size_t c = 0; c < n; ++c) sC[c] = adv[c];
    for (int d = 0; d < 3; ++d) {                                                    /* step 11: Eq. 12 collapsed */
        double wdd[27];
        orc_filter(g, 4 + d, wdd);
        orc_apply_diffusion(g, BC_COPY, wdd, kd[d], C, diff);
        for (size_t c = 0; c < n; ++c) sC[c] += diff[c];
    }
    if (Cnew) for (size_t c = 0; c < n; ++c) Cnew[c] = C[c] - dt * sC[c];            /* step 12: Eq. 55 */
    free(Cx); free(Cy); free(Cz); free(adv); free(a); free(diff);
    for (int d = 0; d < 3; ++d) free(kd[d]);
}
void orc_vof_residual(const orc_grid* g, const double* C, const double* u, const double* v, const double* w,
                      double dt, double* sC, double* Cnew) {
    orc_vof_residual_ex(g, C, u, v, w, dt, 3, sC, Cnew);
}

/* Momentum advection-diffusion residual and predictor (Eqs. 18, 30-32, 45-46; P:198-220,
 * 309-319, 433-441; reading C9 "Momentum").  For each component c of the half-level velocity:
 *   s~_c = rho (q_h . grad c_h) + f^lap(c_h, k_c; w_lap),  k_c = rho min{k_max, k_abs(c_h)} + mu,
 *   k_max = dx|u_h| + dy|v_h| + dz|w_h| (Eq. 30);  k_square of the lost Eq. 28 is omitted;
 *   c~ = c_n - dt s~_c / rho (Eq. 45, sigma = 0);  c_half' = (c_n + c~)/2 (Eq. 46).
 * Pressure-gradient and source terms of Eq. 18 are not part of this residual.
 * qh/qn/qt/qhn are arrays of 3 component pointers (u, v, w). */
/* vbc = NULL: every velocity halo is a zero-derivative copy (BASELINE config 5's synthetic benchmark).  Otherwise
 * vbc[6 * c + f] is the halo code of velocity component c on face f: free-slip walls make the component NORMAL to a
 * wall odd about it (ghost = -mirror: zero normal velocity on the wall face, the interpolation rule of Fig. 2) and the
 * tangential components even (zero normal derivative); at an outlet every component is copied.  The halo of a
 * component enters its gradient (the advection term) and its diffusion; derived fields keep copy halos (reading C9-iv). */
void orc_mom_predictor_bc(const orc_grid* g, const double* C, const double* const* qh, const double* const* qn, const int* vbc,
                          double rho_l, double rho_g, double mu_l, double mu_g, double dt,
                          double* const* qt, double* const* qhn) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wl[27];
    orc_filter(g, 0, wl);
    double* px = (double*)malloc(n * sizeof(double)); double* py = (double*)malloc(n * sizeof(double));
    double* pz = (double*)malloc(n * sizeof(double)); double* adv = (double*)malloc(n * sizeof(double));
    double* a = (double*)malloc(n * sizeof(double)); double* kc = (double*)malloc(n * sizeof(double));
    double* diff = (double*)malloc(n * sizeof(double));
    for (int comp = 0; comp < 3; ++comp) {
        const int* cbc = vbc ? vbc + 6 * comp : BC_COPY;
        grad_and_adv_bc(g, cbc, qh[comp], qh[0], qh[1], qh[2], px, py, pz, adv);
        mixed_mass_residual(g, adv, a);
        for (size_t c = 0; c < n; ++c) {
            const double rho = mix01(rho_l, rho_g, C[c]);
            const double mu = mix01(mu_l, mu_g, C[c]);
            const double kmax = g->hx * fabs(qh[0][c]) + g->hy * fabs(qh[1][c]) + g->hz * fabs(qh[2][c]);
            const double kabs = k_abs_pg(g, a[c], px[c], py[c], pz[c]);
            kc[c] = rho * fmin(kmax, kabs) + mu;
        }
        orc_apply_diffusion(g, cbc, wl, kc, qh[comp], diff);
        for (size_t c = 0; c < n; ++c) {
            const double rho = mix01(rho_l, rho_g, C[c]);
            const double s = rho * adv[c] + diff[c];
            const double t = qn[comp][c] - dt * s / rho;
            qt[comp][c] = t;
            if (qhn) qhn[comp][c] = 0.5 * (qn[comp][c] + t);
        }
    }
    free(px); free(py); free(pz); free(adv); free(a); free(kc); free(diff);
}

void orc_mom_predictor(const orc_grid* g, const double* C, const double* const* qh, const double* const* qn,
                       double rho_l, double rho_g, double mu_l, double mu_g, double dt,
                       double* const* qt, double* const* qhn) {
    orc_mom_predictor_bc(g, C, qh, qn, NULL, rho_l, rho_g, mu_l, mu_g, dt, qt, qhn);
}

/* Pressure RHS (reading C10; FE divergence structure of Eq. 53):
 * b = -(1/dt) ( f(u~; w_x) + f(v~; w_y) + f(w~; w_z) ), nodal filters, velocity halos copy. */
void orc_pressure_rhs_bc(const orc_grid* g, const double* u, const double* v, const double* w, const int* vbc, double dt, double* b) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wx[27], wy[27], wz[27];
    orc_filter(g, 1, wx); orc_filter(g, 2, wy); orc_filter(g, 3, wz);
    double* t = (double*)malloc(n * sizeof(double));
    orc_apply_filter(g, vbc ? vbc : BC_COPY, wx, u, b);
    orc_apply_filter(g, vbc ? vbc + 6 : BC_COPY, wy, v, t); for (size_t c = 0; c < n; ++c) b[c] += t[c];
    orc_apply_filter(g, vbc ? vbc + 12 : BC_COPY, wz, w, t); for (size_t c = 0; c < n; ++c) b[c] = -(b[c] + t[c]) / dt;
    free(t);
}
void orc_pressure_rhs(const orc_grid* g, const double* u, const double* v, const double* w, double dt, double* b) {
    orc_pressure_rhs_bc(g, u, v, w, NULL, dt, b);     /* velocity halos: copies */
}

/* The PAPER'S OWN stage-3 right-hand side, Eqs. 52-53 (SURVEY 8(f) "next 2"): the density stays on the right and
 * the Laplacian is constant-coefficient,
 *   b = -(1/dt) ( f(rho.u~; w_x) + f(rho.v~; w_y) + f(rho.w~; w_z) )
 *       +(1/dt) ( u~.f(rho; w_x) + v~.f(rho; w_y) + w~.f(rho; w_z) ),     rho = rho_l C + rho_g (1 - C)  (Eq. 2),
 * each term written as its own filter application, exactly as Eq. 53 prints them; halos are copies.
 * With A = f(.; w_lap) positive definite (reading C1-2) the system solved is  A dp = b. */
void orc_pressure_rhs_paper(const orc_grid* g, const double* C, const double* u, const double* v, const double* w,
                            double rho_l, double rho_g, double dt, double* b) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wx[27], wy[27], wz[27];
    orc_filter(g, 1, wx); orc_filter(g, 2, wy); orc_filter(g, 3, wz);
    double* rho = (double*)malloc(n * sizeof(double));
    double* m = (double*)malloc(n * sizeof(double));
    double* t = (double*)malloc(n * sizeof(double));
    for (size_t c = 0; c < n; ++c) { rho[c] = mix01(rho_l, rho_g, C[c]); b[c] = 0.0; }
    const double* vel[3] = {u, v, w};
    const double* flt[3] = {wx, wy, wz};
    for (int d = 0; d < 3; ++d) {
        for (size_t c = 0; c < n; ++c) m[c] = rho[c] * vel[d][c];
        orc_apply_filter(g, BC_COPY, flt[d], m, t);                       /* f(rho q; w_d) */
        for (size_t c = 0; c < n; ++c) b[c] -= t[c] / dt;
        orc_apply_filter(g, BC_COPY, flt[d], rho, t);                     /* q . f(rho; w_d) */
        for (size_t c = 0; c < n; ++c) b[c] += vel[d][c] * t[c] / dt;
    }
    free(rho); free(m); free(t);
}

/* ------------------------------------------------------------------------------------
 * Stage 1, hydrostatic and surface-tension pressure (SURVEY 8(f) "next 3"; Eqs. 4-5, Eqs. 20-23,
 * P:419-427 Eqs. 43-44, bottom boundary condition P:258).
 *   C_x, C_y, C_z = nodal FE gradient of C;  l = |grad C|;  n_t = grad C / (eps_t + l),  eps_t = 1e-7 / h     (Eq. 23)
 *   kappa = -( f(n_tu; w_x) + f(n_tv; w_y) + f(n_tw; w_z) )   (nodal: Eq. 22's w_ml^-1; sign: see below)    (Eqs. 5, 22)
 *   s_t = sigma_t kappa grad C                                                                              (Eqs. 4, 21)
 *   A p_hs = b_hs,  b_hs = f(g rho; w_z) - ( f(s_tu; w_x) + f(s_tv; w_y) + f(s_tw; w_z) )                   (Eq. 43)
 * Readings (N3): Eq. 22 prints n_tu three times and Eq. 23 prints C_x for n_tw -- read as the divergence of
 * (n_tu, n_tv, n_tw) with n_tw from C_z (Eq. 5).  The signs of Eq. 5 (kappa = +div n_t), Eq. 43 and Eq. 44 cannot all hold:
 * with kappa = +div n_t the force sigma kappa grad C points OUT of a drop, Eq. 43 (which is what balances the momentum
 * equation 17: grad p_hs = s_q + s_t) then puts the lower pressure inside, and Eq. 44 has the opposite sign of Eq. 43 on the
 * surface-tension term.  The reading taken is the one that satisfies the physics the paper names (continuum surface force
 * [15], Young-Laplace): kappa = -div n_t, with Eq. 43 and Eq. 17 as printed.  Numerically b_hs is then exactly what Eq. 44
 * as printed gives with Eq. 5 as printed (the two sign slips cancel).  Pinned: dp/dz = -rho g, kappa = +2/r on a sphere,
 * force towards the centre, pressure higher inside by 2 sigma / R.
 * h in eps_t is hx.  Halos of C, n_t, s_t and rho are copies (reading C9-iv).
 * Bottom boundary condition dp_hs/dz = -rho g: the ghost below the bottom plane is p + hz rho g with the density of
 * the nearest node, so its contribution sum_j (-w_ij) hz g rho_j over the ghost plane is added to b on the bottom plane;
 * the solver then treats that face as zero-derivative (copy).
 * kappa_out, st_out[3] may be NULL.
 * ------------------------------------------------------------------------------------ */
void orc_hydrostatic_rhs(const orc_grid* g, const double* C, double rho_l, double rho_g, double grav, double sigma_t,
                         double* b, double* kappa_out, double* const* st_out) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wx[27], wy[27], wz[27], wl[27];
    orc_filter(g, 1, wx); orc_filter(g, 2, wy); orc_filter(g, 3, wz); orc_filter(g, 0, wl);
    double* gc[3]; double* nt[3]; double* st[3];
    for (int d = 0; d < 3; ++d) { gc[d] = (double*)malloc(n * sizeof(double)); nt[d] = (double*)malloc(n * sizeof(double)); st[d] = (double*)malloc(n * sizeof(double)); }
    double* kap = (double*)malloc(n * sizeof(double));
    double* t = (double*)malloc(n * sizeof(double));
    const double* flt[3] = {wx, wy, wz};
    const double eps_t = 1e-7 / g->hx;
    for (int d = 0; d < 3; ++d) orc_apply_filter(g, BC_COPY, flt[d], C, gc[d]);
    for (size_t c = 0; c < n; ++c) {
        const double l = sqrt(gc[0][c] * gc[0][c] + gc[1][c] * gc[1][c] + gc[2][c] * gc[2][c]);
        for (int d = 0; d < 3; ++d) nt[d][c] = gc[d][c] / (eps_t + l);
        kap[c] = 0.0;
    }
    for (int d = 0; d < 3; ++d) {
        orc_apply_filter(g, BC_COPY, flt[d], nt[d], t);
        for (size_t c = 0; c < n; ++c) kap[c] -= t[c];
    }
    for (size_t c = 0; c < n; ++c)
        for (int d = 0; d < 3; ++d) st[d][c] = sigma_t * kap[c] * gc[d][c];
    /* b = f(g rho; w_z) - div(s_t)   (Eq. 43) */
    for (size_t c = 0; c < n; ++c) nt[0][c] = grav * mix01(rho_l, rho_g, C[c]);      /* reuse: g rho */
    orc_apply_filter(g, BC_COPY, wz, nt[0], b);
    for (int d = 0; d < 3; ++d) {
        orc_apply_filter(g, BC_COPY, flt[d], st[d], t);
        for (size_t c = 0; c < n; ++c) b[c] -= t[c];
    }
    /* bottom boundary: ghost = mirror + hz g rho(mirror) */
    for (int j = 0; j < g->ny; ++j)
        for (int i = 0; i < g->nx; ++i) {
            double add = 0.0;
            for (int jj = -1; jj <= 1; ++jj)
                for (int ii = -1; ii <= 1; ++ii)
                    add += -wl[(ii + 1) + 3 * (jj + 1)] * g->hz * ghost(nt[0], g, BC_COPY, i + ii, j + jj, 0);   /* kk = -1 slice */
            b[IDX(g, i, j, 0)] += add;
        }
    if (kappa_out) memcpy(kappa_out, kap, n * sizeof(double));
    for (int d = 0; d < 3; ++d) {
        if (st_out && st_out[d]) memcpy(st_out[d], st[d], n * sizeof(double));
        free(gc[d]); free(nt[d]); free(st[d]);
    }
    free(kap); free(t);
}

/* ------------------------------------------------------------------------------------
 * Stage 2, the forcing terms of Eq. 18 that the advection-diffusion residual above leaves out (
 * SURVEY 8(f) next 3):   + f(p_hs + p~_nh; w_x|y|z)  - f(s_c + s_tc; w_m),   nodal.
 * Eq. 45 is linear in s~, so they are applied to the predicted velocity afterwards:
 *   q~_c  <-  q~_c - (dt / rho) ( d_c p_hs + d_c p~_nh - M (s_c + s_tc) ),   M = consistent mass filter / m_l,
 * with s_u = s_v = 0, s_w = -g rho (Eq. 20) and s_t from orc_hydrostatic_rhs (Eq. 21).
 * Halos: p_hs -- zero derivative on the sides, zero value on the top face (ghost = -mirror), and at the bottom the
 * extrapolation ghost = mirror + hz g rho(nearest node) that enforces dp_hs/dz = -rho g (the same ghost
 * orc_hydrostatic_rhs folds into b_hs);  p~_nh -- the factors pbc of its solver;  sources -- copies (reading C9-iv).
 * p_hs, p_nh, st may be NULL (term absent). */
static double ghost_phs(const double* p, const double* rho, const orc_grid* g, double grav, int i, int j, int k) {
    if (i < 0) i = -1 - i; else if (i >= g->nx) i = 2 * g->nx - 1 - i;
    if (j < 0) j = -1 - j; else if (j >= g->ny) j = 2 * g->ny - 1 - j;
    if (k < 0) return p[IDX(g, i, j, -1 - k)] + g->hz * grav * rho[IDX(g, i, j, -1 - k)];
    if (k >= g->nz) return -p[IDX(g, i, j, 2 * g->nz - 1 - k)];
    return p[IDX(g, i, j, k)];
}
void orc_mom_forcing(const orc_grid* g, const double* C, const double* p_hs, const double* p_nh, const int* pbc,
                     double grav, const double* const* st, double rho_l, double rho_g, double dt, double* const* qt) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wd[27], wm[27];
    orc_filter(g, 7, wm);
    double* rho = (double*)malloc(n * sizeof(double));
    double* src = (double*)malloc(n * sizeof(double));
    double* t = (double*)malloc(n * sizeof(double));
    for (size_t c = 0; c < n; ++c) rho[c] = mix01(rho_l, rho_g, C[c]);
    for (int d = 0; d < 3; ++d) {
        orc_filter(g, 1 + d, wd);
        for (size_t c = 0; c < n; ++c) src[c] = (st && st[d] ? st[d][c] : 0.0) + (d == 2 ? -grav * rho[c] : 0.0);
        orc_apply_filter(g, BC_COPY, wm, src, t);                                   /* f(s_c + s_tc; w_m) */
        for (size_t c = 0; c < n; ++c) qt[d][c] += dt * t[c] / rho[c];
        if (p_nh) {
            orc_apply_filter(g, pbc, wd, p_nh, t);                                  /* f(p~_nh; w_d) */
            for (size_t c = 0; c < n; ++c) qt[d][c] -= dt * t[c] / rho[c];
        }
        if (p_hs)
            for (int k = 0; k < g->nz; ++k)
                for (int j = 0; j < g->ny; ++j)
                    for (int i = 0; i < g->nx; ++i) {
                        double a = 0.0;                                             /* f(p_hs; w_d) */
                        for (int kk = -1; kk <= 1; ++kk)
                            for (int jj = -1; jj <= 1; ++jj)
                                for (int ii = -1; ii <= 1; ++ii)
                                    a += wd[(ii + 1) + 3 * (jj + 1) + 9 * (kk + 1)] * ghost_phs(p_hs, rho, g, grav, i + ii, j + jj, k + kk);
                        qt[d][IDX(g, i, j, k)] -= dt * a / rho[IDX(g, i, j, k)];
                    }
    }
    free(rho); free(src); free(t);
}

/* Velocity projection, Eq. 54 with Eq. 48: q = q~ - dt k . f(p; w_x|y|z),
 * k = 1/rho; halo of p by the solver's BC factors.  In place on u, v, w. */
void orc_project_velocity(const orc_grid* g, const int* bc, const double* p, const double* kcoef, double dt,
                          double* u, double* v, double* w) {
    const size_t n = (size_t)g->nx * g->ny * g->nz;
    double wf[27];
    double* t = (double*)malloc(n * sizeof(double));
    double* q[3] = {u, v, w};
    for (int d = 0; d < 3; ++d) {
        orc_filter(g, 1 + d, wf);
        orc_apply_filter(g, bc, wf, p, t);
        for (size_t c = 0; c < n; ++c) q[d][c] -= dt * kcoef[c] * t[c];
    }
    free(t);
}
