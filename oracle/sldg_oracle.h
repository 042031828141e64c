/*
 * sldg_oracle.h -- plain CPU oracle for the SLDG translation sweep and the
 * Vlasov-Poisson Strang step of arXiv:1907.08316.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, the smoke check
 * in __graft_entry__.py and the cpu_baseline / --impl reference legs of
 * bench.py may build, load or call it.  It shares no code, header, table or
 * constant generator with the CUDA library under paper_1907_08316_b200/csrc/.
 *
 * Citations: "P:n" = line n of PAPER.md, "S:§8(c) Ox/Rx" = the oracle
 * definition / reading in SURVEY.md section 8(c) (restated in DESIGN.md).
 *
 * Conventions (S:§8 "Notation"): dimensions are ordered x_1..x_dx, v_1..v_dv;
 * dimension d has n_d cells, N_d = n_d*o nodes, node index p = i*o + j (cell i,
 * local Gauss-Legendre node j); f is a dense array with linear index
 * sum_d p_d * prod_{e<d} N_e (x_1 fastest).  All directions are periodic (R5).
 * Everything is fp64 except f itself and the rounded A,B in the *_f32 variants
 * (R9); the Gauss-Legendre rule and the A,B quadrature are carried out in long double
 * internally and rounded ONCE to double (O7: 'rounded once' taken literally).  Every function returns 0 on success, nonzero on a bad argument.
 *
 * Pins: P1..P13 of S:§8(c) in tests/test_oracle_pins.py, test_oracle_sweep_pins.py,
 * test_oracle_physics_pins.py, test_oracle_moment_pins.py; the three-dimensional branches
 * (Poisson mode decode, d_v = 3 weights, 3+3 D step), the 2+2 D Landau rate and the global sums
 * against exact summation in tests/test_oracle_3d_pins.py; A,B against exact values (<= 1/2 ulp +
 * 1e-18) in tests/test_oracle_ab_exact.py; ASan/UBSan in tests/test_oracle_sanitizers.py.
 * Config-2 two-stream growth is "parity unpinned" by the paper (its eq. (2) is a different state).
 */
#ifndef SLDG_ORACLE_H
#define SLDG_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

#define ORACLE_MAX_ORDER 8
#define ORACLE_MAX_DIM 6

/* O1: o-point Gauss-Legendre rule mapped to [0,1]; xi ascending, sum w = 1. */
int oracle_gauss_legendre(int o, double *xi, double *w);

/* Lagrange basis l_j on the nodes xi[0..o-1], evaluated at x (O1). */
double oracle_lagrange(int o, const double *xi, int j, double x);

/* R3: delta = -sigma, m = floor(delta), theta = delta - m in [0,1). */
void oracle_shift_split(double sigma, long *m, double *theta);

/* O2 ("L2 projection"): A,B in R^{o x o}, row-major [j][l],
 *   A_jl = 1/w_j int_0^{1-theta} l_j(x) l_l(x+theta)   dx
 *   B_jl = 1/w_j int_{1-theta}^1 l_j(x) l_l(x+theta-1) dx
 * each integral by the o-point rule mapped to its interval (exact: degree 2o-2). */
int oracle_assemble_AB(int o, double theta, double *A, double *B);

/* node coordinates c_d(p) = lo + (i + xi_j) h, p = i*o+j (S:§8 Notation) */
int oracle_node_coords(int n_cells, int o, double lo, double hi, double *c);

/* O2/O7: one periodic line of n cells, contiguous.  A,B already rounded to T.
 *   u_new[i][j] = chain( A[j][.] u_old[i*][.] , B[j][.] u_old[i*+1][.] ),  i* = (i+m) mod n */
int oracle_translate_line_f64(int o, long n, const double *A, const double *B, long m,
                              const double *u_old, double *u_new);
int oracle_translate_line_f32(int o, long n, const float *A, const float *B, long m,
                              const float *u_old, float *u_new);

/* O3 ("for each slice"): sweep along dimension k (0-based) of a D-dimensional
 * array with N[d] nodes per dimension, in place.  The shift of a line (in cell
 * widths) is sigma[q], q = canonical linear index over the dimensions listed in
 * dep[0..ndep-1] (ascending), none of which may be k. */
int oracle_translate_f64(double *f, int D, const long *N, int o, int k,
                         const double *sigma, int ndep, const int *dep);
int oracle_translate_f32(float *f, int D, const long *N, int o, int k,
                         const double *sigma, int ndep, const int *dep);

/* O3/R4/R8: physics sweep.  dim < dx: sigma = c_{v_a}(p) tau / h_{x_a} (a = dim);
 * dim >= dx: sigma = -E_a(x) tau / h_{v_a} (a = dim-dx), E = [dx][X] fp64. */
int oracle_advect_f64(double *f, int dx, int dv, const int *cells, int o,
                      const double *lo, const double *hi, int dim, double tau, const double *E);
int oracle_advect_f32(float *f, int dx, int dv, const int *cells, int o,
                      const double *lo, const double *hi, int dim, double tau, const double *E);

/* O4: rho[x] = - sum_v W_v f[v][x]: the sum over all velocity nodes in canonical order,
 * accumulated in long double and rounded to double once (no grouping, D:O4). */
int oracle_rho_f64(const double *f, int dx, int dv, const int *cells, int o,
                   const double *lo, const double *hi, double *rho);
int oracle_rho_f32(const float *f, int dx, int dv, const int *cells, int o,
                   const double *lo, const double *hi, double *rho);

/* O5/R6/R13: -Lap phi = rho + 1 periodic, E = -grad phi at the x-nodes; direct
 * DFT sums over the modes |m_a| <= floor((n_a-1)/2); E is [dx][X]. */
int oracle_poisson_E(const double *rho, int dx, const int *cells, int o,
                     const double *lo, const double *hi, double *E);

/* O6 row a-5: Strang step.  rho_out/E_out ([X], [dx][X]) may be NULL. */
int oracle_step_f64(double *f, int dx, int dv, const int *cells, int o,
                    const double *lo, const double *hi, double dt);
int oracle_step_f32(float *f, int dx, int dv, const int *cells, int o,
                    const double *lo, const double *hi, double dt);

/* O6 row a-6 / R12: mass = sum W f, l2 = sqrt(sum W f^2) as single running sums over all N nodes in
 * canonical order, long double accumulator rounded once; ee = 1/2 sum_x W_x |E|^2. */
int oracle_diagnostics_f64(const double *f, int dx, int dv, const int *cells, int o,
                           const double *lo, const double *hi,
                           double *mass, double *l2, double *ee);
int oracle_diagnostics_f32(const float *f, int dx, int dv, const int *cells, int o,
                           const double *lo, const double *hi,
                           double *mass, double *l2, double *ee);

/* S:8(f) NEXT-4 (Fig. 15): momentum[a] = int int v_a f (a < dv) and
 * kinetic = 1/2 int int |v|^2 f by Gauss quadrature on the nodes: single running sums in long double (R12). */
int oracle_moments_f64(const double *f, int dx, int dv, const int *cells, int o,
                       const double *lo, const double *hi, double *momentum, double *kinetic);
int oracle_moments_f32(const float *f, int dx, int dv, const int *cells, int o,
                       const double *lo, const double *hi, double *momentum, double *kinetic);

/* threads the sweeps/reductions will use (OpenMP over lines), for the bench report */
int oracle_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
