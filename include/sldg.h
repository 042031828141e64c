/*
 * sldg.h -- C-ABI boundary of the B200-native SLDG Vlasov-Poisson hot path
 * (arXiv:1907.08316, "Semi-Lagrangian Vlasov simulation on GPUs").
 *
 * Citations: "P:n" = line n of the paper text; "D:Rx / D:Ox" = the
 * readings and definitions listed in DESIGN.md (taken from SURVEY.md section 8(c)).
 *
 * What the library computes (section 1, section 2, section 3):
 *   - the semi-Lagrangian discontinuous-Galerkin translation of f along one
 *     phase-space direction: in every cell the o Gauss-Legendre nodal values become
 *         u_new[i][j] = sum_l A_jl u_old[i*][l] + sum_l B_jl u_old[i*+1][l]
 *     with A(theta), B(theta) in R^{o x o} the L2 projection of the exactly shifted
 *     piecewise polynomial, applied "for each slice of the high-dimensional
 *     problem";
 *   - rho(x) = -int f dv, the periodic Poisson problem -Lap phi = rho + 1,
 *     E = -grad phi, the Strang step and the invariants mass, L2 norm and
 *     electric energy.
 *
 * Layout of f at this boundary ("canonical"): dense array of N = prod_d N_d values,
 * N_d = cells[d]*order, dimensions ordered x_1..x_dx, v_1..v_dv, linear index
 * sum_d p_d * prod_{e<d} N_e (x_1 fastest), node index p_d = i_d*order + j_d (cell i_d,
 * local Gauss-Legendre node j_d, nodes ascending).  All directions are periodic (D:R5).
 *
 * Memory: the two f buffers are CALLER-owned DEVICE memory (N*sizeof(T) bytes each,
 * 16-byte aligned); the library ping-pongs between them and allocates only small
 * tables (A/B, rho, E, partial sums, DFT matrices) of size O(X + sum N_d + splits*X).
 * Streams: every call enqueues on the stream given to sldg_create and returns without
 * synchronising, except where stated.
 *
 * Errors: every int-returning call returns SLDG_OK (0) or a negative sldg_status; the
 * library never throws, exits or falls back to a CPU path.  sldg_last_error() gives a
 * human-readable message for the last failure on that context (or the last failed
 * sldg_create when ctx == NULL).
 */
#ifndef SLDG_H
#define SLDG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sldg_ctx sldg_ctx;            /* opaque; owned by the library            */

typedef enum { SLDG_F64 = 0, SLDG_F32 = 1 } sldg_dtype;   /* storage/arithmetic type T of f */

typedef enum {
    SLDG_OK = 0,
    SLDG_ERR_ARG = -1,          /* null pointer, dimension/order/count out of range      */
    SLDG_ERR_UNSUPPORTED = -2,  /* (order, dtype, dims) combination not instantiated     */
    SLDG_ERR_CUDA = -3,         /* a CUDA runtime call or kernel launch failed           */
    SLDG_ERR_STATE = -4         /* call needs something not yet computed (E, rho, f)     */
} sldg_status;

#define SLDG_MAX_DIM 6
#define SLDG_MAX_ORDER 6

/* Create a solver context (template parameters (d_x, d_v, o) become run-time here).
 *   dx, dv      1..3 each, dv >= dx (E has dx components and accelerates v_1..v_dx)
 *   cells       [dx+dv] host ints, n_d >= 1
 *   order       o in 1..SLDG_MAX_ORDER (number of Gauss-Legendre nodes per cell per dim)
 *   lo, hi      [dx+dv] host doubles, hi > lo
 *   f_buf0/1    device pointers, N*sizeof(T) bytes each, distinct, not freed by the library
 *   cuda_stream a cudaStream_t (0 = legacy default stream)
 * The current buffer is f_buf0 until a sweep flips it. */
int sldg_create(sldg_ctx **out, int dx, int dv, const int *cells, int order,
                const double *lo, const double *hi, sldg_dtype dtype,
                void *f_buf0, void *f_buf1, void *cuda_stream);

/* Synchronises the stream, frees the library's tables.  The f buffers stay the caller's. */
int sldg_destroy(sldg_ctx *ctx);

const char *sldg_last_error(const sldg_ctx *ctx);

size_t sldg_num_dofs(const sldg_ctx *ctx);          /* N                                   */
size_t sldg_num_x(const sldg_ctx *ctx);             /* X = prod_{d<dx} N_d                 */

/* Node coordinates c_d(p) = lo_d + (i + xi_j) h_d, p = i*o + j, host_out[N_dim].   */
int sldg_node_coords(const sldg_ctx *ctx, int dim, double *host_out);

/* Copy N values of type T into / out of the current buffer.  Host copies use
 * cudaMemcpyAsync on the stream followed by a stream synchronise. */
int sldg_set_initial(sldg_ctx *ctx, const void *f_src, int is_device);
int sldg_get_f(sldg_ctx *ctx, void *dst, int is_device);
/* Device pointer holding f now.  The pointer is writable: the library assumes the caller may edit f through
 * it and forgets the invariants it remembered for the current f (see sldg_invariants).  rho and E held in the
 * context are NOT dropped; after editing f in place call sldg_compute_rho / sldg_poisson_E (or sldg_diagnostics,
 * which does both) before a v-sweep that should see the new field. */
void *sldg_current(sldg_ctx *ctx);

/* Fill the current buffer with f[g] = U(seed, tag, g) in [0,1) rounded to T, g = canonical
 * linear index: the counter-based generator of the config-4 microbenchmark (DESIGN.md
 * "Input recipe"; splitmix64 finaliser, top 53 bits * 2^-53). */
int sldg_fill_uniform(sldg_ctx *ctx, unsigned long long seed, unsigned tag);

/* Row a-1 + a-2: raw translation sweep along dimension `dim` (0-based), the
 * shift sigma_q of every line given in CELL WIDTHS (new(x) = old(x - sigma h), D:R3):
 *   dim <  dx (x_a):  count = N_{v_a},  q = node index of v_a
 *   dim >= dx (v_a):  count = X,        q = x-node index (x_1 fastest)
 * shift_cells is a HOST array read before the call returns.  Flips the current buffer. */
int sldg_translate(sldg_ctx *ctx, int dim, const double *shift_cells_host, size_t count);

/* As sldg_translate but the shift table is already in DEVICE memory (fp64) and is read
 * on the stream; nothing is copied from the host.  This is what the microbenchmark times. */
int sldg_translate_dev(sldg_ctx *ctx, int dim, const double *shift_cells_device, size_t count);

/* Physics sweep (D:O3, D:R4): dim < dx: sigma = c_{v_a}(q) dt / h_{x_a};
 * dim >= dx: sigma = -E_a(x_q) dt / h_{v_a} with the stored E (SLDG_ERR_STATE if none). */
int sldg_advect(sldg_ctx *ctx, int dim, double dt);

/* Two consecutive sweeps in ONE pass over f: the result is identical, bit for
 * bit, to sldg_advect(dim1, dt) followed by sldg_advect(dim2, dt) (resp. two sldg_translate_dev
 * calls), but f is read and written once instead of twice.  dim1 < dim2, both x-dimensions or both
 * v-dimensions (their shifts do not depend on each other's coordinate, D:R8).  sldg_step uses this
 * for (x_1,x_2) and (v_1,v_2) unless SLDG_NO_FUSE=1 is set in the environment at sldg_create.
 * The fused v-kernels are built for the physical regime |shift| < 1 cell; a block that meets a line shifted by
 * a cell or more falls back to reading its neighbours from global memory -- same bits, about 2.5x the time of
 * the two single sweeps when most lines are that wide.  All four calls are asynchronous like the rest of the
 * library and none checks the width: a field with |E| dt >= h_v is outside the regime the splitting is accurate
 * in and costs bandwidth there, never correctness.  A caller that feeds sldg_translate_pair_dev / _triple_dev
 * wide v-shifts on purpose can set SLDG_ROUTE_WIDE=1 in the environment at sldg_create: those two calls then
 * assemble the tables first, read back (STREAM SYNCHRONISATION, so not inside a stream capture) whether any
 * line is a cell or more wide, and run such a call as single sweeps. */
int sldg_advect_pair(sldg_ctx *ctx, int dim1, int dim2, double dt);
int sldg_translate_pair_dev(sldg_ctx *ctx, int dim1, const double *shift1_device, size_t count1,
                            int dim2, const double *shift2_device, size_t count2);

/* Did a fused v-sweep run outside its regime?  *seen = 1 when, since sldg_create (or the last call with
 * reset != 0), a fused pair / triple along v-dimensions -- sldg_advect_pair / _triple, the v-group of sldg_step /
 * sldg_step_n, the raw fused calls -- was launched on shift tables with at least one line shifted by a cell or more
 * (|E| dt >= h_v), i.e. some of its blocks took the slow global-read fallback (about 2.5x the time of the single
 * sweeps where most lines are that wide; results unaffected).  A caller who sees 1 should shorten dt or issue
 * single sweeps.  The mark is left by the table assembly on the device; this call synchronises the stream. */
int sldg_wide_shift_seen(sldg_ctx *ctx, int *seen, int reset);

/* Three consecutive sweeps (dim1 < dim2 < dim3, all x- or all v-dimensions: the 3+3 D step) in one
 * pass over f; identical, bit for bit, to the three single sweeps.  The fused kernel exists for
 * order <= 2; above that the call runs a fused pair followed by a single sweep (same result). */
int sldg_advect_triple(sldg_ctx *ctx, int dim1, int dim2, int dim3, double dt);
int sldg_translate_triple_dev(sldg_ctx *ctx, int dim1, const double *shift1_device, size_t count1,
                              int dim2, const double *shift2_device, size_t count2,
                              int dim3, const double *shift3_device, size_t count3);

/* rho[X] = -sum_v W_v f[v][x] (fp64 accumulation for both dtypes) into the
 * context and, if rho_device_or_null != NULL, also to that device array. */
int sldg_compute_rho(sldg_ctx *ctx, double *rho_device_or_null);

/* E[dx][X] from the stored rho: -Lap phi = rho + 1 periodic, E = -grad phi at the x-nodes,
 * spectral with the modes |m_a| <= floor((n_a - 1)/2) and the mean mode dropped (D:R6, D:R13). */
int sldg_poisson_E(sldg_ctx *ctx, double *E_device_or_null);

/* Overwrite the stored E ([dx][X] fp64, host or device): lets a caller drive sldg_advect in v.  The next
 * sldg_diagnostics / sldg_invariants re-reads f and replaces this E by the one that belongs to the current f. */
int sldg_set_E(sldg_ctx *ctx, const double *E, int is_device);

/* S:8(f) NEXT-1: the x half-step and the density that follows it ("advection x", "compute rho") as ONE
 * pass over f: sweeps x_1..x_dx with increment tau exactly as sldg_advect / _pair / _triple would (f is
 * bit-identical), and leaves rho of the result in the context (and in rho_device_or_null, X doubles on the
 * device, if not NULL).  When d_x = 2 or 3 and the fused sweep kernels apply, rho is accumulated while the
 * last sweep writes f (no separate read of f); otherwise it is the sweeps followed by sldg_compute_rho.
 * sldg_step uses this call for its first x half-step.
 * Reproducibility: every sum in the library has a fixed order, so a run repeats bit for bit on the same GPU
 * model and library build.  The NUMBER of partial rows of the rho accumulated here is sized to one wave of
 * blocks (SM count x resident blocks), and the stand-alone pass sizes its v-splits from the SM count too, so rho
 * -- and through E every later f -- may differ at rounding level (1e-16 relative per step) between GPU models
 * or toolkit versions.  f from the sweeps alone (sldg_translate*, sldg_advect* with a given E) has no such
 * dependence. */
int sldg_advect_x_rho(sldg_ctx *ctx, double tau, double *rho_device_or_null);

/* Strang step (D:O6 row a-5): x_1..x_dx with dt/2, rho, Poisson, v_1..v_dx with dt,
 * x_1..x_dx with dt/2. */
int sldg_step(sldg_ctx *ctx, double dt);

/* nsteps Strang steps: the result of nsteps calls of sldg_step -- bit for bit when rho is a pass of its own in
 * both (SLDG_NO_FUSE_RHO=1), else up to the rounding-level difference between rho accumulated inside a sweep
 * (sldg_step, see sldg_advect_x_rho) and rho from its own pass (this call) -- with the x
 * half-steps that end one step and begin the next -- nothing happens between them when no invariant is written
 * -- done as ONE pass over f: x(dt/2) applied twice inside the kernel (sldg_advect_x_twice), not x(dt).
 * Per step: v-group (1R+1W), x-group twice (1R+1W), rho (1R) instead of the 7 N s of sldg_step in d_x >= 2.
 * Where no kernel applies the whole x-group twice in one pass (d_x = 2 with order >= 4, d_x = 3: there two passes of
 * the x-triple are faster than its twice-applied variant) the call is nsteps calls of sldg_step.
 * f(t_n) is materialised only at the end; call sldg_diagnostics etc. between calls of sldg_step_n. */
int sldg_step_n(sldg_ctx *ctx, double dt, int nsteps);

/* The x-group x_1..x_dx with increment tau applied twice; bit-identical to issuing the group twice.  One pass
 * over f when one kernel performs the whole group (d_x = 1; d_x = 2 with order <= 3; d_x = 3 with order <= 2
 * and a small x-grid), else two. */
int sldg_advect_x_twice(sldg_ctx *ctx, double tau);

/* mass = sum W f, l2 = sqrt(sum W f^2), electric_energy = 1/2 sum_x W_x |E|^2 from the
 * current f (D:R12); recomputes rho and E (they describe the current f afterwards); synchronises the
 * stream.  Any of the three output pointers (host) may be NULL. */
int sldg_diagnostics(sldg_ctx *ctx, double *mass, double *l2, double *electric_energy);

/* S:8(f) NEXT-4 ("physical invariants", P:224 momentum conservation, Fig. 15 kinetic / total
 * energy): momentum[a] = int int v_a f dx dv for a < dv (host array of dv doubles) and
 * kinetic_energy = 1/2 int int |v|^2 f dx dv from the current f; one read of f; synchronises the
 * stream.  Either pointer may be NULL.  Total energy = kinetic_energy + electric_energy. */
int sldg_moments(sldg_ctx *ctx, double *momentum, double *kinetic_energy);

/* All invariants the paper writes once per time step ("once at the beginning of the time step
 * to write the electric energy and other invariant") in ONE read of the current f: the pass that forms
 * rho also forms sum W f^2, sum v_a W f and sum |v|^2 W f (S:8(f) NEXT-4 "fused into the rho pass").
 * Outputs as in sldg_diagnostics / sldg_moments (host pointers, any may be NULL; momentum has dv entries);
 * synchronises the stream once.  The library remembers the result until f changes: sldg_diagnostics,
 * sldg_moments and sldg_invariants called in any order on the same f read it from HBM once.  "Changes" means:
 * through a library call (a sweep, a step, sldg_set_initial, sldg_fill_uniform), or possibly through the caller's
 * own hands -- sldg_current() hands out a writable pointer and therefore forgets the remembered result, and so
 * does sldg_set_E (the remembered electric energy belonged to the old E).  A caller that keeps a pointer from an
 * earlier sldg_current() and edits f later must call sldg_current() again before asking for invariants. */
int sldg_invariants(sldg_ctx *ctx, double *mass, double *l2, double *electric_energy, double *momentum,
                    double *kinetic_energy);

/* Number of kernels this context has launched since sldg_create (bench "gpu_launches"). */
unsigned long long sldg_launch_count(const sldg_ctx *ctx);

/* The rho pass (as sldg_compute_rho) for callers that are not allowed to allocate device memory.
 *
 * Every context-based call needs sldg_create, and sldg_create calls cudaMalloc for its tables.  Some users
 * cannot have that: a host code that gave the whole device heap to its own pool at start-up, a plug-in or
 * callback inside another program's time loop (an allocation may synchronise the whole device and stall that
 * program's other streams), a job with a memory budget fixed and audited before it starts.  This one call needs
 * no context and calls no cudaMalloc, cudaFree or any library routine that allocates:
 *
 *     rho[x] = - sum_{v < V} Wv[v] * f[v*X + x],   x < X        (fp64 products and sums for both dtypes)
 *
 *   f_device    X*V values of type T = dtype in the canonical layout (x fastest); device memory; read only
 *   Wv_device   V doubles, the quadrature weight of every v-node (prod_a h_a w_j on [0,1]); device; read only
 *   rho_device  X doubles; device; written
 *   cuda_stream a cudaStream_t of the CURRENT device (0 = legacy default); the kernels are enqueued on it and
 *               the call returns without synchronising
 *   err/err_len optional caller-owned buffer for a message when the call fails (may be NULL / 0)
 * All three arrays must live on the device that is current in the calling thread.
 *
 * The partial sums between its two kernels live in a fixed device array that is part of the library image:
 * SLDG_RHO_NOALLOC_SCRATCH_BYTES (4 MiB) on every GPU that loads the library, held until the process exits.
 * Hence the limit: X <= SLDG_RHO_NOALLOC_MAX_X x-nodes (any V); a larger X returns SLDG_ERR_ARG with the
 * reason in err and launches nothing.  (Config 4 has X = 147 456, config 5 X = 32 768.)
 *
 * The FIRST call on each device looks up the array's device address (cudaGetSymbolAddress) and the SM count
 * before it launches; make that first call outside any stream capture.
 * All calls on a device share the one array.  Nothing in it has to start at zero -- each call's first kernel
 * writes every partial sum its second kernel reads, so what an earlier call left behind is never read -- but two
 * calls whose kernels can overlap on the GPU (different streams, no dependency between them) race on it: keep
 * calls on one device on one stream, or order them with events.
 * The result agrees with sldg_compute_rho to rounding (the number of partial sums differs), not bit for bit. */
#define SLDG_RHO_NOALLOC_SCRATCH_BYTES 4194304
#define SLDG_RHO_NOALLOC_MAX_X 524288
int sldg_rho_noalloc(const void *f_device, sldg_dtype dtype, size_t X, size_t V, const double *Wv_device,
                     double *rho_device, void *cuda_stream, char *err, size_t err_len);

#ifdef __cplusplus
}
#endif
#endif /* SLDG_H */
