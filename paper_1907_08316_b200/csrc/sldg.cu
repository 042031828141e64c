// sldg.cu -- implementation of include/sldg.h: context, dispatch and the Strang step.
// Every step of the path runs in the kernels of sweep.cuh / reduce.cuh / poisson.cuh; there is
// no CPU fallback (a missing device or an uninstantiated (order, dtype) is an error).
#include "../../include/sldg.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <map>
#include <mutex>
#include <utility>
#include <vector>

#include "fill.cuh"
#include "poisson.cuh"
#include "reduce.cuh"
#include "sweep.cuh"
#include "sweep_tma.cuh"
#include "sweep_fused.cuh"
#include "tables.hpp"

using namespace sldg;

namespace {
char g_create_error[512] = "";
}

struct sldg_ctx {
    int dx = 0, dv = 0, D = 0, o = 0;
    sldg_dtype dtype = SLDG_F64;
    size_t esize = 8;
    int cells[SLDG_MAX_DIM] = {0};
    long N[SLDG_MAX_DIM] = {0};
    double lo[SLDG_MAX_DIM] = {0}, hi[SLDG_MAX_DIM] = {0}, h[SLDG_MAX_DIM] = {0};
    long X = 1, V = 1, ndof = 1;
    double xi[SLDG_MAX_ORDER] = {0}, w[SLDG_MAX_ORDER] = {0};
    void *buf[2] = {nullptr, nullptr};
    int cur = 0;
    cudaStream_t stream = nullptr;
    int device = 0;                    // the device the context was created on; every entry point runs there
    int sm_count = 148;
    // tuning switches, read from the environment ONCE in sldg_create
    struct Tune {
        int tile_w = 0;                // SLDG_TILE_W: columns per TMA tile of the v-sweeps (0 = default)
        bool plane_pair = true;        // SLDG_NO_PLANE_PAIR=1 -> false
        bool plane_single = true;      // SLDG_NO_PLANE_SINGLE=1 -> false: register-window kernel for the single x_2 sweep
        int tile_pair = -1;            // SLDG_TILE_PAIR: -1 default (o >= 3), 0 never, 1 always
        bool tile_triple = true;       // SLDG_NO_TILE_TRIPLE=1 -> false
        int vt_variant = -1;           // SLDG_VTRIPLE_VARIANT: staged v-triple variant (-1 = default)
        int xt_parts = 0;              // SLDG_XTRIPLE_PARTS: x_2-ranges per velocity node in the x-triple (0 = default, 1 = whole plane)
        bool xt_two = true;            // SLDG_XTRIPLE_ONE=1 -> false: one x_2-cell per thread in the part-plane x-triple
        bool twice_triple = false;     // SLDG_TWICE_TRIPLE=1: sldg_step_n also merges the x half-steps in 3+3 D (slower, section 9)
        bool twice = true;             // SLDG_NO_TWICE=1 -> false: sldg_step_n never merges the x half-steps of two steps
        bool fuse_rho = true;          // SLDG_NO_FUSE_RHO=1 -> false: rho is a pass of its own after the x-group
        bool route_wide = false;       // SLDG_ROUTE_WIDE=1: raw fused v-calls read a flag back (stream sync) and run wide shifts as single sweeps
        bool rho_triple = false;       // SLDG_RHO_TRIPLE=1: also fuse rho into the x-triple (3+3 D: measured break-even, off)
        int x1_chunk_kb = 0, x1_block = 128;   // SLDG_X1_CHUNK_KB / SLDG_X1_BLOCK: bulk x_1 kernel geometry (0 = default)
        int rho_cells = 0;             // SLDG_RHO_CELLS: cells per block range in the fused x-group + rho kernels (0 = default)
    } tune;
    // TMA descriptors depend only on (buffer, view), both fixed for the life of the context: encoded once
    struct TmapSlot { CUtensorMap map; bool valid = false; int p0 = 0, p1 = 0; };
    TmapSlot tmap3[SLDG_MAX_DIM][2], tmap4[SLDG_MAX_DIM][2], tmap5[2];

    // device tables
    double *d_coef = nullptr;          // A/B polynomial coefficients [2][o][o][2o]
    double *d_coords[SLDG_MAX_DIM] = {nullptr};   // node coordinates per dimension
    long tab_cap = 0;                  // capacity (entries) of the general sweep tables
    // Sweep tables (a-1).  Storage: gen[0..1] (capacity tab_cap: v-sweeps, raw sldg_translate calls,
    // the two halves of a fused pair) and xt[a] (capacity N_{v_a}: the physics x_a sweep, whose
    // shifts c_v*tau/h never change, cached per tau so that sigma + assembly run once, not per step).
    struct Tab {
        double *sigma = nullptr;       // [cap] shift in cell widths
        int *m = nullptr;              // [cap] cell offset mod n
        void *ab = nullptr;            // [2 o^2][cap] of T
        double tau = 0.0;
        bool valid = false;            // m/ab hold the assembled table for `tau`
        double pending_tau = 0.0;      // sigma was filled for this tau; valid once the sweep that assembles succeeded
        bool pending = false;
    };
    Tab gen[3], xt[3];
    // the table set(s) the next sweep launch reads: aliases into gen[] / xt[]
    double *d_sigma = nullptr, *d_sigma2 = nullptr, *d_sigma3 = nullptr;
    int *d_m = nullptr, *d_m2 = nullptr, *d_m3 = nullptr;
    void *d_ab = nullptr, *d_ab2 = nullptr, *d_ab3 = nullptr;
    bool skip_asm1 = false, skip_asm2 = false, skip_asm3 = false;
    double *d_Wv = nullptr, *d_Wx = nullptr;      // quadrature weights over v-nodes / x-nodes
    double *d_va = nullptr, *d_v2 = nullptr;      // per v-node: coordinates v_a [dv][V] and |v|^2 [V]
    double *d_rho = nullptr, *d_s2 = nullptr, *d_E = nullptr;   // [X], [X], [dx][X]
    double *d_mom = nullptr;           // [dv + 1][X]: v_a f and |v|^2 f summed over v
    int max_splits = 1;
    double *d_part = nullptr;          // [3 + dv][max_splits][X]: rho, f^2, v_a f, |v|^2 f partials
    double *d_scal = nullptr;          // [8]: mass, l2^2, ee, momentum[dv], |v|^2 moment
    int *d_wide = nullptr;             // [1]: some line of a raw fused v-call is shifted by a cell or more
    int *d_wide_seen = nullptr;        // [1]: sticky -- a fused v-sweep was launched on tables with such a line (sldg_wide_shift_seen)
    // Poisson
    long K[3] = {1, 1, 1}, Mmax[3] = {0, 0, 0}, KK = 1;
    double2 *d_F[3] = {nullptr, nullptr, nullptr}, *d_G[3] = {nullptr, nullptr, nullptr};
    double *d_t[4] = {nullptr, nullptr, nullptr, nullptr};   // complex scratch (re, im) x 2
    double *d_gh[2] = {nullptr, nullptr};                    // g_hat (re, im) [KK]

    // CUDA graphs for launch-bound (small) problems: the kernels of one Strang step captured once per
    // (dt, buffer parity) on an internal stream and replayed on the caller's stream (SLDG_NO_GRAPH=1: off)
    struct StepGraph {
        cudaGraphExec_t exec = nullptr;
        double dt = 0.0;
        int cur_in = -1, cur_out = 0;
        unsigned long long launches = 0;
        unsigned long long xt_epoch = 0;   // the cached x-tables the captured kernels read
    };
    StepGraph graphs[2];
    unsigned long long xt_epoch = 0;       // bumped whenever a cached x-table is rewritten
    cudaStream_t capture_stream = nullptr;
    bool use_graph = true;
    double last_eager_dt[2] = {0.0, 0.0};   // dt of the last eager step that started from parity 0 / 1
    bool eager_seen[2] = {false, false};
    unsigned long long eager_epoch[2] = {0, 0};   // xt_epoch right after that eager step
    bool use_fuse = true;              // SLDG_NO_FUSE=1: sldg_step issues one sweep per pass
    bool use_tma = true;               // SLDG_NO_TMA=1 in the environment selects the plain kernels
    bool have_rho = false, have_E = false;
    bool twice_req = false;            // the next x-group kernel should apply the group twice in its one pass
    bool twice_done = false;           // ... and it did
    bool want_rho = false;             // the next fused x-group sweep should also leave the rho partials (NEXT-1)
    int rho_rows = 0;                  // > 0: that sweep left rho_rows partial rows [rho_rows][X] in d_part
    bool have_inv = false;             // d_part holds the one-read invariant partials of the CURRENT f
    unsigned long long launches = 0;
    char err[512] = "";
};

namespace {

int fail(sldg_ctx *c, int code, const char *fmt, ...) {
    char *dst = c ? c->err : g_create_error;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

#define CUDA_TRY(c, call)                                                                  \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess)                                                             \
            return fail((c), SLDG_ERR_CUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                               \
    } while (0)

#define LAUNCH_CHECK(c)                                                                     \
    do {                                                                                    \
        (c)->launches++;                                                                    \
        cudaError_t e_ = cudaGetLastError();                                                \
        if (e_ != cudaSuccess)                                                              \
            return fail((c), SLDG_ERR_CUDA, "kernel launch: %s (%s:%d)", cudaGetErrorString(e_), \
                        __FILE__, __LINE__);                                                \
    } while (0)

inline long cdiv(long a, long b) { return (a + b - 1) / b; }

// f was (or is about to be) rewritten: everything derived from the old f is stale
inline void f_changed(sldg_ctx *c) { c->have_rho = false; c->have_inv = false; }

// Runs the enclosing entry point on the context's device, whatever device is current in the calling
// thread, and restores the caller's device on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const sldg_ctx *c) {
        if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
            switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// Opt in to `bytes` of dynamic shared memory for `kernel` on this context's device.  The attribute
// (cudaFuncAttributeMaxDynamicSharedMemorySize) belongs to the (device, kernel) pair, not to a context, and
// cudaFuncSetAttribute stores exactly the value it is given -- so it is remembered process-wide under that key
// and only ever RAISED: a second context with a smaller grid must not lower what a live context's launches need.
std::mutex g_smem_mutex;
std::map<std::pair<int, const void *>, size_t> g_smem_attr;
template <typename K>
cudaError_t ensure_smem(sldg_ctx *c, K kernel, size_t bytes) {
    if (bytes <= 32 * 1024) return cudaSuccess;          // static + dynamic must stay under the 48 KB default
    std::lock_guard<std::mutex> lock(g_smem_mutex);
    size_t &have = g_smem_attr[std::make_pair(c->device, (const void *)kernel)];
    if (bytes <= have) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) have = bytes;
    return e;
}

int env_int(const char *name, int dflt, int lo, int hi) {
    const char *e = getenv(name);
    if (!e || !e[0]) return dflt;
    char *end = nullptr;
    long v = strtol(e, &end, 10);
    if (end == e || v < lo || v > hi) return dflt;       // out of range or not a number: ignored
    return (int)v;
}
bool env_flag(const char *name) {
    const char *e = getenv(name);
    return e && e[0] == '1';
}

template <typename P>
cudaError_t dalloc(P **p, size_t count) {
    return cudaMalloc((void **)p, (count ? count : 1) * sizeof(P));
}

void free_tables(sldg_ctx *c) {
    cudaFree(c->d_coef);
    for (int d = 0; d < SLDG_MAX_DIM; ++d) cudaFree(c->d_coords[d]);
    for (auto &t : c->gen) { cudaFree(t.sigma); cudaFree(t.m); cudaFree(t.ab); }
    for (auto &t : c->xt) { cudaFree(t.sigma); cudaFree(t.m); cudaFree(t.ab); }
    cudaFree(c->d_Wv); cudaFree(c->d_Wx); cudaFree(c->d_va); cudaFree(c->d_v2);
    cudaFree(c->d_rho); cudaFree(c->d_s2); cudaFree(c->d_E); cudaFree(c->d_mom);
    cudaFree(c->d_part); cudaFree(c->d_scal); cudaFree(c->d_wide); cudaFree(c->d_wide_seen);
    for (int a = 0; a < 3; ++a) { cudaFree(c->d_F[a]); cudaFree(c->d_G[a]); }
    for (int i = 0; i < 4; ++i) cudaFree(c->d_t[i]);
    cudaFree(c->d_gh[0]); cudaFree(c->d_gh[1]);
}

void host_node_coords(const sldg_ctx *c, int d, std::vector<double> &out) {
    out.resize(c->N[d]);
    for (int i = 0; i < c->cells[d]; ++i)
        for (int j = 0; j < c->o; ++j) out[(size_t)i * c->o + j] = c->lo[d] + ((double)i + c->xi[j]) * c->h[d];
}

}  // namespace

extern "C" const char *sldg_last_error(const sldg_ctx *ctx) { return ctx ? ctx->err : g_create_error; }
extern "C" size_t sldg_num_dofs(const sldg_ctx *ctx) { return ctx ? (size_t)ctx->ndof : 0; }
extern "C" size_t sldg_num_x(const sldg_ctx *ctx) { return ctx ? (size_t)ctx->X : 0; }
extern "C" unsigned long long sldg_launch_count(const sldg_ctx *ctx) { return ctx ? ctx->launches : 0; }
// The pointer is writable and the buffer is the caller's: whoever asks for it may edit f in place (a source or
// collision term, a rescale), so the remembered invariants of "the current f" are dropped here.
extern "C" void *sldg_current(sldg_ctx *ctx) {
    if (!ctx) return nullptr;
    ctx->have_inv = false;
    return ctx->buf[ctx->cur];
}

extern "C" int sldg_node_coords(const sldg_ctx *ctx, int dim, double *host_out) {
    if (!ctx || !host_out || dim < 0 || dim >= ctx->D) return SLDG_ERR_ARG;
    std::vector<double> c;
    host_node_coords(ctx, dim, c);
    memcpy(host_out, c.data(), c.size() * sizeof(double));
    return SLDG_OK;
}

// ------------------------------------------------------------------------------------------
// create / destroy
// ------------------------------------------------------------------------------------------
extern "C" int sldg_create(sldg_ctx **out, int dx, int dv, const int *cells, int order,
                           const double *lo, const double *hi, sldg_dtype dtype, void *f_buf0,
                           void *f_buf1, void *cuda_stream) {
    if (!out) return fail(nullptr, SLDG_ERR_ARG, "sldg_create: out is NULL");
    *out = nullptr;
    if (dx < 1 || dx > 3 || dv < 1 || dv > 3 || dv < dx)
        return fail(nullptr, SLDG_ERR_ARG, "sldg_create: need 1 <= dx <= dv <= 3 (got %d+%d)", dx, dv);
    if (!cells || !lo || !hi || !f_buf0 || !f_buf1 || f_buf0 == f_buf1)
        return fail(nullptr, SLDG_ERR_ARG, "sldg_create: null or aliased argument");
    if (order < 1 || order > SLDG_MAX_ORDER)
        return fail(nullptr, SLDG_ERR_UNSUPPORTED, "sldg_create: order %d not in 1..%d", order, SLDG_MAX_ORDER);
    if (dtype != SLDG_F64 && dtype != SLDG_F32)
        return fail(nullptr, SLDG_ERR_UNSUPPORTED, "sldg_create: unknown dtype %d", (int)dtype);
    if (((uintptr_t)f_buf0 | (uintptr_t)f_buf1) & 15)
        return fail(nullptr, SLDG_ERR_ARG, "sldg_create: f buffers must be 16-byte aligned");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1)
        return fail(nullptr, SLDG_ERR_CUDA, "sldg_create: no CUDA device (this library has no CPU path)");

    sldg_ctx *c = new sldg_ctx();
    c->dx = dx; c->dv = dv; c->D = dx + dv; c->o = order; c->dtype = dtype;
    c->esize = dtype == SLDG_F64 ? 8 : 4;
    c->stream = (cudaStream_t)cuda_stream;
    c->buf[0] = f_buf0; c->buf[1] = f_buf1;
    for (int d = 0; d < c->D; ++d) {
        if (cells[d] < 1 || !(hi[d] > lo[d])) {
            delete c;
            return fail(nullptr, SLDG_ERR_ARG, "sldg_create: bad cells/domain in dimension %d", d);
        }
        c->cells[d] = cells[d]; c->lo[d] = lo[d]; c->hi[d] = hi[d];
        c->h[d] = (hi[d] - lo[d]) / cells[d];
        c->N[d] = (long)cells[d] * order;
        c->ndof *= c->N[d];
        if (d < dx) c->X *= c->N[d]; else c->V *= c->N[d];
    }
    gauss_legendre_01(order, c->xi, c->w);
    {   // the environment is read here and nowhere else
        c->use_tma = !env_flag("SLDG_NO_TMA");
        c->use_fuse = !env_flag("SLDG_NO_FUSE");
        c->use_graph = !env_flag("SLDG_NO_GRAPH") && c->ndof <= (1L << 24);
        c->tune.plane_pair = !env_flag("SLDG_NO_PLANE_PAIR");
        c->tune.plane_single = !env_flag("SLDG_NO_PLANE_SINGLE");
        c->tune.tile_triple = !env_flag("SLDG_NO_TILE_TRIPLE");
        c->tune.tile_pair = env_int("SLDG_TILE_PAIR", -1, 0, 1);
        c->tune.vt_variant = env_int("SLDG_VTRIPLE_VARIANT", -1, 0, 15);
        c->tune.fuse_rho = !env_flag("SLDG_NO_FUSE_RHO");
        c->tune.twice = !env_flag("SLDG_NO_TWICE");
        c->tune.xt_two = !env_flag("SLDG_XTRIPLE_ONE");
        c->tune.twice_triple = env_flag("SLDG_TWICE_TRIPLE");
        c->tune.xt_parts = env_int("SLDG_XTRIPLE_PARTS", 0, 1, 8);
        c->tune.rho_triple = env_flag("SLDG_RHO_TRIPLE");
        c->tune.route_wide = env_flag("SLDG_ROUTE_WIDE");
        c->tune.rho_cells = env_int("SLDG_RHO_CELLS", 0, 1, 8);
        c->tune.x1_chunk_kb = env_int("SLDG_X1_CHUNK_KB", 0, 2, 96);
        c->tune.x1_block = env_int("SLDG_X1_BLOCK", 128, 64, 256) / 32 * 32;
        // columns per tile: a power of two in [8, 128] whose row is a multiple of 16 bytes; anything else is ignored
        int w = env_int("SLDG_TILE_W", 0, 8, 128);
        if (w > 0 && (w & (w - 1)) == 0 && (w * (int)c->esize) % 16 == 0) c->tune.tile_w = w;
    }
    {   // the context lives on the device that owns the caller's buffers (falls back to the current device)
        cudaPointerAttributes pa;
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaPointerGetAttributes(&pa, f_buf0) == cudaSuccess && pa.type == cudaMemoryTypeDevice) dev = pa.device;
        else cudaGetLastError();
        c->device = dev;
        cudaPointerAttributes pb;
        if (cudaPointerGetAttributes(&pb, f_buf1) == cudaSuccess && pb.type == cudaMemoryTypeDevice && pb.device != dev) {
            delete c;
            return fail(nullptr, SLDG_ERR_ARG, "sldg_create: the two f buffers live on different devices");
        }
        cudaGetLastError();
    }
    DeviceGuard guard(c);
    cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, c->device);

#define CREATE_TRY(call)                                                                        \
    do {                                                                                        \
        cudaError_t e_ = (call);                                                                \
        if (e_ != cudaSuccess) {                                                                \
            fail(nullptr, SLDG_ERR_CUDA, "sldg_create: %s: %s", #call, cudaGetErrorString(e_)); \
            free_tables(c); delete c; return SLDG_ERR_CUDA;                                     \
        }                                                                                       \
    } while (0)

    // A/B polynomial coefficients
    std::vector<double> coef = ab_polynomial_coefficients(order);
    CREATE_TRY(dalloc(&c->d_coef, coef.size()));
    CREATE_TRY(cudaMemcpy(c->d_coef, coef.data(), coef.size() * sizeof(double), cudaMemcpyHostToDevice));

    // node coordinates, sweep tables
    long maxN = 0;
    for (int d = 0; d < c->D; ++d) {
        std::vector<double> cc;
        host_node_coords(c, d, cc);
        CREATE_TRY(dalloc(&c->d_coords[d], cc.size()));
        CREATE_TRY(cudaMemcpy(c->d_coords[d], cc.data(), cc.size() * sizeof(double), cudaMemcpyHostToDevice));
        if (c->N[d] > maxN) maxN = c->N[d];
    }
    c->tab_cap = c->X > maxN ? c->X : maxN;
    for (auto &t : c->gen) {
        CREATE_TRY(dalloc(&t.sigma, c->tab_cap));
        CREATE_TRY(dalloc(&t.m, c->tab_cap));
        CREATE_TRY(cudaMalloc(&t.ab, (size_t)2 * order * order * c->tab_cap * c->esize));
    }
    for (int a = 0; a < dx; ++a) {
        sldg_ctx::Tab &t = c->xt[a];
        long cap = c->N[dx + a];
        CREATE_TRY(dalloc(&t.sigma, cap));
        CREATE_TRY(dalloc(&t.m, cap));
        CREATE_TRY(cudaMalloc(&t.ab, (size_t)2 * order * order * cap * c->esize));
    }

    // quadrature weights W_v = prod_a h_va w_ja (v_1 fastest), W_x likewise
    {
        std::vector<double> Wv(c->V), Wx(c->X);
        for (long v = 0; v < c->V; ++v) {
            long rem = v; double W = 1.0;
            for (int a = 0; a < dv; ++a) {
                long p = rem % c->N[dx + a]; rem /= c->N[dx + a];
                W *= c->h[dx + a] * c->w[p % order];
            }
            Wv[v] = W;
        }
        for (long x = 0; x < c->X; ++x) {
            long rem = x; double W = 1.0;
            for (int a = 0; a < dx; ++a) {
                long p = rem % c->N[a]; rem /= c->N[a];
                W *= c->h[a] * c->w[p % order];
            }
            Wx[x] = W;
        }
        {   // v-node coordinates and |v|^2 for the moment pass
            std::vector<double> va((size_t)dv * c->V), v2(c->V);
            std::vector<std::vector<double>> cv(dv);
            for (int a = 0; a < dv; ++a) host_node_coords(c, dx + a, cv[a]);
            for (long v = 0; v < c->V; ++v) {
                long rem = v; double s2 = 0.0;
                for (int a = 0; a < dv; ++a) {
                    long p = rem % c->N[dx + a]; rem /= c->N[dx + a];
                    va[(size_t)a * c->V + v] = cv[a][p];
                    s2 += cv[a][p] * cv[a][p];
                }
                v2[v] = s2;
            }
            CREATE_TRY(dalloc(&c->d_va, va.size()));
            CREATE_TRY(dalloc(&c->d_v2, v2.size()));
            CREATE_TRY(cudaMemcpy(c->d_va, va.data(), va.size() * sizeof(double), cudaMemcpyHostToDevice));
            CREATE_TRY(cudaMemcpy(c->d_v2, v2.data(), v2.size() * sizeof(double), cudaMemcpyHostToDevice));
        }
        CREATE_TRY(dalloc(&c->d_Wv, Wv.size()));
        CREATE_TRY(dalloc(&c->d_Wx, Wx.size()));
        CREATE_TRY(cudaMemcpy(c->d_Wv, Wv.data(), Wv.size() * sizeof(double), cudaMemcpyHostToDevice));
        CREATE_TRY(cudaMemcpy(c->d_Wx, Wx.data(), Wx.size() * sizeof(double), cudaMemcpyHostToDevice));
    }
    CREATE_TRY(dalloc(&c->d_rho, c->X));
    CREATE_TRY(dalloc(&c->d_s2, c->X));
    CREATE_TRY(dalloc(&c->d_E, c->X * dx));
    CREATE_TRY(dalloc(&c->d_mom, c->X * (dv + 1)));
    CREATE_TRY(cudaMemset(c->d_E, 0, c->X * dx * sizeof(double)));
    CREATE_TRY(cudaMemset(c->d_s2, 0, c->X * sizeof(double)));
    CREATE_TRY(dalloc(&c->d_scal, 8));
    CREATE_TRY(dalloc(&c->d_wide, 1));
    CREATE_TRY(dalloc(&c->d_wide_seen, 1));
    CREATE_TRY(cudaMemset(c->d_wide_seen, 0, sizeof(int)));
    {
        // enough v-splits that X/VEC * splits threads fill the machine several times over (6 waves of 2048/SM: with
        // 1-2 waves the last, partly filled wave cost up to half the pass -- fp32 config 5 had 1.003 waves, 4.6 TB/s)
        long target = (long)c->sm_count * 2048 * 6;
        const long vmax = 16 / (long)c->esize;
        long per = c->X / vmax > 0 ? c->X / vmax : 1;
        long s = cdiv(target, per);
        long smax = c->V / 256 > 0 ? c->V / 256 : 1;     // partials stay under 1/256 of f per quantity
        if (s > smax) s = smax;
        if (s < 1) s = 1;
        if (s > 8192) s = 8192;
        c->max_splits = (int)s;
        CREATE_TRY(dalloc(&c->d_part, (size_t)(3 + dv) * c->max_splits * c->X));
    }

    // Poisson: dense DFT matrices per x-dimension (D:R6)
    {
        const double PI = 3.14159265358979323846264338327950288;
        long big = c->X;
        for (int a = 0; a < dx; ++a) {
            c->Mmax[a] = (c->cells[a] - 1) / 2;
            c->K[a] = 2 * c->Mmax[a] + 1;
            c->KK *= c->K[a];
        }
        for (int a = 0; a < dx; ++a) {
            long Na = c->N[a], Ka = c->K[a];
            double L = c->hi[a] - c->lo[a];
            std::vector<double> cc;
            host_node_coords(c, a, cc);
            std::vector<double2> F((size_t)Ka * Na), G((size_t)Na * Ka);
            for (long r = 0; r < Ka; ++r) {
                double k = 2.0 * PI * (double)(r - c->Mmax[a]) / L;
                for (long p = 0; p < Na; ++p) {
                    double ph = k * cc[p];
                    double wq = c->w[p % order] * c->h[a] / L;
                    F[(size_t)r * Na + p] = make_double2(wq * cos(ph), -wq * sin(ph));
                    G[(size_t)p * Ka + r] = make_double2(cos(ph), sin(ph));
                }
            }
            CREATE_TRY(dalloc(&c->d_F[a], F.size()));
            CREATE_TRY(dalloc(&c->d_G[a], G.size()));
            CREATE_TRY(cudaMemcpy(c->d_F[a], F.data(), F.size() * sizeof(double2), cudaMemcpyHostToDevice));
            CREATE_TRY(cudaMemcpy(c->d_G[a], G.data(), G.size() * sizeof(double2), cudaMemcpyHostToDevice));
        }
        for (int i = 0; i < 4; ++i) CREATE_TRY(dalloc(&c->d_t[i], big));
        CREATE_TRY(dalloc(&c->d_gh[0], c->KK));
        CREATE_TRY(dalloc(&c->d_gh[1], c->KK));
    }
#undef CREATE_TRY
    *out = c;
    return SLDG_OK;
}

extern "C" int sldg_destroy(sldg_ctx *ctx) {
    if (!ctx) return SLDG_ERR_ARG;
    DeviceGuard guard(ctx);
    cudaStreamSynchronize(ctx->stream);
    for (auto &g : ctx->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
    if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
    free_tables(ctx);
    delete ctx;
    return SLDG_OK;
}

// ------------------------------------------------------------------------------------------
// f in / out
// ------------------------------------------------------------------------------------------
extern "C" int sldg_set_initial(sldg_ctx *c, const void *src, int is_device) {
    if (!c || !src) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    size_t bytes = (size_t)c->ndof * c->esize;
    CUDA_TRY(c, cudaMemcpyAsync(c->buf[c->cur], src, bytes,
                                is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    if (!is_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    f_changed(c);
    return SLDG_OK;
}

extern "C" int sldg_get_f(sldg_ctx *c, void *dst, int is_device) {
    if (!c || !dst) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    size_t bytes = (size_t)c->ndof * c->esize;
    CUDA_TRY(c, cudaMemcpyAsync(dst, c->buf[c->cur], bytes,
                                is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    if (!is_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return SLDG_OK;
}

extern "C" int sldg_fill_uniform(sldg_ctx *c, unsigned long long seed, unsigned tag) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int blocks = c->sm_count * 8;
    if (c->dtype == SLDG_F64)
        fill_uniform_kernel<double><<<blocks, 256, 0, c->stream>>>((double *)c->buf[c->cur], c->ndof, seed, tag);
    else
        fill_uniform_kernel<float><<<blocks, 256, 0, c->stream>>>((float *)c->buf[c->cur], c->ndof, seed, tag);
    LAUNCH_CHECK(c);
    f_changed(c);
    return SLDG_OK;
}

// ------------------------------------------------------------------------------------------
// sweeps: a-1 (assemble) + a-2 (translate), d_sigma[0..count) already filled on the stream
// ------------------------------------------------------------------------------------------
namespace {

template <typename T, int O, int VEC, bool QV>
void launch_strided(sldg_ctx *c, const T *in, T *out, long inner, int n, long outer, long count,
                    long qdiv, long qmod) {
    constexpr int UB = (O <= 4) ? 4 : 2;
    long lines_v = outer * (inner / VEC);
    // split lines into segments only when there are too few of them to fill the machine
    long target = (long)c->sm_count * 2048;
    int nseg = 1;
    if (lines_v < target) {
        nseg = (int)cdiv(target, lines_v);
        int maxseg = n / 4 > 0 ? n / 4 : 1;
        if (nseg > maxseg) nseg = maxseg;
    }
    int cps = (int)cdiv(n, nseg);
    nseg = (int)cdiv(n, cps);
    long threads = lines_v * nseg;
    int block = 256;
    long blocks = cdiv(threads, block);
    sweep_strided_kernel<T, O, VEC, QV, UB><<<(unsigned)blocks, block, 0, c->stream>>>(
        in, out, inner, n, outer, nseg, cps, c->d_m, (const T *)c->d_ab, count, qdiv, qmod, c->X);
}

template <typename T, int O>
int run_sweep_t(sldg_ctx *c, int dim, long count) {
    const int n = c->cells[dim];
    const T *in = (const T *)c->buf[c->cur];
    T *out = (T *)c->buf[c->cur ^ 1];
    // a-1
    if (!c->skip_asm1) {
        int block = 128;
        size_t sh = (size_t)2 * O * O * 2 * O * 2 * sizeof(double);
        assemble_ab_kernel<T><<<(unsigned)cdiv(count, block), block, sh, c->stream>>>(
            c->d_sigma, count, O, n, c->d_coef, c->d_m, (T *)c->d_ab);
        LAUNCH_CHECK(c);
    }
    long inner = 1, outer = 1;
    for (int d = 0; d < dim; ++d) inner *= c->N[d];
    for (int d = dim + 1; d < c->D; ++d) outer *= c->N[d];
    if (dim == 0) {
        // lines sharing a shift: q = (line / qdiv) % N_{v_1}, qdiv = prod_{1<=d<dx} N_d
        long qdiv = 1;
        for (int d = 1; d < c->dx; ++d) qdiv *= c->N[d];
        long ngroups = outer / qdiv;
        long cpg = qdiv * n;                       // cells per group
        const size_t line_bytes = (size_t)n * O * sizeof(T);
        bool done = false;
        if (c->use_tma && line_bytes % 16 == 0 && line_bytes <= 96 * 1024) {
            // staged variant: R whole lines per block through shared memory (bulk copies)
            // 16 KB chunks and 128-thread blocks at every order: ~7 blocks per SM, so that loads, arithmetic and stores
            // of different blocks overlap (config 4 dim 0, GB/s: 32 KB x 256 threads 6391, 16 KB x 128 7038, 8 KB x 128
            // 6068, 12 KB x 128 7054, 48 KB x 256 5995; fp32 6198 -> 7045)
            long chunk_bytes = 16 * 1024;
            int max_block = 128;
            if (c->tune.x1_chunk_kb) { chunk_bytes = (long)c->tune.x1_chunk_kb * 1024; max_block = c->tune.x1_block; }
            // shift groups: d_x >= 2: qdiv contiguous lines per (v_1 node, rest); d_x = 1: the lines of one
            // v_1 node are N_v1 lines apart (group = v_1 node, outer / N_v1 strided lines)
            const bool strided_group = (qdiv == 1 && outer > c->N[c->dx]);
            const long lpg = strided_group ? outer / c->N[c->dx] : qdiv;          // lines per group
            const long groups = strided_group ? c->N[c->dx] : ngroups;
            const long group_stride = strided_group ? (long)n * O : qdiv * (long)n * O;
            const long line_stride = strided_group ? c->N[c->dx] * (long)n * O : (long)n * O;
            long R = chunk_bytes / (long)line_bytes;
            if (R < 1) R = 1;
            if (R > lpg) R = lpg;
            int chunks = (int)cdiv(lpg, R);
            size_t half = ((size_t)R * line_bytes + 127) & ~(size_t)127;
            size_t smem = 2 * half;
            // O >= 4: a cell's outputs split over two threads
            constexpr int JH = (O >= 4) ? (O + 1) / 2 : O;
            auto go = [&](auto kern, int NP) -> int {
                CUDA_TRY(c, ensure_smem(c, kern, smem));
                long nitem = R * n * NP;
                const int mb = max_block;
                int block = nitem >= mb ? mb : (int)(cdiv(nitem, 32) * 32);
                if (block < 64) block = 64;
                if (block % NP) block = (block / NP + 1) * NP;
                kern<<<(unsigned)(groups * chunks), block, smem, c->stream>>>(
                    in, out, n, lpg, (int)R, chunks, c->d_m, (const T *)c->d_ab, count, c->N[c->dx], group_stride,
                    line_stride);
                return SLDG_OK;
            };
            // measured (2+2 D, fp64, GB/s): o = 2 whole cell 6690 / per node 6001; o = 3 whole 6617 / split 5881;
            // o = 4 whole 5764 / split 7046; o = 6 whole 3700 / split 5663
            int rc;
            if (c->twice_req && c->dx == 1) {            // x(tau) x(tau) of two consecutive steps in one pass
                rc = go(sweep_x1_bulk_kernel<T, O, JH, true>, (O + JH - 1) / JH);
                c->twice_done = true;
            } else {
                rc = go(sweep_x1_bulk_kernel<T, O, JH>, (O + JH - 1) / JH);
            }
            if (rc) return rc;
            done = true;
        }
        if (!done) {
            int block = 256;
            int cpb = 2048;                        // cells per block
            if (cpg < cpb) { cpb = (int)cpg; if (cpb < block) block = (int)(cdiv(cpb, 32) * 32); }
            int bpg = (int)cdiv(cpg, cpb);
            sweep_x1_kernel<T, O><<<(unsigned)(ngroups * bpg), block, 0, c->stream>>>(
                in, out, n, ngroups, cpg, cpb, bpg, c->d_m, (const T *)c->d_ab, count, c->N[c->dx]);
        }
    } else if (dim == 1 && c->dx >= 2 && sizeof(T) == 8 && O <= 5 && c->use_tma && c->tune.plane_single && c->cells[0] <= 256 && n >= 3 &&
               ((size_t)O * c->cells[0] * O * sizeof(T)) % 16 == 0 &&
               4 * (((size_t)O * c->cells[0] * O * sizeof(T) + 127) & ~(size_t)127) <= 96 * 1024 && outer < (1L << 31)) {
        // x_2: one block per (x_1,x_2) plane, the plane kernel of the fused x-pair with the x_1 rule skipped (slabs
        // streamed by the copy engine): config 4 dim 1 6.44 -> 6.6 TB/s against the register-window kernel below; fp64
        // only (fp32, config 4: 5.9 against 6.4 TB/s for the 128-bit register-window kernel) and o <= 5 (2+2 D, 3.3e9 DOF,
        // plane / register-window in TB/s: o = 3 6.62 / 6.16, o = 4 6.51 / 6.21, o = 5 6.43 / 5.40, o = 6 4.19 / 5.54 --
        // at o = 6 the 2 o^2 = 72 coefficients per thread no longer fit beside the window)
        const int n1 = c->cells[0];
        const size_t slot = ((size_t)O * n1 * O * sizeof(T) + 127) & ~(size_t)127;
        long qd2 = 1;                                        // q of a plane: (first element / qd2) % qm2
        for (int d = 0; d < c->dx + 1; ++d) qd2 *= c->N[d];
        const long qm2 = c->N[c->dx + 1];
        int ppb = 32 / n1;
        if (ppb < 1) ppb = 1;
        if (ppb > 8) ppb = 8;
        const int blk = (int)(cdiv((long)ppb * n1, 32) * 32);
        if (ppb > 1) {
            CUDA_TRY(c, ensure_smem(c, sweep_xpair_plane_kernel<T, O, true, true>, 4 * slot * ppb));
            sweep_xpair_plane_kernel<T, O, true, true><<<(unsigned)cdiv(outer, ppb), blk, 4 * slot * ppb, c->stream>>>(
                in, out, n1, n, ppb, outer, nullptr, nullptr, 0, 1, 1, c->d_m, (const T *)c->d_ab, count, qd2, qm2);
        } else {
            CUDA_TRY(c, ensure_smem(c, sweep_xpair_plane_kernel<T, O, true>, 4 * slot));
            sweep_xpair_plane_kernel<T, O, true><<<(unsigned)outer, blk, 4 * slot, c->stream>>>(
                in, out, n1, n, 1, outer, nullptr, nullptr, 0, 1, 1, c->d_m, (const T *)c->d_ab, count, qd2, qm2);
        }
    } else if (dim < c->dx) {
        const int dep = c->dx + dim;
        long qdiv = 1;
        for (int d = dim + 1; d < dep; ++d) qdiv *= c->N[d];
        const long qmod = c->N[dep];
        constexpr int VMAX = 16 / (int)sizeof(T);
        if (inner % VMAX == 0) launch_strided<T, O, VMAX, false>(c, in, out, inner, n, outer, count, qdiv, qmod);
        else if (inner % 2 == 0) launch_strided<T, O, 2, false>(c, in, out, inner, n, outer, count, qdiv, qmod);
        else launch_strided<T, O, 1, false>(c, in, out, inner, n, outer, count, qdiv, qmod);
    } else {
        bool done = false;
        const long Nk = (long)n * O;
        // rows of up to 1 KB (at most 128 columns = one per thread), halved below until the tile fits: 512-byte rows at
        // configs 3 and 4 (+0.5-0.9 % over 256 B), 1 KB rows at config 5 (40-node lines: v-sweeps 6.35-6.73 -> 6.64-6.85 TB/s)
        int W = 1024 / (int)sizeof(T);
        if (W > 128) W = 128;
        if (c->tune.tile_w) W = c->tune.tile_w;              // tuning knob (columns per tile), validated in sldg_create
        while (W > 8 && W > inner) W /= 2;                   // never wider than the line of columns
        int nbox = (int)cdiv(Nk, 256);
        int box_rows = (int)cdiv(Nk, nbox);
        while (W > 8 && (size_t)nbox * box_rows * W * sizeof(T) > 100 * 1024) W /= 2;
        {   // every TMA box must land on a 128-byte aligned shared-memory address
            int align = 128 / (W * (int)sizeof(T));
            if (align > 1) box_rows = (int)(cdiv(box_rows, align) * align);
            if (box_rows > 256) { nbox += 1; box_rows = (int)(cdiv(cdiv(Nk, nbox), align > 1 ? align : 1) * (align > 1 ? align : 1)); }
        }
        size_t smem = (size_t)nbox * box_rows * W * sizeof(T);
        if (c->use_tma && (inner * sizeof(T)) % 16 == 0 && inner >= W && smem <= 200 * 1024 &&
            inner < (1L << 31) && outer < (1L << 31)) {
            sldg_ctx::TmapSlot &ts = c->tmap3[dim][c->cur];
            if (!ts.valid || ts.p0 != W || ts.p1 != box_rows) {
                ts.valid = make_tensor_map_3d(&ts.map, in, sizeof(T) == 8, (uint64_t)inner, (uint64_t)Nk, (uint64_t)outer,
                                              (uint32_t)W, (uint32_t)box_rows);
                ts.p0 = W; ts.p1 = box_rows;
            }
            if (ts.valid) {
                const CUtensorMap &tmap = ts.map;
                CUDA_TRY(c, ensure_smem(c, sweep_tile_tma_kernel<T, O>, smem));
                int nseg = 128 / W;                       // (256 / 512 threads per tile measured: 1-2 % / 15 % slower)
                int cps = (int)cdiv(n, nseg);
                long tpo = cdiv(inner, W);
                sweep_tile_tma_kernel<T, O><<<(unsigned)(tpo * outer), 128, smem, c->stream>>>(
                    tmap, out, inner, n, tpo, W, nbox, box_rows, cps, c->d_m, (const T *)c->d_ab, count, c->X);
                done = true;
            }
        }
        if (!done) launch_strided<T, O, 1, true>(c, in, out, inner, n, outer, count, 1, 1);
    }
    LAUNCH_CHECK(c);
    c->cur ^= 1;
    f_changed(c);
    return SLDG_OK;
}

template <typename T>
int run_sweep_o(sldg_ctx *c, int dim, long count) {
    switch (c->o) {
    case 1: return run_sweep_t<T, 1>(c, dim, count);
    case 2: return run_sweep_t<T, 2>(c, dim, count);
    case 3: return run_sweep_t<T, 3>(c, dim, count);
    case 4: return run_sweep_t<T, 4>(c, dim, count);
    case 5: return run_sweep_t<T, 5>(c, dim, count);
    case 6: return run_sweep_t<T, 6>(c, dim, count);
    }
    return fail(c, SLDG_ERR_UNSUPPORTED, "order %d not instantiated", c->o);
}

int run_sweep(sldg_ctx *c, int dim, long count) {
    return c->dtype == SLDG_F64 ? run_sweep_o<double>(c, dim, count) : run_sweep_o<float>(c, dim, count);
}

// ---- fused pair of sweeps (sweep_fused.cuh); d_sigma / d_sigma2 hold the two shift tables ----
// x_1 x_2 pair + rho (sweep_xpair_rho_kernel): ONE wave of equal blocks = (x_2-cell groups) x (plane chunks)
template <typename T, int O, int C2R>
int launch_xpair_rho(sldg_ctx *c, const T *in, T *out, int n1, int n2, long planes, long count1, long qd1, long qm1,
                     long count2, long qd2, long qm2) {
    const size_t slab_bytes = (size_t)O * n1 * O * sizeof(T);
    const size_t slot = (slab_bytes + 127) & ~(size_t)127;
    const size_t smem = 8 * slot;
    auto kern = sweep_xpair_rho_kernel<T, O, C2R>;
    // shift index of plane p: q_i = (p / pdiv_i) % pmod_i (a plane is X = qd1 elements when d_x = 2)
    const long X = (long)n1 * O * n2 * O;
    qd1 /= X; qd2 /= X;
    CUDA_TRY(c, ensure_smem(c, kern, smem));
    const int blk = (int)(cdiv(n1, 32) * 32);
    int per_sm = 0;
    CUDA_TRY(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, blk, smem));
    if (per_sm < 1) per_sm = 1;
    const long G = cdiv(n2, C2R);
    long nchunk = (long)c->sm_count * per_sm / G;
    const long cap = (long)(3 + c->dv) * c->max_splits;
    if (nchunk > cap) nchunk = cap;
    if (nchunk > planes) nchunk = planes;
    if (nchunk < 1) nchunk = 1;
    kern<<<(unsigned)(nchunk * G), blk, smem, c->stream>>>(
        in, out, n1, n2, planes, (int)nchunk, c->d_m, (const T *)c->d_ab, count1, qd1, qm1, c->d_m2,
        (const T *)c->d_ab2, count2, qd2, qm2, c->d_Wv, c->d_part);
    LAUNCH_CHECK(c);
    c->rho_rows = (int)nchunk;
    return SLDG_OK;
}

template <typename T, int O>
int run_pair_t(sldg_ctx *c, int k1, int k2, long count1, long count2) {
    const int n1 = c->cells[k1], n2 = c->cells[k2];
    const T *in = (const T *)c->buf[c->cur];
    T *out = (T *)c->buf[c->cur ^ 1];
    int block = 128;
    size_t sh = (size_t)2 * O * O * 2 * O * 2 * sizeof(double);
    // fused v-sweeps are built for |shift| < 1 cell: a wider line costs bandwidth (per-block fallback); the table
    // assembly leaves a sticky mark the caller can read (sldg_wide_shift_seen)
    int *seen = k1 >= c->dx ? c->d_wide_seen : nullptr;
    if (!c->skip_asm1) {
        assemble_ab_kernel<T><<<(unsigned)cdiv(count1, block), block, sh, c->stream>>>(
            c->d_sigma, count1, O, n1, c->d_coef, c->d_m, (T *)c->d_ab, seen);
        LAUNCH_CHECK(c);
    }
    if (!c->skip_asm2) {
        assemble_ab_kernel<T><<<(unsigned)cdiv(count2, block), block, sh, c->stream>>>(
            c->d_sigma2, count2, O, n2, c->d_coef, c->d_m2, (T *)c->d_ab2, seen);
        LAUNCH_CHECK(c);
    }
    long inner1 = 1, midN = 1, outer2 = 1;
    for (int d = 0; d < k1; ++d) inner1 *= c->N[d];
    for (int d = k1 + 1; d < k2; ++d) midN *= c->N[d];
    for (int d = k2 + 1; d < c->D; ++d) outer2 *= c->N[d];
    auto qmap = [&](int k, long &qdiv, long &qmod) {
        if (k < c->dx) {
            qdiv = 1;
            for (int d = 0; d < c->dx + k; ++d) qdiv *= c->N[d];
            qmod = c->N[c->dx + k];
        } else { qdiv = 1; qmod = c->X; }
    };
    long qd1, qm1, qd2, qm2;
    qmap(k1, qd1, qm1);
    qmap(k2, qd2, qm2);
    long lines = inner1 * n1 * midN * outer2;
    long target = (long)c->sm_count * 1024;
    int nseg = 1;
    if (lines < target) {
        nseg = (int)cdiv(target, lines);
        int maxseg = n2 / 4 > 0 ? n2 / 4 : 1;
        if (nseg > maxseg) nseg = maxseg;
    }
    int cps = (int)cdiv(n2, nseg);
    nseg = (int)cdiv(n2, cps);
    long threads = lines * nseg;
    int chunk = 32;
    while (inner1 % chunk) chunk /= 2;
    // x_1 x_2 (the whole x-group of a d_x = 2 step) with rho accumulated in the same pass
    if (c->want_rho && c->use_tma && (O == 2 || O == 3 || c->tune.rho_cells) && k1 == 0 && k2 == 1 && c->dx == 2 && n1 <= 256 && n2 >= 2 &&
        ((size_t)O * n1 * O * sizeof(T)) % 16 == 0 && 8 * (((size_t)O * n1 * O * sizeof(T) + 127) & ~(size_t)127) <= 96 * 1024) {
        const long planes = midN * outer2;                   // = V
        int cells = c->tune.rho_cells ? c->tune.rho_cells : (O == 1 ? 8 : 4);   // config 3: 4 cells 0.717 ms, 8 cells 0.822 ms (186 registers)
        int rc = -1;
        if constexpr (O <= 2) {
            if (cells >= 8) rc = launch_xpair_rho<T, O, 8>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
            else if (cells >= 4) rc = launch_xpair_rho<T, O, 4>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
            else rc = launch_xpair_rho<T, O, 2>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
        } else if constexpr (O == 3) {
            if (cells >= 4) rc = launch_xpair_rho<T, O, 4>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
            else rc = launch_xpair_rho<T, O, 2>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
        } else {
            rc = launch_xpair_rho<T, O, 2>(c, in, out, n1, n2, planes, count1, qd1, qm1, count2, qd2, qm2);
        }
        if (rc) return rc;
        c->cur ^= 1;
        f_changed(c);
        return SLDG_OK;
    }
    // x_1 x_2: copy-engine staged plane kernel, one block per (x_1, x_2) plane
    {
        const size_t slab_bytes = (size_t)O * n1 * O * sizeof(T);
        const size_t slot = (slab_bytes + 127) & ~(size_t)127;
        const long planes = midN * outer2;           // midN == 1 for (0, 1)
        if (c->use_tma && c->tune.plane_pair && k1 == 0 && k2 == 1 && slab_bytes % 16 == 0 && 4 * slot <= 96 * 1024 &&
            n1 <= 256 && n2 >= 3 && planes < (1L << 31)) {
            int blk = (int)(cdiv(n1, 32) * 32);
            bool twice = false;
            if constexpr (O <= 3) twice = c->twice_req && c->dx == 2;
            if (twice) {
                if constexpr (O <= 3) {                      // x(tau) x(tau) of two consecutive steps in one pass
                    CUDA_TRY(c, ensure_smem(c, sweep_xpair_plane2_kernel<T, O>, 5 * slot));
                    sweep_xpair_plane2_kernel<T, O><<<(unsigned)planes, blk, 5 * slot, c->stream>>>(
                        in, out, n1, n2, c->d_m, (const T *)c->d_ab, count1, qd1, qm1, c->d_m2, (const T *)c->d_ab2,
                        count2, qd2, qm2);
                    c->twice_done = true;
                }
            } else {
                // several planes per block when the x_1 line is shorter than a warp (2+3 D, n_1 = 16, o = 4:
                // x-pair 11.5 -> see DESIGN.md)
                int ppb = 32 / n1;
                if (ppb < 1) ppb = 1;
                if (ppb > 8) ppb = 8;
                const size_t smem_pp = 4 * slot * ppb;
                const int blk_pp = (int)(cdiv((long)ppb * n1, 32) * 32);
                if (ppb > 1) {
                    CUDA_TRY(c, ensure_smem(c, sweep_xpair_plane_kernel<T, O, false, true>, smem_pp));
                    sweep_xpair_plane_kernel<T, O, false, true><<<(unsigned)cdiv(planes, ppb), blk_pp, smem_pp, c->stream>>>(
                        in, out, n1, n2, ppb, planes, c->d_m, (const T *)c->d_ab, count1, qd1, qm1, c->d_m2,
                        (const T *)c->d_ab2, count2, qd2, qm2);
                } else {
                    CUDA_TRY(c, ensure_smem(c, sweep_xpair_plane_kernel<T, O>, smem_pp));
                    sweep_xpair_plane_kernel<T, O><<<(unsigned)planes, blk_pp, smem_pp, c->stream>>>(
                        in, out, n1, n2, 1, planes, c->d_m, (const T *)c->d_ab, count1, qd1, qm1, c->d_m2,
                        (const T *)c->d_ab2, count2, qd2, qm2);
                }
            }
            LAUNCH_CHECK(c);
            c->cur ^= 1;
            f_changed(c);
            return SLDG_OK;
        }
    }
    // v_a v_b at o >= 3: TMA-tile staged kernel for |shift| < 1 (lanes along inner1, per-cell tensor boxes);
    // at o <= 2 the register kernel below is as fast
    {
        // SLDG_TILE_PAIR: 0 = never, 1 = also at o <= 2
        const bool want = c->tune.tile_pair >= 0 ? (c->tune.tile_pair == 1) : (O >= 3);
        const long blocks = (inner1 / 32) * (n1 / 4) * outer2;
        if (c->use_tma && want && k1 >= c->dx && midN == 1 && inner1 % 32 == 0 && n1 % 4 == 0 &&
            n1 >= 4 && n2 >= 3 && inner1 < (1L << 31) && outer2 < (1L << 31) && blocks < (1L << 31)) {
            sldg_ctx::TmapSlot &ts = c->tmap4[k1][c->cur];
            if (!ts.valid || ts.p0 != k2) {
                ts.valid = make_tensor_map_4d(&ts.map, in, sizeof(T) == 8, (uint64_t)inner1, (uint64_t)n1 * O,
                                              (uint64_t)n2 * O, (uint64_t)outer2, 32, O, O);
                ts.p0 = k2;
            }
            if (ts.valid) {
                const CUtensorMap &tmap = ts.map;
                const size_t smem = (size_t)3 * 6 * O * O * 32 * sizeof(T);
                CUDA_TRY(c, ensure_smem(c, sweep_vpair_tile_kernel<T, O>, smem));
                sweep_vpair_tile_kernel<T, O><<<(unsigned)blocks, 128, smem, c->stream>>>(
                    tmap, in, out, inner1, n1, n2, outer2, c->d_m, (const T *)c->d_ab, count1, qd1, qm1, c->d_m2,
                    (const T *)c->d_ab2, count2, qd2, qm2);
                LAUNCH_CHECK(c);
                c->cur ^= 1;
                f_changed(c);
                return SLDG_OK;
            }
        }
    }
    // (the vectorised-cell variant VEC1 helps the triple kernel but measured slower for the pair
    //  kernel at config 3: 0.906 vs 0.704 ms, so the pair always uses scalar accesses)
    sweep_pair_kernel<T, O, false><<<(unsigned)cdiv(threads, 128), 128, 0, c->stream>>>(
            in, out, inner1, n1, midN, n2, outer2, nseg, cps, chunk, c->d_m, (const T *)c->d_ab, count1, qd1, qm1,
            c->d_m2, (const T *)c->d_ab2, count2, qd2, qm2);
    LAUNCH_CHECK(c);
    c->cur ^= 1;
    f_changed(c);
    return SLDG_OK;
}

int run_pair(sldg_ctx *c, int k1, int k2, long count1, long count2) {
#define PAIR_CASE(TT)                                                           \
    switch (c->o) {                                                             \
    case 1: return run_pair_t<TT, 1>(c, k1, k2, count1, count2);                \
    case 2: return run_pair_t<TT, 2>(c, k1, k2, count1, count2);                \
    case 3: return run_pair_t<TT, 3>(c, k1, k2, count1, count2);                \
    case 4: return run_pair_t<TT, 4>(c, k1, k2, count1, count2);                \
    }
    if (c->dtype == SLDG_F64) { PAIR_CASE(double) } else { PAIR_CASE(float) }
#undef PAIR_CASE
    return fail(c, SLDG_ERR_UNSUPPORTED, "order %d not instantiated", c->o);
}

// ---- fused triple of sweeps (sweep_fused.cuh: sweep_triple_kernel), o <= 2 -------------------
template <typename T, int O>
int run_triple_t(sldg_ctx *c, int k1, int k2, int k3, long cnt1, long cnt2, long cnt3) {
    const int n1 = c->cells[k1], n2 = c->cells[k2], n3 = c->cells[k3];
    const T *in = (const T *)c->buf[c->cur];
    T *out = (T *)c->buf[c->cur ^ 1];
    int block = 128;
    size_t sh = (size_t)2 * O * O * 2 * O * 2 * sizeof(double);
    const bool skip[3] = {c->skip_asm1, c->skip_asm2, c->skip_asm3};
    double *sg[3] = {c->d_sigma, c->d_sigma2, c->d_sigma3};
    int *mm[3] = {c->d_m, c->d_m2, c->d_m3};
    void *ab[3] = {c->d_ab, c->d_ab2, c->d_ab3};
    const long cnt[3] = {cnt1, cnt2, cnt3};
    const int nn[3] = {n1, n2, n3};
    for (int i = 0; i < 3; ++i)
        if (!skip[i]) {
            assemble_ab_kernel<T><<<(unsigned)cdiv(cnt[i], block), block, sh, c->stream>>>(
                sg[i], cnt[i], O, nn[i], c->d_coef, mm[i], (T *)ab[i], k1 >= c->dx ? c->d_wide_seen : nullptr);
            LAUNCH_CHECK(c);
        }
    long inner1 = 1, mid12 = 1, mid23 = 1, outer3 = 1;
    for (int d = 0; d < k1; ++d) inner1 *= c->N[d];
    for (int d = k1 + 1; d < k2; ++d) mid12 *= c->N[d];
    for (int d = k2 + 1; d < k3; ++d) mid23 *= c->N[d];
    for (int d = k3 + 1; d < c->D; ++d) outer3 *= c->N[d];
    long qd[3], qm[3];
    const int ks[3] = {k1, k2, k3};
    for (int i = 0; i < 3; ++i) {
        if (ks[i] < c->dx) {
            qd[i] = 1;
            for (int d = 0; d < c->dx + ks[i]; ++d) qd[i] *= c->N[d];
            qm[i] = c->N[c->dx + ks[i]];
        } else { qd[i] = 1; qm[i] = c->X; }
    }
    // x_1 x_2 x_3 (the whole x-group of a d_x = 3 step) with rho accumulated in the same pass
    // (config 5: 17.7 ms fused vs 12.0 + 5.3 ms -- the accumulators have to live in shared memory and the plane
    //  kernel is bound by shared-memory wavefronts already; SLDG_RHO_TRIPLE=1 enables it)
    if (c->want_rho && c->tune.rho_triple && c->use_tma && k1 == 0 && k2 == 1 && k3 == 2 && c->dx == 3 && (long)n1 * n2 <= 512 && n3 >= 2 &&
        ((size_t)O * n2 * O * n1 * O * sizeof(T)) % 16 == 0) {
        const size_t slab_bytes = (size_t)O * n2 * O * n1 * O * sizeof(T);
        const size_t slot = (slab_bytes + 127) & ~(size_t)127;
        const size_t slab_acc = (size_t)O * n2 * O * n1 * O * sizeof(double);
        auto go = [&](auto kern, int C3R, int NS) -> int {
            const size_t smem = NS * slot + C3R * slab_acc;
            if (smem > 226 * 1024) return 1;
            if (ensure_smem(c, kern, smem) != cudaSuccess) { cudaGetLastError(); return 1; }
            const int blk = (int)(cdiv((long)n1 * n2, 32) * 32);
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, blk, smem) != cudaSuccess || per_sm < 1) {
                cudaGetLastError();
                return 1;
            }
            const long G = cdiv(n3, C3R);
            long nchunk = (long)c->sm_count * per_sm / G;
            const long cap = (long)(3 + c->dv) * c->max_splits;
            if (nchunk > cap) nchunk = cap;
            if (nchunk > outer3) nchunk = outer3;
            if (nchunk < 1) nchunk = 1;
            kern<<<(unsigned)(nchunk * G), blk, smem, c->stream>>>(
                in, out, n1, n2, n3, outer3, (int)nchunk, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2], c->d_Wv, c->d_part);
            c->rho_rows = (int)nchunk;
            return 0;
        };
        // range of x_3-cells per block: as many as fit beside a 3-deep ring (fewer cells = more neighbour slabs)
        int rc = 1;
        const int want = c->tune.rho_cells;
        if (rc && (want == 0 || want == 5)) rc = go(sweep_xtriple_rho_kernel<T, O, 5, 3>, 5, 3);
        if (rc && (want == 0 || want == 4)) rc = go(sweep_xtriple_rho_kernel<T, O, 4, 4>, 4, 4);
        if (rc && (want == 0 || want == 2)) rc = go(sweep_xtriple_rho_kernel<T, O, 2, 4>, 2, 4);
        if (rc == 0) {
            LAUNCH_CHECK(c);
            c->cur ^= 1;
            f_changed(c);
            return SLDG_OK;
        }
    }
    // x_1 x_2 x_3 with a small x-grid: copy-engine staged plane kernel, one block per velocity node
    {
        const size_t slab_bytes = (size_t)O * n2 * O * n1 * O * sizeof(T);
        const size_t slot = (slab_bytes + 127) & ~(size_t)127;
        if (c->use_tma && k1 == 0 && k2 == 1 && k3 == 2 && c->dx == 3 && slab_bytes % 16 == 0 &&
            4 * slot <= 200 * 1024 && (long)n1 * n2 <= 512 && outer3 < (1L << 31)) {
            // Part-plane blocks (nb2 ranges of x_2-cells per velocity node): two resident blocks whose phases overlap
            {
                // (config 5: single application 12.2 -> 11.5 ms, and -> 9.9 ms with two x_2-cells per thread
                //  (sweep_xtriple_part2_kernel); applied twice the part kernel spills and computes a row of cells
                //  redundantly: 22.9 ms against 21.1 ms for the whole plane, so twice stays on whole planes unless
                //  SLDG_XTRIPLE_PARTS asks otherwise -- and is off in 3+3 D, where two passes of 9.9 ms beat it)
                const int nb2 = c->tune.xt_parts ? c->tune.xt_parts : (c->twice_req ? 1 : 2);
                const int apps = (c->twice_req && n3 >= 2) ? 2 : 1;
                if (nb2 >= 2 && n2 % nb2 == 0 && n2 / nb2 >= 2) {
                    const int c2b = n2 / nb2;
                    const long thr = (long)(c2b + apps - 1) * n1;
                    const int blk = (int)(cdiv(thr, 32) * 32);
                    const size_t rowb = (size_t)O * n1 * sizeof(T);          // one row of the (x_1,x_2)-plane
                    const size_t slot_p = ((size_t)O * (c2b + apps) * O * rowb + 127) & ~(size_t)127;
                    const size_t tb_p = ((size_t)O * (c2b + apps - 1) * O * rowb + 127) & ~(size_t)127;
                    const size_t smem_p = (apps == 1 ? 4 * slot_p : 3 * slot_p + 2 * tb_p) +
                                          (size_t)apps * O * O * O * blk * sizeof(T);
                    if (thr <= 256 && smem_p <= 110 * 1024 && rowb % 16 == 0 && outer3 * nb2 < (1L << 31)) {
                        cudaError_t e;
                        if (apps == 2) {
                            auto kern = sweep_xtriple_part_kernel<T, O, 2>;
                            e = ensure_smem(c, kern, smem_p);
                            if (e == cudaSuccess)
                                kern<<<(unsigned)(outer3 * nb2), blk, smem_p, c->stream>>>(
                                    in, out, n1, n2, n3, c2b, nb2, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                                    (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
                        } else if (c2b % 2 == 0 && c->tune.xt_two) {
                            // two x_2-cells per thread: half the threads, the shared source cell swept once
                            auto kern = sweep_xtriple_part2_kernel<T, O>;
                            const int blk2 = (int)(cdiv((long)(c2b / 2) * n1, 32) * 32);
                            const size_t smem2c = 4 * slot_p + (size_t)2 * O * O * O * blk2 * sizeof(T);
                            e = blk2 <= 128 ? ensure_smem(c, kern, smem2c) : cudaErrorInvalidValue;
                            if (e == cudaSuccess)
                                kern<<<(unsigned)(outer3 * nb2), blk2, smem2c, c->stream>>>(
                                    in, out, n1, n2, n3, c2b, nb2, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                                    (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
                        } else {
                            auto kern = sweep_xtriple_part_kernel<T, O, 1>;
                            e = ensure_smem(c, kern, smem_p);
                            if (e == cudaSuccess)
                                kern<<<(unsigned)(outer3 * nb2), blk, smem_p, c->stream>>>(
                                    in, out, n1, n2, n3, c2b, nb2, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                                    (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
                        }
                        if (e == cudaSuccess) {
                            LAUNCH_CHECK(c);
                            if (apps == 2) c->twice_done = true;
                            c->cur ^= 1;
                            f_changed(c);
                            return SLDG_OK;
                        }
                        cudaGetLastError();
                    }
                }
            }
            // threads per x_2-cell row: dense.  (n1 rounded up to a multiple of 8 makes the 16-byte shared-memory
            // accesses conflict-free -- with n1 = 20 a quarter warp straddles two rows, 23 % of the wavefronts are
            // conflicts -- but the idle lanes cost more: config 5 triple 11.7 -> 12.2 ms, applied twice 20.7 -> 24.6 ms)
            int tpr = n1;
            int block = (int)(cdiv((long)tpr * n2, 32) * 32);
            // twice: ring + the first application's cell + the two parked first cells of the windows
            const size_t smem2 = 5 * slot + (size_t)2 * O * O * O * block * sizeof(T);   // 3-deep ring, 2 cells, parked
            if (c->twice_req && n3 >= 2 && smem2 <= 226 * 1024 &&
                ensure_smem(c, sweep_xtriple_plane2_kernel<T, O>, smem2) == cudaSuccess) {
                sweep_xtriple_plane2_kernel<T, O><<<(unsigned)outer3, block, smem2, c->stream>>>(
                    in, out, n1, n2, n3, tpr, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1], (const T *)ab[1], cnt2,
                    qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
                c->twice_done = true;
            } else {
                cudaGetLastError();
                CUDA_TRY(c, ensure_smem(c, sweep_xtriple_plane_kernel<T, O>, 4 * slot));
                sweep_xtriple_plane_kernel<T, O><<<(unsigned)outer3, block, 4 * slot, c->stream>>>(
                    in, out, n1, n2, n3, tpr, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1], (const T *)ab[1], cnt2,
                    qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
            }
            LAUNCH_CHECK(c);
            c->cur ^= 1;
            f_changed(c);
            return SLDG_OK;
        }
    }
    // v_a v_b v_c in the physical regime |shift| < 1: TMA-tile staged kernel
    if (c->use_tma && c->tune.tile_triple && k1 >= c->dx && mid12 == 1 && mid23 == 1 && n1 % 4 == 0 && n2 % 4 == 0 &&
        n3 >= 4 && inner1 < (1L << 31)) {
        // variants (columns W, owned k2-cells C2, ring depth NS, resident blocks, drifting warps):
        // SLDG_VTRIPLE_VARIANT picks one for A/B runs
        auto launch = [&](auto kern, int W, int C2, int NS) -> int {
            const long blocks = (inner1 / W) * (n1 / 4) * (n2 / C2) * outer3;
            if (inner1 % W || n2 % C2 || (W * sizeof(T)) % 16 || blocks >= (1L << 31)) return 1;          // not applicable
            sldg_ctx::TmapSlot &ts = c->tmap5[c->cur];
            if (!ts.valid || ts.p0 != W) {
                ts.valid = make_tensor_map_5d(&ts.map, in, sizeof(T) == 8, (uint64_t)inner1, (uint64_t)n1 * O,
                                              (uint64_t)n2 * O, (uint64_t)n3 * O, (uint64_t)outer3, W, O, O, O);
                ts.p0 = W;
            }
            if (!ts.valid) return 1;
            const size_t smem = (size_t)NS * 6 * (C2 + 2) * O * O * O * W * sizeof(T);
            if (ensure_smem(c, kern, smem) != cudaSuccess) { cudaGetLastError(); return 1; }
            kern<<<(unsigned)blocks, W * 4 * C2, smem, c->stream>>>(
                ts.map, in, out, inner1, n1, n2, n3, outer3, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
            return 0;
        };
        // two k2-cells per thread (sweep_vtriple_tile2_kernel): threads = W x 4 x C2 / 2, the windows' first cells parked
        auto launch2 = [&](auto kern, int W, int C2, int NS) -> int {
            const long blocks = (inner1 / W) * (n1 / 4) * (n2 / C2) * outer3;
            if (inner1 % W || n2 % C2 || (W * sizeof(T)) % 16 || blocks >= (1L << 31)) return 1;
            sldg_ctx::TmapSlot &ts = c->tmap5[c->cur];
            if (!ts.valid || ts.p0 != W) {
                ts.valid = make_tensor_map_5d(&ts.map, in, sizeof(T) == 8, (uint64_t)inner1, (uint64_t)n1 * O,
                                              (uint64_t)n2 * O, (uint64_t)n3 * O, (uint64_t)outer3, W, O, O, O);
                ts.p0 = W;
            }
            if (!ts.valid) return 1;
            const int thr = W * 2 * C2;
            const size_t smem = (size_t)NS * 6 * (C2 + 2) * O * O * O * W * sizeof(T) + (size_t)2 * O * O * O * thr * sizeof(T);
            if (smem > 226 * 1024 || ensure_smem(c, kern, smem) != cudaSuccess) { cudaGetLastError(); return 1; }
            kern<<<(unsigned)blocks, thr, smem, c->stream>>>(
                ts.map, in, out, inner1, n1, n2, n3, outer3, mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1],
                (const T *)ab[1], cnt2, qd[1], qm[1], mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
            return 0;
        };
        int rc = 1;
        switch (c->tune.vt_variant) {
        case 12: rc = launch2(sweep_vtriple_tile2_kernel<T, O, 32, 2, 2, 2>, 32, 2, 2); break;
        case 13: rc = launch2(sweep_vtriple_tile2_kernel<T, O, 32, 4, 2, 1>, 32, 4, 2); break;
        // kept for A/B runs (DESIGN.md section 5 lists what the others measured): 0 = round-1 geometry (one block of
        // 4 x 4 cells), 1 = the same with per-warp slot release and a 3-deep ring, 2 = fp64 default, 10 = fp32 default
        case 0: rc = launch(sweep_vtriple_tile_kernel<T, O, 32, 4, 2, 1, false>, 32, 4, 2); break;
        case 1: rc = launch(sweep_vtriple_tile_kernel<T, O, 32, 4, 3, 1, true>, 32, 4, 3); break;
        case 2: rc = launch(sweep_vtriple_tile_kernel<T, O, 32, 2, 2, 2, false>, 32, 2, 2); break;
        case 10: rc = launch(sweep_vtriple_tile_kernel<T, O, 64, 1, 2, 2, false>, 64, 1, 2); break;
        default:
            // two k2-cells per thread, two resident blocks of 4 x 2 cells: fp64 13.6 -> 12.6 ms at config 5 (32 columns),
            // fp32 8.35 -> 6.7 ms (64 columns keep the rows at 256 bytes); then the one-cell geometries
            if constexpr (sizeof(T) == 4) rc = launch2(sweep_vtriple_tile2_kernel<T, O, 64, 2, 2, 2>, 64, 2, 2);
            if (rc) rc = launch2(sweep_vtriple_tile2_kernel<T, O, 32, 2, 2, 2>, 32, 2, 2);
            if (rc) rc = launch(sweep_vtriple_tile_kernel<T, O, 32, 2, 2, 2, false>, 32, 2, 2);
            break;
        }
        if (rc == 0) {
            LAUNCH_CHECK(c);
            c->cur ^= 1;
            f_changed(c);
            return SLDG_OK;
        }
    }
    int chunk = 32;
    while (inner1 % chunk) chunk /= 2;
    long threads = inner1 * n1 * mid12 * n2 * mid23 * outer3;
    if (O % 2 == 0 && inner1 == 1)
        sweep_triple_kernel<T, O, (O % 2 == 0)><<<(unsigned)cdiv(threads, 128), 128, 0, c->stream>>>(
            in, out, inner1, n1, mid12, n2, mid23, n3, outer3, chunk,
            mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1], (const T *)ab[1], cnt2, qd[1], qm[1],
            mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
    else
        sweep_triple_kernel<T, O, false><<<(unsigned)cdiv(threads, 128), 128, 0, c->stream>>>(
            in, out, inner1, n1, mid12, n2, mid23, n3, outer3, chunk,
            mm[0], (const T *)ab[0], cnt1, qd[0], qm[0], mm[1], (const T *)ab[1], cnt2, qd[1], qm[1],
            mm[2], (const T *)ab[2], cnt3, qd[2], qm[2]);
    LAUNCH_CHECK(c);
    c->cur ^= 1;
    f_changed(c);
    return SLDG_OK;
}

int run_triple(sldg_ctx *c, int k1, int k2, int k3, long c1, long c2, long c3) {
    if (c->dtype == SLDG_F64) {
        if (c->o == 1) return run_triple_t<double, 1>(c, k1, k2, k3, c1, c2, c3);
        if (c->o == 2) return run_triple_t<double, 2>(c, k1, k2, k3, c1, c2, c3);
    } else {
        if (c->o == 1) return run_triple_t<float, 1>(c, k1, k2, k3, c1, c2, c3);
        if (c->o == 2) return run_triple_t<float, 2>(c, k1, k2, k3, c1, c2, c3);
    }
    return fail(c, SLDG_ERR_UNSUPPORTED, "fused triple is instantiated for order <= 2 (got %d)", c->o);
}

// point table slot 1 or 2 at a storage set; `assembled` = its m/ab are already valid
void use_tab(sldg_ctx *c, int slot, sldg_ctx::Tab &t, bool assembled) {
    if (slot == 1) { c->d_sigma = t.sigma; c->d_m = t.m; c->d_ab = t.ab; c->skip_asm1 = assembled; }
    else if (slot == 2) { c->d_sigma2 = t.sigma; c->d_m2 = t.m; c->d_ab2 = t.ab; c->skip_asm2 = assembled; }
    else { c->d_sigma3 = t.sigma; c->d_m3 = t.m; c->d_ab3 = t.ab; c->skip_asm3 = assembled; }
}

long sweep_count(const sldg_ctx *c, int dim) { return dim < c->dx ? c->N[c->dx + dim] : c->X; }

}  // namespace

extern "C" int sldg_translate(sldg_ctx *c, int dim, const double *shift, size_t count) {
    if (!c || !shift || dim < 0 || dim >= c->D) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if ((long)count != sweep_count(c, dim))
        return fail(c, SLDG_ERR_ARG, "sldg_translate: dim %d needs %ld shifts, got %zu", dim, sweep_count(c, dim), count);
    use_tab(c, 1, c->gen[0], false);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma, shift, count * sizeof(double), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));   // the host array may be reused by the caller
    return run_sweep(c, dim, (long)count);
}

extern "C" int sldg_translate_dev(sldg_ctx *c, int dim, const double *shift, size_t count) {
    if (!c || !shift || dim < 0 || dim >= c->D) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if ((long)count != sweep_count(c, dim))
        return fail(c, SLDG_ERR_ARG, "sldg_translate_dev: dim %d needs %ld shifts, got %zu", dim, sweep_count(c, dim), count);
    use_tab(c, 1, c->gen[0], false);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma, shift, count * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    return run_sweep(c, dim, (long)count);
}

namespace {
// Table of a physics sweep (D:O3, D:R4) into slot 1 or 2: fills sigma on the stream unless the
// cached x-table for this tau is still valid.
int physics_tab(sldg_ctx *c, int slot, int dim, double dt) {
    long count = sweep_count(c, dim);
    int block = 256;
    if (dim < c->dx) {
        sldg_ctx::Tab &t = c->xt[dim];
        if (t.valid && t.tau == dt) { use_tab(c, slot, t, true); return SLDG_OK; }
        use_tab(c, slot, t, false);
        int va = c->dx + dim;
        // the table is being rewritten: not valid until the sweep that assembles it has been enqueued
        // successfully (commit_tables); a failure in between leaves it invalid, never half-written-but-trusted
        t.valid = false;
        t.pending = true;
        t.pending_tau = dt;
        c->xt_epoch++;                  // graphs captured against the old table must not be replayed
        sigma_from_coords_kernel<<<(unsigned)cdiv(count, block), block, 0, c->stream>>>(
            c->d_coords[va], count, dt, c->h[dim], t.sigma);
    } else {
        int a = dim - c->dx;
        if (a >= c->dx) return fail(c, SLDG_ERR_ARG, "sldg_advect: v_%d has no field component (dx = %d)", a + 1, c->dx);
        if (!c->have_E) return fail(c, SLDG_ERR_STATE, "sldg_advect: no E stored (call sldg_poisson_E or sldg_set_E)");
        sldg_ctx::Tab &t = c->gen[slot - 1];
        use_tab(c, slot, t, false);
        sigma_from_E_kernel<<<(unsigned)cdiv(count, block), block, 0, c->stream>>>(
            c->d_E + (long)a * c->X, count, dt, c->h[dim], t.sigma);
    }
    LAUNCH_CHECK(c);
    return SLDG_OK;
}

// after the sweep(s) that assemble the pending cached x-tables were enqueued: rc == 0 makes them valid
int commit_tables(sldg_ctx *c, int rc) {
    for (auto &t : c->xt)
        if (t.pending) {
            t.pending = false;
            if (rc == SLDG_OK) { t.valid = true; t.tau = t.pending_tau; }
        }
    return rc;
}

bool pair_ok(const sldg_ctx *c, int d1, int d2) {
    if (d1 < 0 || d2 <= d1 || d2 >= c->D) return false;
    return (d2 < c->dx) || (d1 >= c->dx);          // both x-dimensions or both v-dimensions
}
}  // namespace

extern "C" int sldg_advect(sldg_ctx *c, int dim, double dt) {
    if (!c || dim < 0 || dim >= c->D) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int rc = physics_tab(c, 1, dim, dt);
    if (rc) return commit_tables(c, rc);
    return commit_tables(c, run_sweep(c, dim, sweep_count(c, dim)));
}

extern "C" int sldg_advect_pair(sldg_ctx *c, int dim1, int dim2, double dt) {
    if (!c) return SLDG_ERR_ARG;
    if (!pair_ok(c, dim1, dim2))
        return fail(c, SLDG_ERR_ARG, "sldg_advect_pair: need dim1 < dim2, both x- or both v-dimensions");
    if (c->o > 4) {                      // the fused kernel is instantiated for o <= 4 (registers)
        int r1 = sldg_advect(c, dim1, dt);
        return r1 ? r1 : sldg_advect(c, dim2, dt);
    }
    DeviceGuard guard(c);
    int rc = physics_tab(c, 1, dim1, dt);
    if (rc) return commit_tables(c, rc);
    if ((rc = physics_tab(c, 2, dim2, dt))) return commit_tables(c, rc);
    return commit_tables(c, run_pair(c, dim1, dim2, sweep_count(c, dim1), sweep_count(c, dim2)));
}

namespace {
// Raw fused calls along v-dimensions with arbitrary caller shifts: the fused v-kernels are built for the physical
// regime |shift| < 1 cell (offsets 0 or n-1); with wider shifts neighbouring lanes read cells far apart and the
// register kernels lose coalescing (measured 70 ms against 2 x 14 ms for a config-4 pair).  The tables are
// assembled first, with a flag raised by any wider shift; the flag is read back (these raw calls synchronise,
// like sldg_translate with host shifts) and such a call runs as single TMA sweeps, which do not care.
int assemble_with_flag(sldg_ctx *c, const int *dims, const size_t *counts, int nd, bool *wide) {
    CUDA_TRY(c, cudaMemsetAsync(c->d_wide, 0, sizeof(int), c->stream));
    for (int i = 0; i < nd; ++i) {
        sldg_ctx::Tab &t = c->gen[i];
        const int block = 128;
        const int O = c->o;
        const size_t sh = (size_t)2 * O * O * 2 * O * 2 * sizeof(double);
        if (c->dtype == SLDG_F64)
            assemble_ab_kernel<double><<<(unsigned)cdiv((long)counts[i], block), block, sh, c->stream>>>(
                t.sigma, (long)counts[i], O, c->cells[dims[i]], c->d_coef, t.m, (double *)t.ab, c->d_wide);
        else
            assemble_ab_kernel<float><<<(unsigned)cdiv((long)counts[i], block), block, sh, c->stream>>>(
                t.sigma, (long)counts[i], O, c->cells[dims[i]], c->d_coef, t.m, (float *)t.ab, c->d_wide);
        LAUNCH_CHECK(c);
    }
    int h = 0;
    CUDA_TRY(c, cudaMemcpyAsync(&h, c->d_wide, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    *wide = h != 0;
    return SLDG_OK;
}
int singles_from_tables(sldg_ctx *c, const int *dims, const size_t *counts, int nd) {
    for (int i = 0; i < nd; ++i) {
        use_tab(c, 1, c->gen[i], true);
        int rc = run_sweep(c, dims[i], (long)counts[i]);
        if (rc) return rc;
    }
    return SLDG_OK;
}
}  // namespace

extern "C" int sldg_translate_pair_dev(sldg_ctx *c, int dim1, const double *shift1, size_t count1, int dim2,
                                       const double *shift2, size_t count2) {
    if (!c || !shift1 || !shift2) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if (!pair_ok(c, dim1, dim2))
        return fail(c, SLDG_ERR_ARG, "sldg_translate_pair_dev: need dim1 < dim2, both x- or both v-dimensions");
    if ((long)count1 != sweep_count(c, dim1) || (long)count2 != sweep_count(c, dim2))
        return fail(c, SLDG_ERR_ARG, "sldg_translate_pair_dev: wrong shift counts");
    if (c->o > 4) {
        int r1 = sldg_translate_dev(c, dim1, shift1, count1);
        return r1 ? r1 : sldg_translate_dev(c, dim2, shift2, count2);
    }
    use_tab(c, 1, c->gen[0], false);
    use_tab(c, 2, c->gen[1], false);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma, shift1, count1 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma2, shift2, count2 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    // v-pair: asynchronous by default (a line shifted by a cell or more takes the fused kernel's per-block
    // fallback: same bits, more traffic); with SLDG_ROUTE_WIDE=1 the call reads back whether any line is that
    // wide (stream synchronisation) and runs such a call as two single sweeps
    if (dim1 >= c->dx && c->tune.route_wide) {
        const int dims[2] = {dim1, dim2};
        const size_t counts[2] = {count1, count2};
        bool wide = false;
        int rc = assemble_with_flag(c, dims, counts, 2, &wide);
        if (rc) return rc;
        if (wide) return singles_from_tables(c, dims, counts, 2);
        use_tab(c, 1, c->gen[0], true);
        use_tab(c, 2, c->gen[1], true);
    }
    return run_pair(c, dim1, dim2, (long)count1, (long)count2);
}

// ------------------------------------------------------------------------------------------
// a-3 rho, a-4 Poisson, a-5 step, a-6 diagnostics
// ------------------------------------------------------------------------------------------
namespace {

int run_poisson_fwd(sldg_ctx *c);

// v-split geometry shared by the rho pass and the one-read invariants pass
struct VSplit { int vec; long vps; int splits; bool small; };
template <typename T>
VSplit vsplit(const sldg_ctx *c, int blocks_per_sm) {
    constexpr int VMAX = 16 / (int)sizeof(T);
    VSplit g;
    g.vec = (c->X % VMAX == 0) ? VMAX : ((c->X % 2 == 0) ? 2 : 1);
    long target = (long)c->sm_count * 2048 * 6;
    long s = cdiv(target, c->X / g.vec > 0 ? c->X / g.vec : 1);
    if (s > c->max_splits) s = c->max_splits;
    if (s < 1) s = 1;
    // Small problems (the 1+1 D configs): one split, every x sums its v-nodes alone -- with a
    // compensated accumulator, so that rho is the exactly summed value rounded once (D:O4).  rho + 1
    // is a difference of O(1) sums (D:R11): a plain running sum is visible at 1e-13 relative in E
    // when the perturbation is 1e-3.  Large problems need the splits for parallelism; their partials
    // are short sums and the pass over the splits is compensated.
    g.small = c->V * c->X <= (1L << 23);
    if (g.small) { s = 1; g.vec = 1; }
    else {
        // whole waves only: blocks = (blocks along x) * splits just under a multiple of the resident-block count
        const long bx = cdiv(c->X / g.vec, 128), slots = (long)c->sm_count * blocks_per_sm;
        const long k = bx * s / slots;
        if (k >= 1 && k * slots / bx >= 1) s = k * slots / bx;
    }
    g.vps = cdiv(c->V, s);
    g.splits = (int)cdiv(c->V, g.vps);
    return g;
}

template <typename T, int VEC, int UB, bool COMP = false>
void launch_vsum(sldg_ctx *c, int splits, long vps, int block) {
    long xv = c->X / VEC;
    if (xv < block) block = (int)(cdiv(xv, 32) * 32);
    dim3 grid((unsigned)cdiv(xv, block), (unsigned)splits);
    vsum_partial_kernel<T, VEC, UB, COMP><<<grid, block, 0, c->stream>>>(
        (const T *)c->buf[c->cur], c->X, c->V, vps, c->d_Wv, c->d_part);
}

// pass over the splits: rho (and s2 when the partials come from the invariants pass)
int finish_vsum(sldg_ctx *c, int splits, double *rho_copy, bool with_s2) {
    int block = 256;
    vsum_final_kernel<<<(unsigned)cdiv(c->X * 32, block), block, 0, c->stream>>>(
        c->d_part, with_s2 ? c->d_part + (size_t)c->max_splits * c->X : nullptr, c->X, splits, c->d_rho,
        rho_copy, with_s2 ? c->d_s2 : nullptr);
    LAUNCH_CHECK(c);
    c->have_rho = true;
    return SLDG_OK;
}

// a-3: rho only (the Strang step)
template <typename T>
int run_vsum(sldg_ctx *c, double *rho_copy) {
    constexpr int VMAX = 16 / (int)sizeof(T);
    const VSplit g = vsplit<T>(c, 16);
    c->have_inv = false;                                   // d_part is overwritten
    if (g.small) launch_vsum<T, 1, 32, true>(c, g.splits, g.vps, 32);     // thread per x, 32 rows in flight
    else if (g.vec == VMAX) launch_vsum<T, VMAX, 8>(c, g.splits, g.vps, 128);
    else if (g.vec == 2) launch_vsum<T, 2, 8>(c, g.splits, g.vps, 128);
    else launch_vsum<T, 1, 8>(c, g.splits, g.vps, 128);
    LAUNCH_CHECK(c);
    return finish_vsum(c, g.splits, rho_copy, false);
}

int run_rho(sldg_ctx *c, double *rho_copy) {
    return c->dtype == SLDG_F64 ? run_vsum<double>(c, rho_copy) : run_vsum<float>(c, rho_copy);
}

// a-6 + NEXT-4: ONE read of the current f leaves the partials of rho, f^2, v_a f and |v|^2 f in d_part
// (vall_partial_kernel) and rho, s2 in d_rho, d_s2; remembered until f changes, so that
// sldg_diagnostics followed by sldg_moments (or sldg_invariants) reads f once.
template <typename T, int VEC, int DV, int UB, bool COMP, int BLK>
void launch_vall(sldg_ctx *c, int splits, long vps) {
    long xv = c->X / VEC;
    dim3 grid((unsigned)cdiv(xv, BLK), (unsigned)splits);
    vall_partial_kernel<T, VEC, DV, UB, COMP, BLK><<<grid, BLK, 0, c->stream>>>(
        (const T *)c->buf[c->cur], c->X, c->V, vps, (long)c->max_splits * c->X, c->d_Wv, c->d_va, c->d_v2,
        c->d_part);
}
template <typename T, int DV>
int run_vall_dv(sldg_ctx *c) {
    constexpr int VMAX = 16 / (int)sizeof(T);
    const VSplit g = vsplit<T>(c, 8);
    if (g.small) launch_vall<T, 1, DV, 16, true, 32>(c, g.splits, g.vps);
    else if (g.vec == VMAX) launch_vall<T, VMAX, DV, 16, false, 128>(c, g.splits, g.vps);
    else if (g.vec == 2) launch_vall<T, 2, DV, 8, false, 128>(c, g.splits, g.vps);
    else launch_vall<T, 1, DV, 8, false, 128>(c, g.splits, g.vps);
    LAUNCH_CHECK(c);
    int rc = finish_vsum(c, g.splits, nullptr, true);
    if (rc) return rc;
    // momentum and |v|^2 moment: sum over splits and x of partials 2 .. 2+dv -> d_scal[3 .. 3+dv]
    {
        const int nk = c->dv + 1, block = 256;
        vrows_final_kernel<<<(unsigned)cdiv((long)nk * c->X * 32, block), block, 0, c->stream>>>(
            c->d_part + (size_t)2 * c->max_splits * c->X, c->X, g.splits, c->max_splits, nk, c->d_mom);
        LAUNCH_CHECK(c);
        moments_final_kernel<<<1, 1024, 0, c->stream>>>(c->d_mom, c->d_Wx, c->X, nk, c->d_scal + 3);
        LAUNCH_CHECK(c);
    }
    c->have_inv = true;
    return SLDG_OK;
}
template <typename T>
int run_vall_t(sldg_ctx *c) {
    if (c->dv == 1) return run_vall_dv<T, 1>(c);
    if (c->dv == 2) return run_vall_dv<T, 2>(c);
    return run_vall_dv<T, 3>(c);
}
// all invariants of the current f into d_scal[0 .. 3+dv] (no read of f when they are already there)
int run_invariants(sldg_ctx *c) {
    int rc;
    if (!c->have_inv) {
        rc = c->dtype == SLDG_F64 ? run_vall_t<double>(c) : run_vall_t<float>(c);
        if (rc) return rc;
        if ((rc = run_poisson_fwd(c))) return rc;
        scalars_kernel<<<1, 1024, 0, c->stream>>>(c->d_rho, c->d_s2, c->d_E, c->d_Wx, c->X, c->dx, c->d_scal);
        LAUNCH_CHECK(c);
    }
    return SLDG_OK;
}

// apply M (rows x cols) along dimension b of a complex tensor with extents shape[] (index 0 fastest)
template <bool IN_REAL, bool OUT_REAL>
int apply_along(sldg_ctx *c, const double *in_re, const double *in_im, long *shape, int nd, int b,
                const double2 *M, long rows, double *out_re, double *out_im) {
    long inner = 1, outer = 1, cols = shape[b];
    for (int d = 0; d < b; ++d) inner *= shape[d];
    for (int d = b + 1; d < nd; ++d) outer *= shape[d];
    long total = outer * rows * inner;             // one warp per output element
    int block = 256;
    cplx_apply_kernel<IN_REAL, OUT_REAL><<<(unsigned)cdiv(total * 32, block), block, 0, c->stream>>>(
        in_re, in_im, outer, cols, inner, M, rows, out_re, out_im);
    LAUNCH_CHECK(c);
    shape[b] = rows;
    return SLDG_OK;
}

int run_poisson(sldg_ctx *c, double *E_copy) {
    const double PI = 3.14159265358979323846264338327950288;
    const int dx = c->dx;
    long shape[3] = {1, 1, 1};
    for (int a = 0; a < dx; ++a) shape[a] = c->N[a];
    // forward transform of rho + 1, one dimension at a time
    const double *ir = c->d_rho, *ii = nullptr;
    int rc;
    for (int a = 0; a < dx; ++a) {
        double *orr = (a == dx - 1) ? c->d_gh[0] : c->d_t[(a & 1) * 2];
        double *oi = (a == dx - 1) ? c->d_gh[1] : c->d_t[(a & 1) * 2 + 1];
        if (a == 0) rc = apply_along<true, false>(c, ir, ii, shape, dx, a, c->d_F[a], c->K[a], orr, oi);
        else rc = apply_along<false, false>(c, ir, ii, shape, dx, a, c->d_F[a], c->K[a], orr, oi);
        if (rc) return rc;
        ir = orr; ii = oi;
    }
    double kf[3] = {0, 0, 0};
    for (int a = 0; a < dx; ++a) kf[a] = 2.0 * PI / (c->hi[a] - c->lo[a]);
    for (int a = 0; a < dx; ++a) {
        int block = 128;
        poisson_scale_kernel<<<(unsigned)cdiv(c->KK, block), block, 0, c->stream>>>(
            c->d_gh[0], c->d_gh[1], c->KK, dx, a, c->K[0], c->K[1], c->K[2], c->Mmax[0], c->Mmax[1],
            c->Mmax[2], kf[0], kf[1], kf[2], c->d_t[0], c->d_t[1]);
        LAUNCH_CHECK(c);
        for (int b = 0; b < dx; ++b) shape[b] = c->K[b];
        const double *sr = c->d_t[0], *si = c->d_t[1];
        for (int b = 0; b < dx; ++b) {
            bool last = (b == dx - 1);
            double *orr = last ? c->d_E + (long)a * c->X : c->d_t[((b + 1) & 1) * 2];
            double *oi = last ? nullptr : c->d_t[((b + 1) & 1) * 2 + 1];
            if (last) rc = apply_along<false, true>(c, sr, si, shape, dx, b, c->d_G[b], c->N[b], orr, oi);
            else rc = apply_along<false, false>(c, sr, si, shape, dx, b, c->d_G[b], c->N[b], orr, oi);
            if (rc) return rc;
            sr = orr; si = oi;
        }
    }
    c->have_E = true;
    if (E_copy)
        CUDA_TRY(c, cudaMemcpyAsync(E_copy, c->d_E, (size_t)dx * c->X * sizeof(double),
                                    cudaMemcpyDeviceToDevice, c->stream));
    return SLDG_OK;
}

int run_poisson_fwd(sldg_ctx *c) { return run_poisson(c, nullptr); }

}  // namespace

extern "C" int sldg_wide_shift_seen(sldg_ctx *c, int *seen, int reset) {
    if (!c || !seen) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int h = 0;
    CUDA_TRY(c, cudaMemcpyAsync(&h, c->d_wide_seen, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    if (reset) CUDA_TRY(c, cudaMemsetAsync(c->d_wide_seen, 0, sizeof(int), c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    *seen = h != 0;
    return SLDG_OK;
}

extern "C" int sldg_compute_rho(sldg_ctx *c, double *rho_out) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    return run_rho(c, rho_out);
}

extern "C" int sldg_poisson_E(sldg_ctx *c, double *E_out) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if (!c->have_rho) return fail(c, SLDG_ERR_STATE, "sldg_poisson_E: rho of the current f not computed");
    return run_poisson(c, E_out);
}

extern "C" int sldg_set_E(sldg_ctx *c, const double *E, int is_device) {
    if (!c || !E) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_E, E, (size_t)c->dx * c->X * sizeof(double),
                                is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, c->stream));
    if (!is_device) CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->have_E = true;
    c->have_inv = false;               // the remembered electric energy belonged to the E just overwritten
    return SLDG_OK;
}

extern "C" int sldg_advect_triple(sldg_ctx *c, int dim1, int dim2, int dim3, double dt) {
    if (!c) return SLDG_ERR_ARG;
    if (!pair_ok(c, dim1, dim2) || !pair_ok(c, dim2, dim3) || !pair_ok(c, dim1, dim3))
        return fail(c, SLDG_ERR_ARG, "sldg_advect_triple: need dim1 < dim2 < dim3, all x- or all v-dimensions");
    if (c->o > 2) {                      // the triple kernel is instantiated for o <= 2 (registers)
        int r = sldg_advect_pair(c, dim1, dim2, dt);
        return r ? r : sldg_advect(c, dim3, dt);
    }
    DeviceGuard guard(c);
    int rc;
    if ((rc = physics_tab(c, 1, dim1, dt))) return commit_tables(c, rc);
    if ((rc = physics_tab(c, 2, dim2, dt))) return commit_tables(c, rc);
    if ((rc = physics_tab(c, 3, dim3, dt))) return commit_tables(c, rc);
    return commit_tables(c, run_triple(c, dim1, dim2, dim3, sweep_count(c, dim1), sweep_count(c, dim2), sweep_count(c, dim3)));
}

extern "C" int sldg_translate_triple_dev(sldg_ctx *c, int dim1, const double *shift1, size_t count1, int dim2,
                                         const double *shift2, size_t count2, int dim3, const double *shift3,
                                         size_t count3) {
    if (!c || !shift1 || !shift2 || !shift3) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if (!pair_ok(c, dim1, dim2) || !pair_ok(c, dim2, dim3) || !pair_ok(c, dim1, dim3))
        return fail(c, SLDG_ERR_ARG, "sldg_translate_triple_dev: need dim1 < dim2 < dim3, all x- or all v-dimensions");
    if ((long)count1 != sweep_count(c, dim1) || (long)count2 != sweep_count(c, dim2) ||
        (long)count3 != sweep_count(c, dim3))
        return fail(c, SLDG_ERR_ARG, "sldg_translate_triple_dev: wrong shift counts");
    if (c->o > 2) {
        int r = sldg_translate_pair_dev(c, dim1, shift1, count1, dim2, shift2, count2);
        return r ? r : sldg_translate_dev(c, dim3, shift3, count3);
    }
    use_tab(c, 1, c->gen[0], false);
    use_tab(c, 2, c->gen[1], false);
    use_tab(c, 3, c->gen[2], false);
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma, shift1, count1 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma2, shift2, count2 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    CUDA_TRY(c, cudaMemcpyAsync(c->d_sigma3, shift3, count3 * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    if (dim1 >= c->dx && c->tune.route_wide) {   // v-triple: as the v-pair (three single sweeps when wide)
        const int dims[3] = {dim1, dim2, dim3};
        const size_t counts[3] = {count1, count2, count3};
        bool wide = false;
        int rc = assemble_with_flag(c, dims, counts, 3, &wide);
        if (rc) return rc;
        if (wide) return singles_from_tables(c, dims, counts, 3);
        use_tab(c, 1, c->gen[0], true);
        use_tab(c, 2, c->gen[1], true);
        use_tab(c, 3, c->gen[2], true);
    }
    return run_triple(c, dim1, dim2, dim3, (long)count1, (long)count2, (long)count3);
}

namespace {
// sweeps along dimensions base .. base+cnt-1 with increment tau, fusing the first two when allowed;
// with_rho: the fused kernel that performs the WHOLE group may also leave the rho partials (c->rho_rows)
int advect_group(sldg_ctx *c, int base, int cnt, double tau, bool with_rho = false, bool twice = false) {
    int rc, a = 0;
    c->rho_rows = 0;
    const bool whole = c->use_fuse && ((cnt == 3 && c->o <= 2) || (cnt == 2 && c->o <= 4));
    c->want_rho = with_rho && whole && c->tune.fuse_rho && base == 0;
    // twice: only a kernel that performs the WHOLE group may apply it twice in its pass (c->twice_done tells)
    c->twice_req = twice && base == 0 && c->tune.twice && (whole || cnt == 1) && (cnt < 3 || c->tune.twice_triple);
    c->twice_done = false;
    struct Clear { sldg_ctx *c; ~Clear() { c->want_rho = false; c->twice_req = false; } } clear{c};
    if (c->use_fuse && cnt == 3 && c->o <= 2) return sldg_advect_triple(c, base, base + 1, base + 2, tau);
    if (c->use_fuse && cnt >= 2) {
        if ((rc = sldg_advect_pair(c, base, base + 1, tau))) return rc;
        a = 2;
    }
    for (; a < cnt; ++a) if ((rc = sldg_advect(c, base + a, tau))) return rc;
    return SLDG_OK;
}
}  // namespace

namespace {
// x-group with increment tau, then rho of the result: one pass when the fused kernels apply (NEXT-1)
int advect_x_rho(sldg_ctx *c, double tau, double *rho_copy) {
    int rc = advect_group(c, 0, c->dx, tau, true);
    if (rc) return rc;
    if (c->rho_rows > 0) {
        const int rows = c->rho_rows;
        c->rho_rows = 0;
        return finish_vsum(c, rows, rho_copy, false);
    }
    return run_rho(c, rho_copy);
}

// the x-group applied twice with increment tau: one pass when a kernel takes the whole group (plane kernels,
// bulk x_1 kernel), else the group twice; bit-identical either way
int advect_x_twice(sldg_ctx *c, double tau) {
    int rc = advect_group(c, 0, c->dx, tau, false, true);
    if (rc) return rc;
    if (c->twice_done) { c->twice_done = false; return SLDG_OK; }
    return advect_group(c, 0, c->dx, tau);
}

int step_body(sldg_ctx *c, double dt) {
    int rc;
    if ((rc = advect_x_rho(c, 0.5 * dt, nullptr))) return rc;
    if ((rc = run_poisson(c, nullptr))) return rc;
    if ((rc = advect_group(c, c->dx, c->dx, dt))) return rc;
    if ((rc = advect_group(c, 0, c->dx, 0.5 * dt))) return rc;
    return SLDG_OK;
}

// Capture one step (starting from the current buffer parity) into an executable graph.  Nothing runs
// during the capture; the context's bookkeeping advances exactly as in an eager step.
int capture_step(sldg_ctx *c, double dt, sldg_ctx::StepGraph &g) {
    if (!c->capture_stream)
        CUDA_TRY(c, cudaStreamCreateWithFlags(&c->capture_stream, cudaStreamNonBlocking));
    if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    cudaStream_t user = c->stream;
    // nothing executes during a capture: on ANY failure the bookkeeping below is put back, so that the
    // caller can run the step eagerly from exactly the state it had
    const int cur_in = c->cur;
    const unsigned long long l0 = c->launches;
    const bool rho_in = c->have_rho, E_in = c->have_E;
    const bool inv_in = c->have_inv;
    auto restore = [&]() { c->cur = cur_in; c->launches = l0; c->have_rho = rho_in; c->have_E = E_in; c->have_inv = inv_in; };
    CUDA_TRY(c, cudaStreamBeginCapture(c->capture_stream, cudaStreamCaptureModeThreadLocal));
    c->stream = c->capture_stream;
    int rc = step_body(c, dt);
    c->stream = user;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->capture_stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); restore(); return rc; }
    if (e != cudaSuccess) { restore(); return fail(c, SLDG_ERR_CUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e)); }
    e = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) {
        g.exec = nullptr;
        restore();
        return fail(c, SLDG_ERR_CUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
    }
    g.dt = dt; g.cur_in = cur_in; g.cur_out = c->cur; g.launches = c->launches - l0;
    g.xt_epoch = c->xt_epoch;
    return SLDG_OK;
}
}  // namespace

extern "C" int sldg_advect_x_twice(sldg_ctx *c, double tau) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    return advect_x_twice(c, tau);
}

extern "C" int sldg_step_n(sldg_ctx *c, double dt, int nsteps) {
    if (!c || nsteps < 0) return SLDG_ERR_ARG;
    if (nsteps == 0) return SLDG_OK;
    // launch-bound problems replay the CUDA graph of one step; merging is for the bandwidth-bound ones, and only
    // where one kernel applies the whole x-group twice (else it would be the same passes as sldg_step)
    const bool one_pass = c->dx == 1 || (c->use_fuse && c->dx == 2 && c->o <= 3) ||
                          (c->use_fuse && c->dx == 3 && c->o <= 2 && c->tune.twice_triple);
    if (c->use_graph || nsteps == 1 || !c->tune.twice || !one_pass) {
        for (int s = 0; s < nsteps; ++s) {
            int rc = sldg_step(c, dt);
            if (rc) return rc;
        }
        return SLDG_OK;
    }
    DeviceGuard guard(c);
    int rc;
    if ((rc = advect_x_rho(c, 0.5 * dt, nullptr))) return rc;
    for (int s = 0; s < nsteps; ++s) {
        if ((rc = run_poisson(c, nullptr))) return rc;
        if ((rc = advect_group(c, c->dx, c->dx, dt))) return rc;
        if (s + 1 < nsteps) {
            // the last x half-step of this step and the first of the next: x(dt/2) x(dt/2) in one pass, then rho
            if ((rc = advect_x_twice(c, 0.5 * dt))) return rc;
            if ((rc = run_rho(c, nullptr))) return rc;
        } else {
            if ((rc = advect_group(c, 0, c->dx, 0.5 * dt))) return rc;
        }
    }
    return SLDG_OK;
}

extern "C" int sldg_advect_x_rho(sldg_ctx *c, double tau, double *rho_out) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    return advect_x_rho(c, tau, rho_out);
}

extern "C" int sldg_step(sldg_ctx *c, double dt) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    if (!c->use_graph) return step_body(c, dt);
    const int p = c->cur;
    sldg_ctx::StepGraph &g = c->graphs[p];
    if (g.exec && g.dt == dt && g.cur_in == p && g.xt_epoch == c->xt_epoch) {   // replay
        CUDA_TRY(c, cudaGraphLaunch(g.exec, c->stream));
        c->cur = g.cur_out; c->launches += g.launches;
        f_changed(c); c->have_E = true;
        return SLDG_OK;
    }
    if (c->eager_seen[p] && c->last_eager_dt[p] == dt && c->eager_epoch[p] == c->xt_epoch) {
        // second step with this (dt, parity) and untouched x-tables: capture (no table kernels inside)
        int rc = capture_step(c, dt, g);
        if (rc == SLDG_OK) {
            CUDA_TRY(c, cudaGraphLaunch(g.exec, c->stream));
            return SLDG_OK;
        }
        // capture or instantiation failed (state restored): graphs off for this context, step eagerly
        cudaGetLastError();
        c->use_graph = false;
        return step_body(c, dt);
    }
    // first step with this (dt, parity): eager (it also fills the cached x-tables and kernel attributes)
    c->eager_seen[p] = true;
    c->last_eager_dt[p] = dt;
    int rc = step_body(c, dt);
    c->eager_epoch[p] = c->xt_epoch;
    return rc;
}

extern "C" int sldg_moments(sldg_ctx *c, double *momentum, double *kinetic) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int rc = run_invariants(c);
    if (rc) return rc;
    double h[4];
    CUDA_TRY(c, cudaMemcpyAsync(h, c->d_scal + 3, (c->dv + 1) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (momentum) for (int a = 0; a < c->dv; ++a) momentum[a] = h[a];
    if (kinetic) *kinetic = 0.5 * h[c->dv];
    return SLDG_OK;
}

extern "C" int sldg_diagnostics(sldg_ctx *c, double *mass, double *l2, double *ee) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int rc = run_invariants(c);
    if (rc) return rc;
    double h[3];
    CUDA_TRY(c, cudaMemcpyAsync(h, c->d_scal, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (mass) *mass = h[0];
    if (l2) *l2 = sqrt(h[1]);
    if (ee) *ee = h[2];
    return SLDG_OK;
}

extern "C" int sldg_invariants(sldg_ctx *c, double *mass, double *l2, double *ee, double *momentum,
                               double *kinetic) {
    if (!c) return SLDG_ERR_ARG;
    DeviceGuard guard(c);
    int rc = run_invariants(c);
    if (rc) return rc;
    double h[8];
    CUDA_TRY(c, cudaMemcpyAsync(h, c->d_scal, (4 + c->dv) * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (mass) *mass = h[0];
    if (l2) *l2 = sqrt(h[1]);
    if (ee) *ee = h[2];
    if (momentum) for (int a = 0; a < c->dv; ++a) momentum[a] = h[3 + a];
    if (kinetic) *kinetic = 0.5 * h[3 + c->dv];
    return SLDG_OK;
}
