// rho_noalloc.cu -- sldg_rho_noalloc (include/sldg.h): the rho reduction rho[x] = -sum_v W_v f[v][x]
// for callers that must not allocate device memory.
//
// Who that is: code that runs where cudaMalloc / cudaFree are off the table -- a host program that has handed
// the whole device heap to its own pool allocator up front, a callback or plug-in running inside somebody else's
// time loop where an allocation would synchronise the device (cudaFree does, cudaMalloc may) and stall every
// other stream, or a deployment whose memory budget is fixed at start-up and audited.  sldg_create allocates its
// tables (rho, E, partial sums, ...) with cudaMalloc, so none of the context-based calls fit there.
//
// What is different here: the rho pass needs scratch memory -- part[split][x], the sums over one range of
// v-nodes each, which a second kernel adds up (the v-index is the slow one in the canonical layout, so the
// splits are what gives the first kernel enough blocks to fill 148 SMs).  In sldg_compute_rho that scratch is
// c->d_part from cudaMalloc.  Here it is the fixed array g_rho_part below: SLDG_RHO_NOALLOC_SCRATCH_BYTES
// (4 MiB) of device memory that is part of the library image, so every GPU on which the library's module is
// loaded holds it from then until the process exits, used or not.  The call itself makes no cudaMalloc,
// cudaFree or other allocating call; inputs (f, W_v) and the output (rho) are the caller's.
//
// The kernels are variants of vsum_partial_kernel / vsum_final_kernel (reduce.cuh) with the same arithmetic:
// fp64 products and sums for either storage type, a compensated sum wherever one thread adds a whole
// v-line alone, a compensated fixed-order pass over the splits.  The number of splits follows from the scratch
// size, not from the context's table size, so the summation ORDER differs from sldg_compute_rho's and the two
// agree to rounding (1e-13 of max|rho| in the tests), not bit for bit.
#include "../../include/sldg.h"

#include <cuda_runtime.h>
#include <stdarg.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

namespace {

constexpr long SCRATCH_DOUBLES = SLDG_RHO_NOALLOC_SCRATCH_BYTES / sizeof(double);
static_assert(SCRATCH_DOUBLES == SLDG_RHO_NOALLOC_MAX_X, "one split of the widest x-grid must fit the scratch");

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address,
// and a kernel handed `g_rho_part` from the host side would read and write the wrong memory (or fault).
static __device__ __align__(256) double g_rho_part[SCRATCH_DOUBLES];

constexpr int MAX_DEVICES = 64;
struct DeviceSetup {
    double *part = nullptr;      // device address of g_rho_part on this device
    int sm_count = 0;
    bool ready = false;
};
DeviceSetup g_setup[MAX_DEVICES];
std::mutex g_setup_mutex;

int fail(char *err, size_t err_len, int code, const char *fmt, ...) {
    if (err && err_len) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

template <typename T, int VEC> struct alignas(sizeof(T) * VEC) Pack { T v[VEC]; };

__device__ __forceinline__ void two_sum(double &hi, double &lo, double t) {
    const double s = hi + t;
    const double bb = s - hi;
    lo += (hi - (s - bb)) + (t - bb);
    hi = s;
}

// part[split][x] = sum_{v in split} W_v f[v][x].  COMP: the product's rounding error (one FMA) and the sum's
// (two-sum) are carried along, so a thread that adds a whole v-line alone still returns the exact sum rounded once.
template <typename T, int VEC, int UB, bool COMP>
__global__ void __launch_bounds__(128)
rho_noalloc_partial_kernel(const T *__restrict__ f, long X, long V, long vps, const double *__restrict__ Wv,
                           double *__restrict__ part) {
    using Vt = Pack<T, VEC>;
    const long x = ((long)blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    if (x >= X) return;
    const long split = blockIdx.y;
    const long v0 = split * vps;
    long v1 = v0 + vps;
    if (v1 > V) v1 = V;
    double acc[VEC], lo[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) { acc[e] = 0.0; lo[e] = 0.0; }
    auto add = [&](const Vt &u, double w) {
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            const double val = (double)u.v[e];
            const double p = w * val;
            if (COMP) {
                lo[e] += fma(w, val, -p);
                two_sum(acc[e], lo[e], p);
            } else {
                acc[e] += p;
            }
        }
    };
    const T *p = f + v0 * X + x;
    long v = v0;
    for (; v + UB <= v1; v += UB) {                       // UB rows in flight per thread
        Vt u[UB];
        double w[UB];
#pragma unroll
        for (int b = 0; b < UB; ++b) {
            u[b] = *reinterpret_cast<const Vt *>(p + (long)b * X);
            w[b] = Wv[v + b];
        }
#pragma unroll
        for (int b = 0; b < UB; ++b) add(u[b], w[b]);
        p += (long)UB * X;
    }
    for (; v < v1; ++v, p += X) add(*reinterpret_cast<const Vt *>(p), Wv[v]);
#pragma unroll
    for (int e = 0; e < VEC; ++e) part[split * X + x + e] = COMP ? acc[e] + lo[e] : acc[e];
}

// rho[x] = -sum_split part[split][x]: one warp per x, lane l adds splits l, l + 32, ... in ascending order, then a
// fixed shuffle tree on (hi, lo) pairs -- the same order on every run.
__global__ void __launch_bounds__(256)
rho_noalloc_final_kernel(const double *__restrict__ part, long X, int splits, double *__restrict__ rho) {
    const long x = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (x >= X) return;
    double a = 0.0, al = 0.0;
    for (int s = lane; s < splits; s += 32) two_sum(a, al, part[(long)s * X + x]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double oh = __shfl_down_sync(0xffffffffu, a, off), ol = __shfl_down_sync(0xffffffffu, al, off);
        two_sum(a, al, oh);
        al += ol;
    }
    if (lane == 0) rho[x] = -(a + al);
}

inline long cdiv(long a, long b) { return (a + b - 1) / b; }

template <typename T, int VEC>
cudaError_t launch_partial(const T *f, long X, long V, long vps, int splits, bool comp, const double *Wv,
                           double *part, cudaStream_t stream) {
    const long xv = X / VEC;
    int block = 128;
    if (xv < block) block = (int)(cdiv(xv, 32) * 32);
    const dim3 grid((unsigned)cdiv(xv, block), (unsigned)splits);
    if (comp) rho_noalloc_partial_kernel<T, VEC, 8, true><<<grid, block, 0, stream>>>(f, X, V, vps, Wv, part);
    else rho_noalloc_partial_kernel<T, VEC, 8, false><<<grid, block, 0, stream>>>(f, X, V, vps, Wv, part);
    return cudaGetLastError();
}

template <typename T>
cudaError_t run(const void *f_, long X, long V, const double *Wv, double *rho, const DeviceSetup &dev,
                cudaStream_t stream) {
    const T *f = (const T *)f_;
    constexpr int VMAX = 16 / (int)sizeof(T);
    // widest vector load the row pitch X and the alignment of f allow
    int vec = 1;
    if (X % VMAX == 0 && ((uintptr_t)f & 15) == 0) vec = VMAX;
    else if (X % 2 == 0 && ((uintptr_t)f & (2 * sizeof(T) - 1)) == 0) vec = 2;
    // splits: enough blocks for a few waves over the SMs, as many as the scratch holds, at most one per v-node
    const long bx = cdiv(X / vec, 128);
    long s = cdiv((long)dev.sm_count * 16 * 4, bx);
    if (s > SCRATCH_DOUBLES / X) s = SCRATCH_DOUBLES / X;
    if (s > V) s = V;
    if (s > 65535) s = 65535;                              // gridDim.y
    if (s < 1) s = 1;
    const long vps = cdiv(V, s);
    const int splits = (int)cdiv(V, vps);
    const bool comp = splits == 1;
    cudaError_t e;
    if (vec == VMAX) e = launch_partial<T, VMAX>(f, X, V, vps, splits, comp, Wv, dev.part, stream);
    else if (vec == 2) e = launch_partial<T, 2>(f, X, V, vps, splits, comp, Wv, dev.part, stream);
    else e = launch_partial<T, 1>(f, X, V, vps, splits, comp, Wv, dev.part, stream);
    if (e != cudaSuccess) return e;
    rho_noalloc_final_kernel<<<(unsigned)cdiv(X * 32, 256), 256, 0, stream>>>(dev.part, X, splits, rho);
    return cudaGetLastError();
}

}  // namespace

extern "C" int sldg_rho_noalloc(const void *f_device, sldg_dtype dtype, size_t X, size_t V,
                                const double *Wv_device, double *rho_device, void *cuda_stream, char *err,
                                size_t err_len) {
    if (err && err_len) err[0] = '\0';
    if (!f_device || !Wv_device || !rho_device)
        return fail(err, err_len, SLDG_ERR_ARG, "sldg_rho_noalloc: null pointer");
    if (dtype != SLDG_F64 && dtype != SLDG_F32)
        return fail(err, err_len, SLDG_ERR_UNSUPPORTED, "sldg_rho_noalloc: unknown dtype %d", (int)dtype);
    if (X < 1 || V < 1) return fail(err, err_len, SLDG_ERR_ARG, "sldg_rho_noalloc: X and V must be at least 1");
    if (X > (size_t)SLDG_RHO_NOALLOC_MAX_X)
        return fail(err, err_len, SLDG_ERR_ARG,
                    "sldg_rho_noalloc: X = %zu x-nodes exceeds SLDG_RHO_NOALLOC_MAX_X = %ld (the fixed %ld-byte scratch "
                    "holds one partial row of at most that many doubles); use sldg_compute_rho on a context instead",
                    X, (long)SLDG_RHO_NOALLOC_MAX_X, (long)SLDG_RHO_NOALLOC_SCRATCH_BYTES);
    if (V > (size_t)1 << 40 || (double)X * (double)V > 9.0e18)
        return fail(err, err_len, SLDG_ERR_ARG, "sldg_rho_noalloc: X * V out of range");
    const size_t esize = dtype == SLDG_F64 ? 8 : 4;
    if ((uintptr_t)f_device & (esize - 1) || (uintptr_t)Wv_device & 7 || (uintptr_t)rho_device & 7)
        return fail(err, err_len, SLDG_ERR_ARG, "sldg_rho_noalloc: misaligned pointer");

    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess)
        return fail(err, err_len, SLDG_ERR_CUDA, "sldg_rho_noalloc: cudaGetDevice: %s", cudaGetErrorString(e));
    if (device < 0 || device >= MAX_DEVICES)
        return fail(err, err_len, SLDG_ERR_UNSUPPORTED, "sldg_rho_noalloc: device %d beyond the %d this build tracks",
                    device, MAX_DEVICES);
    DeviceSetup dev;
    {
        // Set-up, once per device, with that device current (it is: `device` IS the current one): the device
        // address of the scratch array and the SM count.  No allocation -- the array came with the module.
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        DeviceSetup &slot = g_setup[device];
        if (!slot.ready) {
            double *ptr = nullptr;
            e = cudaGetSymbolAddress((void **)&ptr, g_rho_part);
            if (e != cudaSuccess || !ptr)
                return fail(err, err_len, SLDG_ERR_CUDA, "sldg_rho_noalloc: cudaGetSymbolAddress(g_rho_part) on device %d: %s",
                            device, cudaGetErrorString(e));
            int sms = 0;
            e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
            if (e != cudaSuccess || sms < 1)
                return fail(err, err_len, SLDG_ERR_CUDA, "sldg_rho_noalloc: SM count of device %d: %s", device,
                            cudaGetErrorString(e));
            slot.part = ptr;
            slot.sm_count = sms;
            slot.ready = true;
        }
        dev = slot;
    }
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    e = dtype == SLDG_F64 ? run<double>(f_device, (long)X, (long)V, Wv_device, rho_device, dev, stream)
                          : run<float>(f_device, (long)X, (long)V, Wv_device, rho_device, dev, stream);
    if (e != cudaSuccess)
        return fail(err, err_len, SLDG_ERR_CUDA, "sldg_rho_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return SLDG_OK;
}
