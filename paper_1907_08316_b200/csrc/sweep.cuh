// sweep.cuh -- rows a-1 and a-2 of the hot path: shift split + A/B assembly, and the
// translation sweep kernels (section 2).
//
//   u_new[i][j] = sum_l A_jl u_old[i*][l] + sum_l B_jl u_old[i*+1][l],  i* = (i+m) mod n
//
// Arithmetic contract (D:O7 / D:R9): A,B are evaluated in fp64 and rounded once to T; every
// output is one multiply followed by 2o-1 fused multiply-adds in T, in the order
// A[j][0..o-1] then B[j][0..o-1].
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sldg {

// ------------------------------------------------------------------------------------------
// a-1: per distinct line parameter q:  delta = -sigma, m = floor(delta), theta = delta - m
// (D:R3), A(theta), B(theta) by Horner on the precomputed polynomial coefficients.
// Table layout (SoA so that per-thread reads in the v-sweeps coalesce over q):
//     mtab[q]            = m mod n  in [0, n)
//     ab[e*count + q]    = e-th entry of [A row-major | B row-major], e in [0, 2 o^2)
// ------------------------------------------------------------------------------------------
// Double-double Horner step: (hi,lo) <- (hi,lo)*theta + (chi,clo), error-free transformations
// (two-product by FMA, two-sum by Knuth); keeps the evaluated polynomial good to ~1e-30 so the
// single rounding to T below is the only one (D:O7 "rounded once").
__device__ __forceinline__ void dd_horner_step(double &hi, double &lo, double theta, double chi,
                                               double clo) {
    double p = __dmul_rn(hi, theta);
    double pe = __fma_rn(hi, theta, -p);           // hi*theta = p + pe exactly
    pe = __fma_rn(lo, theta, pe);
    double s = __dadd_rn(p, chi);                  // two-sum(p, chi)
    double bb = __dadd_rn(s, -p);
    double se = __dadd_rn(__dadd_rn(p, -__dadd_rn(s, -bb)), __dadd_rn(chi, -bb));
    se = __dadd_rn(se, __dadd_rn(pe, clo));
    hi = __dadd_rn(s, se);                         // fast two-sum renormalisation
    lo = __dadd_rn(se, -__dadd_rn(hi, -s));
}

// wide (optional): set to 1 when some line's cell offset is neither 0 nor n-1, i.e. |shift| >= 1 cell somewhere
// (the fused v-kernels keep their loads coalesced only when neighbouring lanes look at neighbouring cells)
template <typename T>
__global__ void assemble_ab_kernel(const double *__restrict__ sigma, long count, int o, int n,
                                   const double *__restrict__ coef, int *__restrict__ mtab,
                                   T *__restrict__ ab, int *__restrict__ wide = nullptr) {
    extern __shared__ double s_coef[];             // [2 o^2][2o][hi,lo]
    const int nc = 2 * o, ne = 2 * o * o;
    for (int t = threadIdx.x; t < ne * nc * 2; t += blockDim.x) s_coef[t] = coef[t];
    __syncthreads();
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= count) return;
    double delta = -sigma[q];
    double fl = floor(delta);
    double theta = delta - fl;
    if (theta >= 1.0) { fl += 1.0; theta = 0.0; }  // |delta| < 2^-54 negative: rounds to 1, is the next integer shift (D:R3)
    // m mod n without overflow for large |shift|: fmod on the (integer-valued) double
    double mm = fmod(fl, (double)n);
    if (mm < 0.0) mm += (double)n;
    int m = (int)mm;
    if (m >= n) m = 0;
    mtab[q] = m;
    if (wide && m != 0 && m != n - 1) *wide = 1;         // benign race: every writer stores the same value
    for (int e = 0; e < ne; ++e) {
        const double *c = s_coef + (size_t)e * nc * 2;
        double hi = c[(nc - 1) * 2], lo = c[(nc - 1) * 2 + 1];
        for (int k = nc - 2; k >= 0; --k) dd_horner_step(hi, lo, theta, c[k * 2], c[k * 2 + 1]);
        ab[(long)e * count + q] = (T)hi;
    }
}

// sigma for the physics sweeps (D:O3, D:R4)
//   x_a: sigma[q] = c_{v_a}(q) * tau / h_{x_a}           (coords precomputed on the host, fp64)
__global__ void sigma_from_coords_kernel(const double *__restrict__ c, long count, double tau,
                                         double h, double *__restrict__ sigma) {
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < count) sigma[q] = c[q] * tau / h;
}
//   v_a: sigma[q] = -E_a(x_q) * tau / h_{v_a}
__global__ void sigma_from_E_kernel(const double *__restrict__ E, long count, double tau, double h,
                                    double *__restrict__ sigma) {
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < count) sigma[q] = -E[q] * tau / h;
}

// ------------------------------------------------------------------------------------------
// small vector type for 128-bit (or narrower) accesses along the contiguous `inner` index
// ------------------------------------------------------------------------------------------
template <typename T, int VEC>
struct alignas(sizeof(T) * VEC) Vec {
    T v[VEC];
};

template <typename T>
__device__ __forceinline__ T fma_t(T a, T b, T c);
template <>
__device__ __forceinline__ double fma_t<double>(double a, double b, double c) { return __fma_rn(a, b, c); }
template <>
__device__ __forceinline__ float fma_t<float>(float a, float b, float c) { return __fmaf_rn(a, b, c); }
template <typename T>
__device__ __forceinline__ T mul_t(T a, T b);
template <>
__device__ __forceinline__ double mul_t<double>(double a, double b) { return __dmul_rn(a, b); }
template <>
__device__ __forceinline__ float mul_t<float>(float a, float b) { return __fmul_rn(a, b); }

// the O7 chain for local node j
template <typename T, int O>
__device__ __forceinline__ T chain(const T (&A)[O * O], const T (&B)[O * O], int j, const T *u0,
                                   const T *u1) {
    T acc = mul_t<T>(A[j * O], u0[0]);
#pragma unroll
    for (int l = 1; l < O; ++l) acc = fma_t<T>(A[j * O + l], u0[l], acc);
#pragma unroll
    for (int l = 0; l < O; ++l) acc = fma_t<T>(B[j * O + l], u1[l], acc);
    return acc;
}

// ------------------------------------------------------------------------------------------
// a-2, strided lines: f viewed as [outer][N_k = n*O][inner], element stride along the line
// = inner (>= VEC).  One thread owns VEC adjacent `inner` indices of one line segment and
// walks the cells with a sliding register window (each input row is loaded once).
//   QV = false: q = (oo / qdiv) % qmod  (x_a sweeps, a >= 2: the shift is a digit of `outer`)
//   QV = true : q = ii % X              (v_a sweeps: per-thread shift; VEC must be 1)
// UB cells are loaded per batch before any arithmetic to keep UB*O rows in flight per thread.
// ------------------------------------------------------------------------------------------
template <typename T, int O, int VEC, bool QV, int UB>
__global__ void __launch_bounds__(256)
sweep_strided_kernel(const T *__restrict__ in, T *__restrict__ out, long inner, int n, long outer,
                     int nseg, int cps, const int *__restrict__ mtab, const T *__restrict__ ab,
                     long count, long qdiv, long qmod, long X) {
    static_assert(!QV || VEC == 1, "per-thread shifts need scalar accesses");
    using V = Vec<T, VEC>;
    const long inner_v = inner / VEC;
    long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
    long iv = tid % inner_v;
    long rest = tid / inner_v;
    int seg = (int)(rest % nseg);
    long oo = rest / nseg;
    if (oo >= outer) return;
    const long ii = iv * VEC;
    const long q = QV ? (ii % X) : ((oo / qdiv) % qmod);

    T A[O * O], B[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A[e] = ab[(long)e * count + q];
        B[e] = ab[(long)(O * O + e) * count + q];
    }
    const int m = mtab[q];

    const int c0 = seg * cps;
    int c1 = c0 + cps;
    if (c1 > n) c1 = n;
    if (c0 >= c1) return;

    const long line_base = oo * (long)n * O * inner + ii;
    const T *src = in + line_base;
    T *dst = out + line_base + (long)c0 * O * inner;

    int is = c0 + m;                 // source cell i* of the first output cell
    if (is >= n) is -= n;
    V u0[O];
#pragma unroll
    for (int l = 0; l < O; ++l) u0[l] = *reinterpret_cast<const V *>(src + ((long)is * O + l) * inner);

    for (int c = c0; c < c1; c += UB) {
        V ub[UB][O];
#pragma unroll
        for (int b = 0; b < UB; ++b) {
            if (c + b < c1) {
                if (++is == n) is = 0;
#pragma unroll
                for (int l = 0; l < O; ++l)
                    ub[b][l] = *reinterpret_cast<const V *>(src + ((long)is * O + l) * inner);
            }
        }
#pragma unroll
        for (int b = 0; b < UB; ++b) {
            if (c + b < c1) {
#pragma unroll
                for (int j = 0; j < O; ++j) {
                    V r;
#pragma unroll
                    for (int e = 0; e < VEC; ++e) {
                        T a0[O], a1[O];
#pragma unroll
                        for (int l = 0; l < O; ++l) { a0[l] = u0[l].v[e]; a1[l] = ub[b][l].v[e]; }
                        r.v[e] = chain<T, O>(A, B, j, a0, a1);
                    }
                    *reinterpret_cast<V *>(dst + (long)j * inner) = r;
                }
#pragma unroll
                for (int l = 0; l < O; ++l) u0[l] = ub[b][l];
                dst += (long)O * inner;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// a-2, contiguous lines (sweep along x_1, inner = 1): f viewed as [lines][n cells][O].
// Lines that share one shift are contiguous: q = (line / qdiv) % qmod, group = qdiv lines.
// A block owns `cpb` consecutive cells of one group (a group holds qdiv*n cells); A,B are
// staged once per block in shared memory and kept in registers; one thread per cell, cells
// taken with stride blockDim so that a warp reads/writes 32 consecutive cells.
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(256)
sweep_x1_kernel(const T *__restrict__ in, T *__restrict__ out, int n, long ngroups,
                long cells_per_group, int cpb, int blocks_per_group, const int *__restrict__ mtab,
                const T *__restrict__ ab, long count, long qmod) {
    __shared__ T s_ab[2 * O * O];
    __shared__ int s_m;
    const long g = blockIdx.x / blocks_per_group;
    const int bg = blockIdx.x % blocks_per_group;
    if (g >= ngroups) return;
    const long q = g % qmod;
    for (int e = threadIdx.x; e < 2 * O * O; e += blockDim.x) s_ab[e] = ab[(long)e * count + q];
    if (threadIdx.x == 0) s_m = mtab[q];
    __syncthreads();
    T A[O * O], B[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) { A[e] = s_ab[e]; B[e] = s_ab[O * O + e]; }
    const int m = s_m;

    const long cbeg = (long)bg * cpb;
    long cend = cbeg + cpb;
    if (cend > cells_per_group) cend = cells_per_group;
    const T *gin = in + g * cells_per_group * O;
    T *gout = out + g * cells_per_group * O;
    for (long c = cbeg + threadIdx.x; c < cend; c += blockDim.x) {
        long line = c / n;
        int i = (int)(c - line * n);
        int is = i + m;
        if (is >= n) is -= n;
        int is1 = is + 1;
        if (is1 == n) is1 = 0;
        const T *p0 = gin + (line * n + is) * O;
        const T *p1 = gin + (line * n + is1) * O;
        T u0[O], u1[O];
#pragma unroll
        for (int l = 0; l < O; ++l) { u0[l] = p0[l]; u1[l] = p1[l]; }
        T *po = gout + c * O;
#pragma unroll
        for (int j = 0; j < O; ++j) po[j] = chain<T, O>(A, B, j, u0, u1);
    }
}

}  // namespace sldg
