// reduce.cuh -- rows a-3 and a-6: rho(x) = -sum_v W_v f[v][x] and the invariants mass,
// L2 norm, electric energy (D:R12).  fp64 accumulators for both storage types and a
// hierarchical, deterministic reduction thread -> split -> final pass.
//
// In the canonical layout the reduced index v is the SLOW one, so the bulk of the work is a
// per-thread column sum over a range of v (coalesced, 128-bit loads along x); the ranges
// ("splits") exist only to expose enough parallelism.  Full reductions to a scalar over the
// X-sized results use warp shuffles + one shared-memory stage in a single block.
#pragma once
#include <cuda_runtime.h>

#include "sweep.cuh"   // Vec<T,VEC>

namespace sldg {

// Compensated accumulation (Knuth two-sum + the exact product error from one FMA): (hi, lo) carries
// the running sum to about twice the working precision, so hi + lo is the exactly summed value rounded
// once -- what D:O4 defines rho to be.  Used where a thread sums a whole v-line alone (one split) and
// in the pass over the splits; the split partials of large problems are short sums already.
__device__ __forceinline__ void two_sum_acc(double &hi, double &lo, double t) {
    const double s = hi + t;
    const double bb = s - hi;
    lo += (hi - (s - bb)) + (t - bb);
    hi = s;
}
__device__ __forceinline__ void comp_add_product(double &hi, double &lo, double w, double val) {
    const double p = w * val;
    lo += fma(w, val, -p);
    two_sum_acc(hi, lo, p);
}

// part_rho[split][x] = sum_{v in split} W_v f[v][x]   (the rho pass of the Strang step: rho only)
// COMP: compensated accumulation (one-split launches: the partial IS rho).
template <typename T, int VEC, int UB, bool COMP = false>
__global__ void __launch_bounds__(128)
vsum_partial_kernel(const T *__restrict__ f, long X, long V, long vps,
                    const double *__restrict__ Wv, double *__restrict__ part_rho) {
    using Vt = Vec<T, VEC>;
    const long xv = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long x = xv * VEC;
    if (x >= X) return;
    const long split = blockIdx.y;
    const long v0 = split * vps;
    long v1 = v0 + vps;
    if (v1 > V) v1 = V;
    double acc[VEC], lo[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) { acc[e] = 0.0; lo[e] = 0.0; }
    const T *p = f + v0 * X + x;
    long v = v0;
    for (; v + UB <= v1; v += UB) {
        Vt u[UB];
        double w[UB];
#pragma unroll
        for (int b = 0; b < UB; ++b) {
            u[b] = *reinterpret_cast<const Vt *>(p + (long)b * X);
            w[b] = Wv[v + b];
        }
#pragma unroll
        for (int b = 0; b < UB; ++b)
#pragma unroll
            for (int e = 0; e < VEC; ++e) {
                double val = (double)u[b].v[e];
                if (COMP) comp_add_product(acc[e], lo[e], w[b], val);
                else acc[e] += w[b] * val;
            }
        p += (long)UB * X;
    }
    for (; v < v1; ++v) {
        Vt u = *reinterpret_cast<const Vt *>(p);
        double w = Wv[v];
#pragma unroll
        for (int e = 0; e < VEC; ++e) {
            double val = (double)u.v[e];
            if (COMP) comp_add_product(acc[e], lo[e], w, val);
            else acc[e] += w * val;
        }
        p += X;
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e) part_rho[split * X + x + e] = COMP ? acc[e] + lo[e] : acc[e];
}

__device__ __forceinline__ double warp_sum(double v);

// rho[x] = -sum_split part_rho[split][x];  s2[x] = +sum_split part_s2[split][x].
// One WARP per x: lane l adds splits l, l+32, ... in ascending order, then a fixed shuffle tree
// (deterministic; with one split it is exactly the single partial).  A thread per x walking
// thousands of splits serially made this pass slower than the partial pass for small X (1+3 D).
__global__ void __launch_bounds__(256)
vsum_final_kernel(const double *__restrict__ part_rho, const double *__restrict__ part_s2, long X, int splits,
                  double *__restrict__ rho, double *__restrict__ rho_copy, double *__restrict__ s2) {
    const long x = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (x >= X) return;
    double a = 0.0, al = 0.0, b = 0.0;
    for (int s = lane; s < splits; s += 32) {
        two_sum_acc(a, al, part_rho[(long)s * X + x]);
        if (part_s2) b += part_s2[(long)s * X + x];
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {             // fixed tree on (hi, lo) pairs
        const double oh = __shfl_down_sync(0xffffffffu, a, off), ol = __shfl_down_sync(0xffffffffu, al, off);
        two_sum_acc(a, al, oh);
        al += ol;
    }
    a += al;
    b = warp_sum(b);
    if (lane == 0) {
        rho[x] = -a;
        if (rho_copy) rho_copy[x] = -a;
        if (s2) s2[x] = b;
    }
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    return v;
}

// One block of 1024 threads.  out[0] = sum_x W_x (-rho[x]) (mass), out[1] = sum_x W_x s2[x]
// (l2 squared), out[2] = 1/2 sum_x W_x sum_a E_a[x]^2 (electric energy).
__global__ void __launch_bounds__(1024)
scalars_kernel(const double *__restrict__ rho, const double *__restrict__ s2,
               const double *__restrict__ E, const double *__restrict__ Wx, long X, int dx,
               double *__restrict__ out) {
    __shared__ double sm[3][32];
    double a = 0.0, b = 0.0, c = 0.0;
    for (long x = threadIdx.x; x < X; x += blockDim.x) {
        double w = Wx[x];
        a -= w * rho[x];
        b += w * s2[x];
        double e2 = 0.0;
        for (int d = 0; d < dx; ++d) { double e = E[(long)d * X + x]; e2 = fma(e, e, e2); }
        c += w * e2;
    }
    a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { sm[0][wid] = a; sm[1][wid] = b; sm[2][wid] = c; }
    __syncthreads();
    if (wid == 0) {
        a = sm[0][lane]; b = sm[1][lane]; c = sm[2][lane];
        a = warp_sum(a); b = warp_sum(b); c = warp_sum(c);
        if (lane == 0) { out[0] = a; out[1] = b; out[2] = 0.5 * c; }
    }
}

}  // namespace sldg

namespace sldg {

// rows[k][x] = sum_split part[k][split][x], k < nk: one WARP per (k, x), lane l adds splits l, l+32, ... in
// ascending order, then a fixed shuffle tree (as vsum_final_kernel; a single block walking splits * X * nk
// values serially took milliseconds at X = 128, V = 2.4e6)
__global__ void __launch_bounds__(256)
vrows_final_kernel(const double *__restrict__ part, long X, int splits, int nsplit_cap, int nk,
                   double *__restrict__ rows) {
    const long w = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= (long)nk * X) return;
    const long k = w / X, x = w - k * X;
    double a = 0.0;
    for (int s = lane; s < splits; s += 32) a += part[(k * nsplit_cap + s) * X + x];
    a = warp_sum(a);
    if (lane == 0) rows[k * X + x] = a;
}

// out[k] = sum_x W_x rows[k][x], k < nk (one block of 1024 threads, fixed order)
__global__ void __launch_bounds__(1024)
moments_final_kernel(const double *__restrict__ rows, const double *__restrict__ Wx, long X, int nk,
                     double *__restrict__ out) {
    __shared__ double sm[32];
    for (int k = 0; k < nk; ++k) {
        double a = 0.0;
        for (long x = threadIdx.x; x < X; x += blockDim.x) a += Wx[x] * rows[(long)k * X + x];
        a = warp_sum(a);
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        if (lane == 0) sm[wid] = a;
        __syncthreads();
        if (wid == 0) {
            a = warp_sum(sm[lane]);
            if (lane == 0) out[k] = a;
        }
        __syncthreads();
    }
}

}  // namespace sldg

namespace sldg {

// S:8(f) NEXT-4 as the survey words it -- "fused into the rho pass" (P:69 lists the invariants together,
// P:92 writes them once per step): ONE read of f emits, per x-node and v-split,
//   part[0] = sum_v W_v f            (-> rho, mass)            part[1] = sum_v W_v f^2   (-> l2)
//   part[2+a] = sum_v v_a W_v f      (-> momentum, a < DV)     part[2+DV] = sum_v |v|^2 W_v f (-> kinetic energy)
// with fp64 accumulators and the split structure of the rho pass.  The rho and f^2 sums are the very
// operations, in the very order, of vsum_partial_kernel<.., WITH_S2 = true, ..>, so sldg_diagnostics gives the
// same bits whichever pass produced its partials.  COMP: compensated rho sum (one-split launches, D:O4).
template <typename T, int VEC, int DV, int UB, bool COMP, int BLK>
__global__ void __launch_bounds__(BLK)
vall_partial_kernel(const T *__restrict__ f, long X, long V, long vps, long part_stride /* cap * X */,
                    const double *__restrict__ Wv, const double *__restrict__ va /* [DV][V] */,
                    const double *__restrict__ v2, double *__restrict__ part) {
    using Vt = Vec<T, VEC>;
    // The per-row scalars (W_v, |v|^2, v_a) of a chunk of CH rows are staged in shared memory, the next chunk's
    // prefetched while this one is summed: read through L1 beside the streaming f rows they missed to L2 several
    // times per batch and every row's arithmetic waited for them (ncu: 33 stall cycles per issue, DRAM at 48 %).
    constexpr int CH = 64, NT = DV + 2, PER = (NT * CH + BLK - 1) / BLK;   // blockDim.x == BLK
    __shared__ double s_tab[2][NT][CH];
    const long xv = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long x = xv * VEC;
    const bool valid = x < X;
    const long split = blockIdx.y;
    const long v0 = split * vps;
    long v1 = v0 + vps;
    if (v1 > V) v1 = V;
    auto table_entry = [&](int idx, long c0) -> double {    // entry idx = t * CH + r of the chunk starting at c0
        const int t = idx / CH, r = idx - t * CH;
        const long v = c0 + r;
        if (idx >= NT * CH || v >= v1) return 0.0;
        return t == 0 ? Wv[v] : (t == 1 ? v2[v] : va[(long)(t - 2) * V + v]);
    };
    double pre[PER];
#pragma unroll
    for (int i = 0; i < PER; ++i) pre[i] = table_entry((int)threadIdx.x + i * (int)blockDim.x, v0);
    double acc[VEC], lo[VEC], acc2[VEC], mom[DV + 1][VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        acc[e] = 0.0; lo[e] = 0.0; acc2[e] = 0.0;
#pragma unroll
        for (int k = 0; k <= DV; ++k) mom[k][e] = 0.0;
    }
    const T *p = f + v0 * X + (valid ? x : 0);
    int cur = 0;
    for (long c0 = v0; c0 < v1; c0 += CH) {
#pragma unroll
        for (int i = 0; i < PER; ++i) {
            const int idx = (int)threadIdx.x + i * (int)blockDim.x;
            if (idx < NT * CH) (&s_tab[cur][0][0])[idx] = pre[i];
        }
        __syncthreads();                                     // chunk c0 staged (and the other buffer free again)
#pragma unroll
        for (int i = 0; i < PER; ++i) pre[i] = table_entry((int)threadIdx.x + i * (int)blockDim.x, c0 + CH);
        const int rows = (int)((v1 - c0 < CH) ? v1 - c0 : CH);
        if (valid) {
            auto add_row = [&](const Vt &u, int r) {
                const double w = s_tab[cur][0][r], s2 = s_tab[cur][1][r];
                double c[DV];
#pragma unroll
                for (int a = 0; a < DV; ++a) c[a] = s_tab[cur][2 + a][r];
#pragma unroll
                for (int e = 0; e < VEC; ++e) {
                    const double val = (double)u.v[e];
                    const double wv = w * val;
                    if (COMP) comp_add_product(acc[e], lo[e], w, val);
                    else acc[e] += wv;
                    acc2[e] = fma(wv, val, acc2[e]);
#pragma unroll
                    for (int a = 0; a < DV; ++a) mom[a][e] = fma(c[a], wv, mom[a][e]);
                    mom[DV][e] = fma(s2, wv, mom[DV][e]);
                }
            };
            int r = 0;
            for (; r + UB <= rows; r += UB) {
                Vt u[UB];
#pragma unroll
                for (int b = 0; b < UB; ++b) u[b] = *reinterpret_cast<const Vt *>(p + (long)b * X);
#pragma unroll
                for (int b = 0; b < UB; ++b) add_row(u[b], r + b);
                p += (long)UB * X;
            }
            for (; r < rows; ++r) {
                Vt u = *reinterpret_cast<const Vt *>(p);
                add_row(u, r);
                p += X;
            }
        }
        cur ^= 1;
    }
    if (!valid) return;
    double *o = part + split * X + x;
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
        o[e] = COMP ? acc[e] + lo[e] : acc[e];
        o[part_stride + e] = acc2[e];
#pragma unroll
        for (int k = 0; k <= DV; ++k) o[(2 + k) * part_stride + e] = mom[k][e];
    }
}

}  // namespace sldg
