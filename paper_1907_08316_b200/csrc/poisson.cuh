// poisson.cuh -- row a-4 (off the hot path): -Lap phi = rho + 1 periodic, E = -grad phi
// evaluated at the Gauss-Legendre x-nodes (D:R6, D:R13).
//
// Spectral, separable, dense DFT matrices per dimension (X is at most ~1.5e5 nodes and the
// solve is "usually cheap compared to operations that involve the entire data set"):
//   g_hat(m) = 1/|Omega| sum_x W_x (rho+1)(x) e^{-i k.x}      (Gauss quadrature of the Fourier
//                                                              coefficient of the piecewise polynomial)
//   phi_hat  = g_hat / |k|^2, mean mode dropped;  E_a(x) = Re sum_m (-i k_a) phi_hat(m) e^{+i k.x}
// modes |m_a| <= M_a = floor((n_a - 1)/2), k_a = 2 pi m_a / L_a.
#pragma once
#include <cuda_runtime.h>

namespace sldg {

// out[oo][r][ii] = sum_c M[r][c] * in[oo][c][ii]   (complex, index ii fastest).
//   IN_REAL : `in_re` is a real array and 1 is added to it (rho + 1); in_im ignored
//   OUT_REAL: only the real part is written, to out_re
// One WARP per output element: lanes stride over c, then a fixed shuffle tree (deterministic).
// The sums have up to 768 terms and few outputs in 1-D (255 modes), so one thread per output
// left the step of the small configs dominated by this kernel (195 of ~600 us under ncu).
template <bool IN_REAL, bool OUT_REAL>
__global__ void __launch_bounds__(256)
cplx_apply_kernel(const double *__restrict__ in_re, const double *__restrict__ in_im, long outer, long cols,
                  long inner, const double2 *__restrict__ M, long rows, double *__restrict__ out_re,
                  double *__restrict__ out_im) {
    const long t = ((long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    const long total = outer * rows * inner;
    if (t >= total) return;                       // whole warps leave together
    const long ii = t % inner;
    const long r = (t / inner) % rows;
    const long oo = t / (inner * rows);
    const double2 *Mr = M + r * cols;
    const long base = oo * cols * inner + ii;
    double sr = 0.0, si = 0.0;
    for (long c = lane; c < cols; c += 32) {
        double2 m = Mr[c];
        double xr = in_re[base + c * inner];
        if (IN_REAL) {
            xr += 1.0;
            sr = fma(m.x, xr, sr);
            si = fma(m.y, xr, si);
        } else {
            double xi = in_im[base + c * inner];
            sr = fma(m.x, xr, fma(-m.y, xi, sr));
            si = fma(m.x, xi, fma(m.y, xr, si));
        }
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        sr += __shfl_down_sync(0xffffffffu, sr, off);
        si += __shfl_down_sync(0xffffffffu, si, off);
    }
    if (lane == 0) {
        out_re[t] = sr;
        if (!OUT_REAL) out_im[t] = si;
    }
}

// (er, ei)[q] = (-i k_a) g_hat[q] / |k|^2  (0 at the mean mode); q over the K_0 x .. x K_{dx-1} modes
__global__ void poisson_scale_kernel(const double *__restrict__ gr, const double *__restrict__ gi,
                                     long KK, int dx, int a, long K0, long K1, long K2, long M0,
                                     long M1, long M2, double kf0, double kf1, double kf2,
                                     double *__restrict__ er, double *__restrict__ ei) {
    long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= KK) return;
    long r0 = q % K0, r1 = (q / K0) % K1, r2 = q / (K0 * K1);
    double k[3];
    k[0] = kf0 * (double)(r0 - M0);
    k[1] = dx > 1 ? kf1 * (double)(r1 - M1) : 0.0;
    k[2] = dx > 2 ? kf2 * (double)(r2 - M2) : 0.0;
    double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
    if (k2 == 0.0) { er[q] = 0.0; ei[q] = 0.0; return; }
    double pr = gr[q] / k2, pi = gi[q] / k2;
    // (-i k)(pr + i pi) = k pi - i k pr
    er[q] = k[a] * pi;
    ei[q] = -k[a] * pr;
}

}  // namespace sldg
