// sweep_fused.cuh -- S:8(f) NEXT-1, pass fusion inside the Strang step: TWO consecutive
// translation sweeps (along dimensions k1 < k2 of the same group: x_a,x_b or v_a,v_b) in ONE
// pass over f -- one read and one write of f instead of two of each (P:92 counts every
// advection as a full read + write; this is the only way past that ceiling).
//
// The result is IDENTICAL, bit for bit, to sweep(k1) followed by sweep(k2): every value goes
// through the same two O7 chains in the same order.  It is legal because the two shifts do not
// depend on the swept coordinates of either dimension (x-shifts depend on v only, v-shifts on x
// only: P:27-31, D:R8).
//
// Mapping: f viewed as [outer2][N_k2][mid][N_k1][inner1].  One thread owns ONE CELL c of the
// k1-line (its O nodes) at fixed (inner1, mid, outer2) and walks the k2-line: for every new
// k2-cell it loads the raw values of the two k1 source cells (c+m1, c+m1+1) for the O rows of that
// k2-cell, applies the k1 rule to get the O x O k1-swept values of ITS OWN cell -- which stay in
// registers as its private sliding window along k2 -- and then emits the O x O outputs of the
// k2 rule.  No shared memory and no synchronisation: a thread only ever needs its own k1-swept
// values.  Lanes run along inner1 (k1 > 0: fully coalesced) or along the cells of the
// contiguous x_1 line (k1 = 0).
#pragma once
#include "sweep.cuh"

namespace sldg {

template <typename T, int O>
__global__ void __launch_bounds__(128)
sweep_pair_kernel(const T *__restrict__ in, T *__restrict__ out, long inner1, int n1, long midN, int n2,
                  long outer2, int nseg, int cps, int chunk,
                  const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                  const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2) {
    // thread order: `chunk` consecutive inner1 indices (lanes, coalesced), then the k1-cell c, then
    // the remaining inner1 blocks: the two threads that read the same raw k1-cell (owners of c and
    // c-1) sit in the same or the neighbouring block, so the second read is an L1/L2 hit.
    long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long il = t % chunk; t /= chunk;
    const int c = (int)(t % n1); t /= n1;
    const long ih = t % (inner1 / chunk); t /= (inner1 / chunk);
    const long ii = ih * chunk + il;
    const long mid = t % midN; t /= midN;
    const int seg = (int)(t % nseg);
    const long oo2 = t / nseg;
    if (oo2 >= outer2) return;

    const long s1 = inner1;                               // element stride between k1 nodes
    const long stride2 = midN * (long)n1 * O * inner1;    // element stride between k2 nodes
    const long plane = (oo2 * (long)n2 * O) * stride2 + mid * (long)n1 * O * inner1 + ii;
    const long lin0 = plane + (long)c * O * s1;           // this thread's first element (k2 node 0)
    const long q1 = (lin0 / qdiv1) % qmod1;
    const long q2 = (lin0 / qdiv2) % qmod2;

    T A1[O * O], B1[O * O], A2[O * O], B2[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1];
        B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2];
        B2[e] = ab2[(long)(O * O + e) * count2 + q2];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2];
    int sa = c + m1;
    if (sa >= n1) sa -= n1;
    int sb = sa + 1;
    if (sb == n1) sb = 0;
    const T *src0 = in + plane + (long)sa * O * s1;       // k1 source cell i*   (k2 node 0)
    const T *src1 = in + plane + (long)sb * O * s1;       // k1 source cell i*+1

    const int c0 = seg * cps;
    int c1 = c0 + cps;
    if (c1 > n2) c1 = n2;
    if (c0 >= c1) return;

    // raw values of the two k1 source cells for the O rows of one k2-cell
    auto load_raw = [&](int cell2, T (&r0)[O][O], T (&r1)[O][O]) {
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2) {
            const long ro = ((long)cell2 * O + l2) * stride2;
#pragma unroll
            for (int l = 0; l < O; ++l) {
                r0[l2][l] = src0[ro + l * s1];
                r1[l2][l] = src1[ro + l * s1];
            }
        }
    };
    // k1 rule on them: the O x O k1-swept values of this thread's own cell, w[l2][j1]
    auto k1_rule = [&](const T (&r0)[O][O], const T (&r1)[O][O], T (&w)[O][O]) {
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2)
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0[l2], r1[l2]);
    };

    // the O x O outputs of k2-cell i2 from the window (w0 = k2 source cell i*, w1 = i*+1)
    auto emit = [&](T *dst, const T (&w0)[O][O], const T (&w1)[O][O]) {
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2) {
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a0[O], a1[O];
#pragma unroll
                for (int l = 0; l < O; ++l) { a0[l] = w0[l][j1]; a1[l] = w1[l][j1]; }
                dst[(long)j2 * stride2 + j1 * s1] = chain<T, O>(A2, B2, j2, a0, a1);
            }
        }
    };

    // Software pipeline: the raw values of the next PF k2-cells are in flight while the current
    // cell is computed (the kernel is bound by memory latency, not by DRAM or arithmetic: ncu
    // shows long-scoreboard stalls with DRAM at 61 % at PF = 1).  Measured at config 3 / config 4,
    // traffic rate of the (x_1,x_2) pair: PF 1/2/3/4 = 4.9/5.7/6.1/6.0 TB/s (O = 2), PF 1/2 = 5.0/5.3 (O = 3).
    constexpr int PF = (O <= 2) ? 3 : (O == 3 ? 2 : 1);
    int is2 = c0 + m2;
    if (is2 >= n2) is2 -= n2;
    T ra[PF][O][O], rb[PF][O][O], w0[O][O], w1[O][O];
    load_raw(is2, ra[0], rb[0]);
    k1_rule(ra[0], rb[0], w0);
#pragma unroll
    for (int p = 0; p < PF; ++p) {
        if (++is2 == n2) is2 = 0;
        if (c0 + p < c1) load_raw(is2, ra[p], rb[p]);
    }
    T *dst = out + lin0 + (long)c0 * O * stride2;
    for (int i2 = c0; i2 < c1; i2 += PF) {
#pragma unroll
        for (int p = 0; p < PF; ++p) {
            if (i2 + p < c1) {
                k1_rule(ra[p], rb[p], w1);
                if (++is2 == n2) is2 = 0;
                if (i2 + p + PF < c1) load_raw(is2, ra[p], rb[p]);
                emit(dst, w0, w1);
#pragma unroll
                for (int l = 0; l < O; ++l)
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) w0[l][j1] = w1[l][j1];
                dst += (long)O * stride2;
            }
        }
    }
}

}  // namespace sldg
