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
#include "sweep_tma.cuh"
#include "tma.cuh"

namespace sldg {

// VEC1: k1 is the contiguous x_1 line (inner1 == 1) and O is even, so the O nodes of a cell are
// read / written as 2-element vectors (16 B in fp64): half the load/store requests and L1
// wavefronts (the x-fused kernels were bound by the LSU pipe: 87 % wavefront utilisation in ncu).
template <typename T, int O, bool VEC1>
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
            if constexpr (VEC1) {
                using V2 = Vec<T, 2>;
#pragma unroll
                for (int l = 0; l < O; l += 2) {
                    V2 a = *reinterpret_cast<const V2 *>(src0 + ro + l);
                    V2 b = *reinterpret_cast<const V2 *>(src1 + ro + l);
                    r0[l2][l] = a.v[0]; r0[l2][l + 1] = a.v[1];
                    r1[l2][l] = b.v[0]; r1[l2][l + 1] = b.v[1];
                }
            } else {
#pragma unroll
                for (int l = 0; l < O; ++l) {
                    r0[l2][l] = src0[ro + l * s1];
                    r1[l2][l] = src1[ro + l * s1];
                }
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
            T res[O];
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a0[O], a1[O];
#pragma unroll
                for (int l = 0; l < O; ++l) { a0[l] = w0[l][j1]; a1[l] = w1[l][j1]; }
                res[j1] = chain<T, O>(A2, B2, j2, a0, a1);
            }
            if constexpr (VEC1) {
                using V2 = Vec<T, 2>;
#pragma unroll
                for (int j1 = 0; j1 < O; j1 += 2) {
                    V2 v; v.v[0] = res[j1]; v.v[1] = res[j1 + 1];
                    *reinterpret_cast<V2 *>(dst + (long)j2 * stride2 + j1) = v;
                }
            } else {
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) dst[(long)j2 * stride2 + j1 * s1] = res[j1];
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

namespace sldg {

// ------------------------------------------------------------------------------------------
// THREE consecutive sweeps (k1 < k2 < k3, all x- or all v-dimensions: the 3+3 D step) in one pass.
// Same idea one level up: a thread owns one k1-cell x one k2-cell (O x O nodes) at fixed other
// indices and walks the k3 line.  For every new k3-cell and each of its O rows it loads the raw
// values of the 2 x 2 source cells (4 O^2 values), applies the k1 rule (-> 2 O^2 values), then
// the k2 rule (-> the O^2 values of ITS OWN cell pair), which form its private sliding window
// along k3; the k3 rule emits O^3 outputs per k3-cell.  Bit-identical to the three sweeps.
// Each raw value is needed by 4 threads (neighbours in c1, c2): L1/L2 hits, DRAM sees one read
// and one write of f for three sweeps.  Instantiated for O <= 2 (4 O^3 raw values per cell).
// ------------------------------------------------------------------------------------------
template <typename T, int O, bool VEC1>
__global__ void __launch_bounds__(128, 3)
sweep_triple_kernel(const T *__restrict__ in, T *__restrict__ out, long inner1, int n1, long mid12, int n2,
                    long mid23, int n3, long outer3, int chunk,
                    const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                    const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                    const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    // thread order: lanes along inner1 (chunk), then c1, then c2: the 4 threads that read one raw
    // value (owners of (c1, c2), (c1-1, c2), (c1, c2-1), (c1-1, c2-1)) are at most chunk*n1 threads
    // apart, so the repeats are L1/L2 hits (with c2 further out, the v-triple re-read f from HBM).
    long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const long il = t % chunk; t /= chunk;
    const int c1 = (int)(t % n1); t /= n1;
    const int c2 = (int)(t % n2); t /= n2;
    const long ih = t % (inner1 / chunk); t /= (inner1 / chunk);
    const long ii = ih * chunk + il;
    const long m12 = t % mid12; t /= mid12;
    const long m23 = t % mid23;
    const long oo3 = t / mid23;
    if (oo3 >= outer3) return;

    const long s1 = inner1;
    const long s2 = mid12 * (long)n1 * O * s1;
    const long s3 = mid23 * (long)n2 * O * s2;
    const long base = oo3 * (long)n3 * O * s3 + m23 * (long)n2 * O * s2 + m12 * (long)n1 * O * s1 + ii;
    const long own = (long)c1 * O * s1 + (long)c2 * O * s2;
    const long lin0 = base + own;
    const long q1 = (lin0 / qdiv1) % qmod1, q2 = (lin0 / qdiv2) % qmod2, q3 = (lin0 / qdiv3) % qmod3;

    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    int sa2 = c2 + m2; if (sa2 >= n2) sa2 -= n2;
    int sb2 = sa2 + 1; if (sb2 == n2) sb2 = 0;
    // offsets of the 2 x 2 source cells (k2 cell, k1 cell) relative to `base`
    const long off[2][2] = {{(long)sa2 * O * s2 + (long)sa1 * O * s1, (long)sa2 * O * s2 + (long)sb1 * O * s1},
                            {(long)sb2 * O * s2 + (long)sa1 * O * s1, (long)sb2 * O * s2 + (long)sb1 * O * s1}};

    // raw[l3][cell2][l2][cell1][l1]
    auto load_raw = [&](int cell3, T (&r)[O][2][O][2][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            const T *row = in + base + ((long)cell3 * O + l3) * s3;
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2)
#pragma unroll
                    for (int e1 = 0; e1 < 2; ++e1) {
                        if constexpr (VEC1) {
                            using V2 = Vec<T, 2>;
#pragma unroll
                            for (int l1 = 0; l1 < O; l1 += 2) {
                                V2 a = *reinterpret_cast<const V2 *>(row + off[e2][e1] + l2 * s2 + l1);
                                r[l3][e2][l2][e1][l1] = a.v[0]; r[l3][e2][l2][e1][l1 + 1] = a.v[1];
                            }
                        } else {
#pragma unroll
                            for (int l1 = 0; l1 < O; ++l1) r[l3][e2][l2][e1][l1] = row[off[e2][e1] + l2 * s2 + l1 * s1];
                        }
                    }
        }
    };
    // k1 rule then k2 rule: w[l3][j2][j1] = the (k1,k2)-swept values of this thread's own cell pair
    auto k12_rule = [&](const T (&r)[O][2][O][2][O], T (&w)[O][O][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[2][O][O];                                   // k1-swept: [cell2][l2][j1]
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2)
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r[l3][e2][l2][0], r[l3][e2][l2][1]);
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };

    // x-triple (VEC1: k1 = x_1 contiguous, k2 = x_2 adjacent): the raw rows of one k3-cell that
    // this thread's k2-cell pair needs are two contiguous spans of O x_1-lines per k3-row; the
    // owner of c1 == 0 asks the copy engine to pull them into L2 two k3-cells ahead, so the
    // demand loads (one cell ahead, in registers) find them in L2 instead of HBM.
    auto prefetch_l2 = [&](int cell3) {
        if constexpr (VEC1) {
            if (c1 == 0 && mid12 == 1) {
                const uint32_t span = (uint32_t)((size_t)O * s2 * sizeof(T));
#pragma unroll
                for (int l3 = 0; l3 < O; ++l3) {
                    const T *row = in + base + ((long)cell3 * O + l3) * s3;
                    bulk_prefetch_l2(row + (long)sa2 * O * s2, span);
                    bulk_prefetch_l2(row + (long)sb2 * O * s2, span);
                }
            }
        }   // (per-lane bulk prefetches in the strided v-triple were tried: 16.6 -> 23.0 ms, removed)
    };

    int is3 = m3;                                            // source k3-cell of output cell 0
    T raw[O][2][O][2][O], w0[O][O][O], w1[O][O][O];
    load_raw(is3, raw);
    k12_rule(raw, w0);
    if (++is3 == n3) is3 = 0;
    load_raw(is3, raw);
    {
        int p3 = is3 + 1;
        if (p3 == n3) p3 = 0;
        prefetch_l2(p3);
    }
    T *dst = out + lin0;
    for (int i3 = 0; i3 < n3; ++i3) {
        k12_rule(raw, w1);
        if (i3 + 1 < n3) {                                   // next cell's loads fly during the arithmetic below
            if (++is3 == n3) is3 = 0;
            load_raw(is3, raw);
            if (i3 + 2 < n3) {
                int p3 = is3 + 1;
                if (p3 == n3) p3 = 0;
                prefetch_l2(p3);
            }
        }
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2) {
                T res[O];
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = w0[l][j2][j1]; a1[l] = w1[l][j2][j1]; }
                    res[j1] = chain<T, O>(A3, B3, j3, a0, a1);
                }
                if constexpr (VEC1) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j1 = 0; j1 < O; j1 += 2) {
                        V2 v; v.v[0] = res[j1]; v.v[1] = res[j1 + 1];
                        *reinterpret_cast<V2 *>(dst + (long)j3 * s3 + (long)j2 * s2 + j1) = v;
                    }
                } else {
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) dst[(long)j3 * s3 + (long)j2 * s2 + j1 * s1] = res[j1];
                }
            }
#pragma unroll
        for (int l = 0; l < O; ++l)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) w0[l][j2][j1] = w1[l][j2][j1];
        dst += (long)O * s3;
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// x_1 x_2 x_3 triple for 3+3 D with a small x-grid, STAGED BY THE COPY ENGINE.
// One block per velocity node v (all shifts and A,B are uniform in a block: they depend on v
// only).  A k3-cell of one v is ONE contiguous slab of O * N2 * N1 values (x_1 and x_2 are the
// two fastest dimensions, consecutive x_3 nodes follow each other), so the block streams the
// n3 slabs through a 3-deep shared-memory ring with one cp.async.bulk per slab (mbarrier
// complete_tx); thread (c1, c2) reads the 2 x 2 source cells from the slab (periodic wrap is
// free in shared memory), applies the k1 and k2 rules, keeps its O^3 values as sliding window
// along x_3 and emits O^3 outputs per cell.  No raw registers, loads fully asynchronous: the
// register-limited latency-bound behaviour of sweep_triple_kernel (4.9 TB/s) is gone.
// The first slab's swept values are kept to close the periodic line (no slab is read twice).
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(512, 1)
sweep_xtriple_plane_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int n3, int tpr,
                           const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                           const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                           const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 4;                                   // ring depth (3 -> 4: 11.36 -> 11.08 ms at config 5; 6: 11.00)
    __shared__ __align__(8) uint64_t full[NS];
    const long N1 = (long)n1 * O, N2 = (long)n2 * O;
    const long slab = O * N2 * N1;                           // elements per k3-cell
    const size_t slab_bytes = (size_t)slab * sizeof(T);
    const size_t slot_stride = (slab_bytes + 127) & ~(size_t)127;
    const long v = blockIdx.x;
    const long base = v * (long)n3 * slab;                   // first element of this v (x-block is contiguous)
    const int tid = threadIdx.x;
    // tpr threads per x_2-cell row, n1 of them active (tpr > n1 pads rows for bank conflicts; measured slower)
    const int c1r = tid % tpr, c2 = tid / tpr;
    const bool active = c2 < n2 && c1r < n1;
    const int c1 = c1r < n1 ? c1r : 0;

    const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2, q3 = (base / qdiv3) % qmod3;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    int sa2 = (active ? c2 : 0) + m2; if (sa2 >= n2) sa2 -= n2;
    int sb2 = sa2 + 1; if (sb2 == n2) sb2 = 0;
    const int off[2][2] = {{(int)(sa2 * O * N1 + sa1 * O), (int)(sa2 * O * N1 + sb1 * O)},
                           {(int)(sb2 * O * N1 + sa1 * O), (int)(sb2 * O * N1 + sb1 * O)}};

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    __syncthreads();
    auto issue = [&](int j) {                                // slab j <-> source k3-cell (m3 + j) mod n3
        int cell = m3 + j;
        if (cell >= n3) cell -= n3;
        const int slot = j % NS;
        mbar_expect_tx(&full[slot], (uint32_t)slab_bytes);
        bulk_g2s(smem_raw + slot * slot_stride, in + base + (long)cell * slab, (uint32_t)slab_bytes, &full[slot]);
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n3; ++j) issue(j);

    // (k1,k2)-swept values of this thread's cell pair from the slab in `slot`
    auto k12_from_slab = [&](int slot, T (&w)[O][O][O]) {
        const T *sl = reinterpret_cast<const T *>(smem_raw + slot * slot_stride);
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[2][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    T r0[O], r1[O];
                    load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][0] + l2 * N1, r0);
                    load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][1] + l2 * N1, r1);
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };
    auto emit = [&](int i3, const T (&w0)[O][O][O], const T (&w1)[O][O][O]) {
        T *dst = out + base + (long)i3 * slab + (long)c2 * O * N1 + (long)c1 * O;
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2) {
                T res[O];
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = w0[l][j2][j1]; a1[l] = w1[l][j2][j1]; }
                    res[j1] = chain<T, O>(A3, B3, j3, a0, a1);
                }
                T *p = dst + (long)j3 * N2 * N1 + (long)j2 * N1;
                if constexpr (O % 2 == 0) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j1 = 0; j1 < O; j1 += 2) {
                        V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                        *reinterpret_cast<V2 *>(p + j1) = vv;
                    }
                } else {
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
                }
            }
    };

    T wfirst[O][O][O], w0[O][O][O], w1[O][O][O];
    for (int j = 0; j < n3; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        if (active) {
            if (j == 0) {
                k12_from_slab(slot, wfirst);
#pragma unroll
                for (int a = 0; a < O; ++a)
#pragma unroll
                    for (int b = 0; b < O; ++b)
#pragma unroll
                        for (int d = 0; d < O; ++d) w0[a][b][d] = wfirst[a][b][d];
            } else {
                k12_from_slab(slot, w1);
                emit(j - 1, w0, w1);
#pragma unroll
                for (int a = 0; a < O; ++a)
#pragma unroll
                    for (int b = 0; b < O; ++b)
#pragma unroll
                        for (int d = 0; d < O; ++d) w0[a][b][d] = w1[a][b][d];
            }
        }
        __syncthreads();                                     // everyone is done with this slot
        if (tid == 0 && j + NS < n3) issue(j + NS);
    }
    if (active) emit(n3 - 1, w0, wfirst);                    // closes the periodic line
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// x_1 x_2 pair, STAGED BY THE COPY ENGINE (the pair analogue of sweep_xtriple_plane_kernel).
// One block per (x_1, x_2) plane, i.e. per value of all higher indices; its shifts and A,B are
// uniform (they depend on v only).  A k2-cell of the plane is ONE contiguous slab of O * N1
// values, streamed through a 3-deep shared-memory ring by cp.async.bulk; thread c1 reads its two
// source cells from the slab, keeps its O x O window along x_2 and emits O x O outputs per cell.
// No raw-value registers and no register prefetch: at o = 3, 4 the register pair kernel is
// occupancy-starved (168 / 255 registers), this one is not.
// ------------------------------------------------------------------------------------------
// K1ID: the k1 rule is the identity (A = I, B = 0, offset 0) and is skipped: the kernel is then the single x_2
// sweep, staged slab by slab by the copy engine (used for sldg_translate / sldg_advect along x_2).
template <typename T, int O, bool K1ID = false, bool MULTI = false>
__global__ void __launch_bounds__(256)
sweep_xpair_plane_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int ppb, long planes,
                         const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                         const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2) {
    // ppb planes per block (> 1 when the x_1 line has fewer cells than a warp has lanes: n_1 = 16 left half of
    // every warp idle); each plane has its own shifts, its own sub-slot of every ring slot and its own slab order
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 4;                                   // ring depth
    constexpr int PPB_MAX = MULTI ? 8 : 1;
    if constexpr (!MULTI) ppb = 1;                           // one plane per block: everything below folds to that
    __shared__ __align__(8) uint64_t full[NS];
    const long N1 = (long)n1 * O;
    const long slab = O * N1;                                // elements per k2-cell of one plane
    const size_t slab_bytes = (size_t)slab * sizeof(T);
    const size_t sub_stride = (slab_bytes + 127) & ~(size_t)127;
    const size_t slot_stride = sub_stride * ppb;
    const int tid = threadIdx.x;
    const int pl = MULTI ? tid / n1 : (tid < n1 ? 0 : 1);    // plane of this thread within the block
    const int c1 = MULTI ? tid - pl * n1 : tid;
    const long plane0 = (long)blockIdx.x * ppb;
    const bool active = pl < ppb && plane0 + pl < planes;
    const long base = (active ? plane0 + pl : plane0) * n2 * slab;          // planes are contiguous
    const size_t sub_off = (size_t)(active ? pl : 0) * sub_stride;

    const long q1 = K1ID ? 0 : (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        if constexpr (!K1ID) { A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1]; }
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
    }
    const int m1 = K1ID ? 0 : mtab1[q1];                     // (the k2 offsets are needed by thread 0 only, below)
    int sa1 = (active ? c1 : 0) + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    __syncthreads();
    // thread 0 issues the copies of every plane of the block: their cell offsets
    int m2s[PPB_MAX];
    int nloc = 0;
    if (tid == 0) {
        for (int p = 0; p < ppb && p < PPB_MAX; ++p)
            if (plane0 + p < planes) {
                m2s[p] = mtab2[(((plane0 + p) * n2 * slab) / qdiv2) % qmod2];
                nloc = p + 1;
            }
    }
    auto issue = [&](int j) {                                // slab j <-> source k2-cell (m2 + j) mod n2, per plane
        const int slot = j % NS;
        mbar_expect_tx(&full[slot], (uint32_t)(slab_bytes * nloc));
#pragma unroll
        for (int p = 0; p < PPB_MAX; ++p)
            if (p < nloc) {
                int cell = m2s[p] + j;
                if (cell >= n2) cell -= n2;
                bulk_g2s(smem_raw + slot * slot_stride + p * sub_stride, in + ((plane0 + p) * n2 + cell) * slab,
                         (uint32_t)slab_bytes, &full[slot]);
            }
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n2; ++j) issue(j);

    auto k1_from_slab = [&](int slot, T (&w)[O][O]) {       // w[l2][j1]
        const T *sl = reinterpret_cast<const T *>(smem_raw + slot * slot_stride + sub_off);
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2) {
            T r0[O], r1[O];
            load_cell<T, O>(sl + l2 * N1 + (long)sa1 * O, r0);
            if constexpr (K1ID) {
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = r0[j1];
            } else {
                load_cell<T, O>(sl + l2 * N1 + (long)sb1 * O, r1);
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
            }
        }
    };
    auto emit = [&](int i2, const T (&w0)[O][O], const T (&w1)[O][O]) {
        T *dst = out + base + (long)i2 * slab + (long)c1 * O;
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2) {
            T res[O];
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a0[O], a1[O];
#pragma unroll
                for (int l = 0; l < O; ++l) { a0[l] = w0[l][j1]; a1[l] = w1[l][j1]; }
                res[j1] = chain<T, O>(A2, B2, j2, a0, a1);
            }
            T *p = dst + (long)j2 * N1;
            if constexpr (O % 2 == 0) {
                using V2 = Vec<T, 2>;
#pragma unroll
                for (int j1 = 0; j1 < O; j1 += 2) {
                    V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                    *reinterpret_cast<V2 *>(p + j1) = vv;
                }
            } else {
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
            }
        }
    };

    T wfirst[O][O], w0[O][O], w1[O][O];
    for (int j = 0; j < n2; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        if (active) {
            if (j == 0) {
                k1_from_slab(slot, wfirst);
#pragma unroll
                for (int a = 0; a < O; ++a)
#pragma unroll
                    for (int b = 0; b < O; ++b) w0[a][b] = wfirst[a][b];
            } else {
                k1_from_slab(slot, w1);
                emit(j - 1, w0, w1);
#pragma unroll
                for (int a = 0; a < O; ++a)
#pragma unroll
                    for (int b = 0; b < O; ++b) w0[a][b] = w1[a][b];
            }
        }
        __syncthreads();                                     // everyone is done with this slot
        if (tid == 0 && j + NS < n2) issue(j + NS);
    }
    if (active) emit(n2 - 1, w0, wfirst);                    // closes the periodic line
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// v_a v_b pair STAGED BY TMA TENSOR TILES, for the physical regime |shift| < 1 cell in both
// dimensions (every lane's cell offsets m1 in {0, n1-1}, m2 in {0, n2-1}; checked per block).
// f viewed as [outer2][N_k2][N_k1][inner1].  A block owns W = 32 inner1 columns (lanes) x C1 = 4
// k1-cells and walks the k2 line.  Per k2-cell it stages the C1 + 2 k1-cells c1_0-1 .. c1_0+C1 -- BOTH
// neighbours, so a lane may look left (m1 = n1-1) or right (m1 = 0) independently of the others
// (the field changes sign every N_1/2 columns of the flattened x index) -- as one TMA box
// [O][O][W] per k1-cell into a ring; stage j holds k2-cell j-1, a lane with m2 = n2-1 consumes it
// at its local step j, a lane with m2 = 0 one iteration later.  Thread (col, t1) keeps its O x O
// window along k2; the first swept cell closes the periodic line.  No raw-value registers, loads
// asynchronous and shared by the block.  A block that sees any other offset reads its raw values
// straight from global memory (same arithmetic).
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(128)
sweep_vpair_tile_kernel(const __grid_constant__ CUtensorMap tmap, const T *__restrict__ in, T *__restrict__ out,
                        long inner1, int n1, int n2, long outer2,
                        const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                        const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2) {
    constexpr int W = 32, C1 = 4, NS = 3;
    constexpr int CELL = O * O * W;                          // elements of one (k2-cell, k1-cell) box
    constexpr int STAGE = (C1 + 2) * CELL;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full[NS];
    T *ring = reinterpret_cast<T *>(smem_raw);

    const long tiles_x = inner1 / W;
    const int groups1 = n1 / C1;
    long b = blockIdx.x;
    const int g1 = (int)(b % groups1); b /= groups1;
    const long tx = b % tiles_x;
    const long oo2 = b / tiles_x;
    const int tid = threadIdx.x, col = tid % W, t1 = tid / W;
    const int c1 = g1 * C1 + t1;
    const long ii = tx * W + col;
    const long s1 = inner1, s2 = (long)n1 * O * inner1;      // element strides of k1 / k2 nodes
    const long plane = oo2 * (long)n2 * O * s2 + ii;
    const long lin0 = plane + (long)c1 * O * s1;
    const long q1 = (lin0 / qdiv1) % qmod1, q2 = (lin0 / qdiv2) % qmod2;

    T A1[O * O], B1[O * O], A2[O * O], B2[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    const bool small = __syncthreads_and((m1 == 0 || m1 == n1 - 1) && (m2 == 0 || m2 == n2 - 1)) != 0;

    int sa = c1 + m1; if (sa >= n1) sa -= n1;                // global path: this thread's k1 source cells
    int sb = sa + 1; if (sb == n1) sb = 0;
    const int la = t1 + (m1 == 0 ? 1 : 0);                   // staged path: block-local index of source cell i*
    const int late = (m2 == 0) ? 1 : 0;                      // staged path: consumes stage j at local step j - late
    // a tile without a sign change of the field needs only one neighbour cell (5 boxes instead of 6)
    const bool needL1 = __syncthreads_or(m1 != 0) != 0, needR1 = __syncthreads_or(m1 == 0) != 0;
    const int nboxes = C1 + (needL1 ? 1 : 0) + (needR1 ? 1 : 0);

    auto issue = [&](int j) {                                // stage j <-> k2-cell (j - 1) mod n2
        int cell2 = j - 1;
        if (cell2 < 0) cell2 += n2;
        if (cell2 >= n2) cell2 -= n2;
        const int slot = j % NS;
        mbar_expect_tx(&full[slot], (uint32_t)(nboxes * CELL * sizeof(T)));
        const uint64_t pol = policy_evict_first();
#pragma unroll
        for (int cc = 0; cc < C1 + 2; ++cc) {
            if ((cc == 0 && !needL1) || (cc == C1 + 1 && !needR1)) continue;
            int cell1 = g1 * C1 - 1 + cc;
            if (cell1 < 0) cell1 += n1;
            if (cell1 >= n1) cell1 -= n1;
            tma_load_4d_hint(ring + (size_t)slot * STAGE + (size_t)cc * CELL, &tmap, (int)(tx * W), cell1 * O, cell2 * O,
                             (int)oo2, &full[slot], pol);
        }
    };
    // k1-swept values of this thread's cell: from stage slot (staged) ...
    auto k1_staged = [&](int slot, T (&w)[O][O]) {
        const T *st = ring + (size_t)slot * STAGE + col;
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2) {
            T r0[O], r1[O];
#pragma unroll
            for (int l = 0; l < O; ++l) {
                r0[l] = st[((la * O + l2) * O + l) * W];
                r1[l] = st[(((la + 1) * O + l2) * O + l) * W];
            }
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
        }
    };
    // ... or from global memory for source k2-cell `cell2`
    auto k1_global = [&](int cell2, T (&w)[O][O]) {
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2) {
            const T *row = in + plane + ((long)cell2 * O + l2) * s2;
            T r0[O], r1[O];
#pragma unroll
            for (int l = 0; l < O; ++l) {
                r0[l] = row[((long)sa * O + l) * s1];
                r1[l] = row[((long)sb * O + l) * s1];
            }
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
        }
    };
    auto emit = [&](int i2, const T (&w0)[O][O], const T (&w1)[O][O]) {
        T *dst = out + lin0 + (long)i2 * O * s2;
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a0[O], a1[O];
#pragma unroll
                for (int l = 0; l < O; ++l) { a0[l] = w0[l][j1]; a1[l] = w1[l][j1]; }
                __stcs(dst + (long)j2 * s2 + (long)j1 * s1, chain<T, O>(A2, B2, j2, a0, a1));
            }
    };
    auto copy = [&](T (&d)[O][O], const T (&s)[O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int c = 0; c < O; ++c) d[a][c] = s[a][c];
    };

    T wfirst[O][O], w0[O][O], w1[O][O];
    if (small) {
        if (tid == 0)
            for (int j = 0; j < NS && j <= n2; ++j) issue(j);
        for (int j = 0; j <= n2 + 1; ++j) {
            const int t = j - late;                          // this thread's local step
            if (j <= n2) {
                mbar_wait(&full[j % NS], (uint32_t)((j / NS) & 1));
                if (t == 0) {
                    k1_staged(j % NS, wfirst);
                    copy(w0, wfirst);
                } else if (t >= 1 && t <= n2 - 1) {
                    k1_staged(j % NS, w1);
                    emit(t - 1, w0, w1);
                    copy(w0, w1);
                }
            }
            if (t == n2) emit(n2 - 1, w0, wfirst);           // closes the periodic line
            if (j <= n2) {
                __syncthreads();                             // everyone is done with this slot
                if (tid == 0 && j + NS <= n2) issue(j + NS);
            }
        }
    } else {
        for (int t = 0; t <= n2; ++t) {
            int cell2 = m2 + t;
            if (cell2 >= n2) cell2 -= n2;
            if (t == 0) {
                k1_global(cell2, wfirst);
                copy(w0, wfirst);
            } else if (t <= n2 - 1) {
                k1_global(cell2, w1);
                emit(t - 1, w0, w1);
                copy(w0, w1);
            } else {
                emit(n2 - 1, w0, wfirst);
            }
        }
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// v_a v_b v_c triple STAGED BY TMA TENSOR TILES for |shift| < 1 cell in all three dimensions (the
// 3+3 D step), one level up from sweep_vpair_tile_kernel.  f viewed as
// [outer3][N_k3][N_k2][N_k1][inner1].  A block owns W = 32 inner1 columns (lanes) x C1 = 4 k1-cells
// x C2 = 4 k2-cells (512 threads) and walks the k3 line; per k3-cell it stages the (C1+2) x (C2+2)
// cell pairs (both neighbours in k1 and in k2) as one 5-D TMA box [O][O][O][W] each into a 2-deep
// ring.  Thread (col, t1, t2) reads its 2 x 2 source cells with its own left/right choices, keeps
// its O^3 window along k3, consumes stage j at local step j (m3 = n3-1) or j-1 (m3 = 0).
// Bit-identical to the three sweeps; per-block fallback to direct global reads otherwise.
// ------------------------------------------------------------------------------------------
// W = columns (lanes along inner1) per block, C2 = owned k2-cells (C1 = 4 k1-cells), NS = ring depth, MINB =
// blocks per SM the register allocation is bounded for; block = W x 4 x C2 threads.
// ncu (profiles/ncu_vtile_r2.md): no unit is saturated (issue 33 %, fp64 26 %, LSU 26 %, L2 35 %, DRAM 58 %);
// 20 % of the warp samples wait for a stage to land and 15 % at the block barrier that recycles a slot: every
// warp of the single resident block is in the same phase at the same time.  DRIFT replaces that barrier by
// per-slot "empty" mbarriers counted in warps: a warp releases a slot as soon as it has read its raw values and
// goes on; only warp 0 (which issues the copies) waits for the others, one iteration later, before it refills.
template <typename T, int O, int W, int C2, int NS, int MINB, bool DRIFT, bool EVF = true>
__global__ void __launch_bounds__(W * 4 * C2, MINB)
sweep_vtriple_tile_kernel(const __grid_constant__ CUtensorMap tmap, const T *__restrict__ in, T *__restrict__ out,
                          long inner1, int n1, int n2, int n3, long outer3,
                          const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                          const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                          const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    constexpr int C1 = 4;
    constexpr int NBOX = (C1 + 2) * (C2 + 2);
    constexpr int NWARP = W * C1 * C2 / 32;
    constexpr int CELL = O * O * O * W;                      // elements of one (k3, k2, k1)-cell box
    constexpr int STAGE = NBOX * CELL;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full[NS], empty[NS];
    T *ring = reinterpret_cast<T *>(smem_raw);

    const long tiles_x = inner1 / W;
    const int groups1 = n1 / C1, groups2 = n2 / C2;
    long b = blockIdx.x;
    const int g1 = (int)(b % groups1); b /= groups1;
    const int g2 = (int)(b % groups2); b /= groups2;
    const long tx = b % tiles_x;
    const long oo3 = b / tiles_x;
    const int tid = threadIdx.x, col = tid % W, t1 = (tid / W) % C1, t2 = tid / (W * C1);
    const int warp = tid >> 5, lane = tid & 31;
    const int c1 = g1 * C1 + t1, c2 = g2 * C2 + t2;
    const long ii = tx * W + col;
    const long s1 = inner1, s2 = (long)n1 * O * s1, s3 = (long)n2 * O * s2;
    const long plane = oo3 * (long)n3 * O * s3 + ii;
    const long lin0 = plane + (long)c1 * O * s1 + (long)c2 * O * s2;
    const long q1 = (lin0 / qdiv1) % qmod1, q2 = (lin0 / qdiv2) % qmod2, q3 = (lin0 / qdiv3) % qmod3;

    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NWARP); }
    }
    const bool small = __syncthreads_and((m1 == 0 || m1 == n1 - 1) && (m2 == 0 || m2 == n2 - 1) &&
                                         (m3 == 0 || m3 == n3 - 1)) != 0;
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;             // global path
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    int sa2 = c2 + m2; if (sa2 >= n2) sa2 -= n2;
    int sb2 = sa2 + 1; if (sb2 == n2) sb2 = 0;
    const int la = t1 + (m1 == 0 ? 1 : 0), lb = t2 + (m2 == 0 ? 1 : 0);   // staged path: local source cells
    const int late = (m3 == 0) ? 1 : 0;
    // which neighbour columns / rows of cells the block really needs (a tile without a sign change of
    // the field needs only one side)
    const bool needL1 = __syncthreads_or(m1 != 0) != 0, needR1 = __syncthreads_or(m1 == 0) != 0;
    const bool needL2 = __syncthreads_or(m2 != 0) != 0, needR2 = __syncthreads_or(m2 == 0) != 0;
    const int nboxes = (C1 + (needL1 ? 1 : 0) + (needR1 ? 1 : 0)) * (C2 + (needL2 ? 1 : 0) + (needR2 ? 1 : 0));

    auto issue = [&](int j) {                                // stage j <-> k3-cell (j - 1) mod n3; warp 0 calls
        int cell3 = j - 1;
        if (cell3 < 0) cell3 += n3;
        if (cell3 >= n3) cell3 -= n3;
        const int slot = j % NS;
        if (lane == 0) mbar_expect_tx(&full[slot], (uint32_t)(nboxes * CELL * sizeof(T)));
        const uint64_t pol = EVF ? policy_evict_first() : policy_evict_last();
#pragma unroll
        for (int bx = lane; bx < NBOX; bx += 32) {
            const int ca = bx % (C1 + 2), cb = bx / (C1 + 2);
            if ((ca > 0 || needL1) && (ca < C1 + 1 || needR1) && (cb > 0 || needL2) && (cb < C2 + 1 || needR2)) {
                int cell1 = g1 * C1 - 1 + ca;
                if (cell1 < 0) cell1 += n1;
                if (cell1 >= n1) cell1 -= n1;
                int cell2 = g2 * C2 - 1 + cb;
                if (cell2 < 0) cell2 += n2;
                if (cell2 >= n2) cell2 -= n2;
                tma_load_5d_hint(ring + (size_t)slot * STAGE + (size_t)bx * CELL, &tmap, (int)(tx * W), cell1 * O,
                                 cell2 * O, cell3 * O, (int)oo3, &full[slot], pol);
            }
        }
    };
    auto k12_staged = [&](int slot, T (&w)[O][O][O]) {
        const T *st = ring + (size_t)slot * STAGE + col;
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[2][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    const T *p0 = st + (size_t)((lb + e2) * (C1 + 2) + la) * CELL + ((l3 * O + l2) * O) * W;
                    T r0[O], r1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { r0[l] = p0[l * W]; r1[l] = p0[CELL + l * W]; }
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };
    auto k12_global = [&](int cell3, T (&w)[O][O][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            const T *row = in + plane + ((long)cell3 * O + l3) * s3;
            T tk[2][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    const T *p = row + ((long)(e2 ? sb2 : sa2) * O + l2) * s2;
                    T r0[O], r1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { r0[l] = p[((long)sa1 * O + l) * s1]; r1[l] = p[((long)sb1 * O + l) * s1]; }
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };
    // The k3 rule in two halves (same operations in the same order as chain<>: one multiply and O-1 FMAs with
    // the A3 row on the older cell, then O FMAs with the B3 row on the newer one).  The A-half is taken as soon
    // as a cell's (k1,k2)-swept values exist and replaces them as the thread's state, so no window is copied.
    auto a_half = [&](const T (&w)[O][O][O], T (&acc)[O][O][O]) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                    for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                    acc[j3][j2][j1] = a;
                }
    };
    auto b_half_store = [&](int i3, const T (&acc)[O][O][O], const T (&w)[O][O][O]) {
        T *dst = out + lin0 + (long)i3 * O * s3;
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = acc[j3][j2][j1];
#pragma unroll
                    for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                    __stcs(dst + (long)j3 * s3 + (long)j2 * s2 + (long)j1 * s1, a);
                }
    };

    T wfirst[O][O][O], acc[O][O][O], w1[O][O][O];
    if (small) {
        if (warp == 0)
            for (int j = 0; j < NS && j <= n3; ++j) issue(j);
        for (int j = 0; j <= n3 + 1; ++j) {
            const int t = j - late;
            bool pending = false;
            if (j <= n3) {
                if constexpr (DRIFT) {
                    // refill the slot of stage j-1 (released by every warp during the previous iteration)
                    if (warp == 0 && j >= 1 && j - 1 + NS <= n3) {
                        mbar_wait(&empty[(j - 1) % NS], (uint32_t)(((j - 1) / NS) & 1));
                        issue(j - 1 + NS);
                    }
                }
                mbar_wait(&full[j % NS], (uint32_t)((j / NS) & 1));
                if (t == 0) {
                    k12_staged(j % NS, wfirst);
                } else if (t >= 1 && t <= n3 - 1) {
                    k12_staged(j % NS, w1);
                    pending = true;
                }
                // the slot is free as soon as its raw values have been read: released BEFORE the k3 rule and
                // the stores, so that the copy engine works during them
                if constexpr (DRIFT) {
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&empty[j % NS]);
                } else {
                    __syncthreads();
                    if (warp == 0 && j + NS <= n3) issue(j + NS);
                }
            }
            if (t == 0) a_half(wfirst, acc);
            if (pending) {
                b_half_store(t - 1, acc, w1);
                a_half(w1, acc);
            }
            if (t == n3) b_half_store(n3 - 1, acc, wfirst);  // closes the periodic line
        }
    } else {
        for (int t = 0; t <= n3; ++t) {
            int cell3 = m3 + t;
            if (cell3 >= n3) cell3 -= n3;
            if (t == 0) {
                k12_global(cell3, wfirst);
                a_half(wfirst, acc);
            } else if (t <= n3 - 1) {
                k12_global(cell3, w1);
                b_half_store(t - 1, acc, w1);
                a_half(w1, acc);
            } else {
                b_half_store(n3 - 1, acc, wfirst);
            }
        }
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// S:8(f) NEXT-1, the rest of it: rho ACCUMULATED IN THE SWEEP THAT PRECEDES IT ("compute rho" follows the
// x half-step).  x_1 x_2 pair + rho for d_x = 2.
//
// sweep_xpair_plane_kernel gives one block a whole (x_1,x_2) plane at fixed v; summing over v inside the
// kernel needs accumulators for every x-node a thread writes.  Here a block owns a RANGE of C2R x_2-cells
// (group g) and walks a contiguous chunk of planes (velocity nodes, the slow index): thread c1 keeps
// C2R * O * O fp64 accumulators (fp64 for both storage types) for its x-nodes and adds W_v * f_new
// plane after plane in ascending v -- the split structure of the stand-alone rho pass with chunks as splits.
// Per plane the block streams the C2R + 1 slabs (k2-cells) its outputs need -- the extra one is the k2
// neighbour, an L2 hit for the group next door -- through the same cp.async.bulk ring, which never drains
// between planes.  The grid is ONE wave of equal blocks (groups x chunks = resident blocks), so the
// partials part[chunk][x] are a fraction (chunks / V) of one write of f and the order of every sum is fixed.
// f is bit-identical to the two separate sweeps; rho = -(pass over the chunks) as in vsum_final_kernel.
// ------------------------------------------------------------------------------------------
template <typename T, int O, int C2R>
__global__ void __launch_bounds__(256)
sweep_xpair_rho_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, long planes, int nchunk,
                       const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long pdiv1, long pmod1,
                       const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long pdiv2, long pmod2,
                       const double *__restrict__ Wv, double *__restrict__ part) {
    // shift index of plane p (a velocity node): q_i = (p / pdiv_i) % pmod_i, kept incrementally (no divisions
    // in the loops: thread 0's producer path holds up the whole block at the next barrier)
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 8;                                   // ring depth
    constexpr int NCO = 4 * O * O;                           // A1 | B1 | A2 | B2
    __shared__ __align__(8) uint64_t full[NS];
    __shared__ T s_co[2][NCO];                               // coefficients of the current / next plane
    __shared__ int s_m1[2];
    __shared__ double s_wv[2];
    const long N1 = (long)n1 * O;
    const long slab = O * N1;                                // elements per k2-cell of one plane
    const uint32_t slab_bytes = (uint32_t)((size_t)slab * sizeof(T));
    const uint32_t slot_stride = (slab_bytes + 127u) & ~127u;
    const int G = (n2 + C2R - 1) / C2R;
    const int g = blockIdx.x % G;
    const long chunk = blockIdx.x / G;
    const long p0 = chunk * planes / nchunk, p1 = (chunk + 1) * planes / nchunk;
    const int i0 = g * C2R;                                  // first owned k2-cell
    const int ncell = (n2 - i0 < C2R) ? n2 - i0 : C2R;       // owned cells (ragged last group)
    const int L = ncell + 1;                                 // slabs per plane
    const long total = (p1 - p0) * L;
    const int tid = threadIdx.x;
    const int c1 = tid;
    const bool active = c1 < n1;
    const long plane_elems = (long)n2 * slab;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    // consumer counters of plane p0
    long q1 = (p0 / pdiv1) % pmod1, r1 = p0 % pdiv1, q2 = (p0 / pdiv2) % pmod2, r2 = p0 % pdiv2;
    auto fetch_coef = [&](int e, long qa, long qb) -> T {    // element e of [A1 | B1 | A2 | B2] of a plane
        return e < 2 * O * O ? ab1[(long)e * count1 + qa] : ab2[(long)(e - 2 * O * O) * count2 + qb];
    };
    for (int e = tid; e < NCO; e += blockDim.x) s_co[0][e] = fetch_coef(e, q1, q2);
    if (tid == 0) { s_m1[0] = mtab1[q1]; s_wv[0] = p0 < p1 ? Wv[p0] : 0.0; }
    __syncthreads();
    // producer state (thread 0): next slab to issue = slab kp of plane ip; m2 of that plane and of the next
    long ip = p0, pq2 = q2, pr2 = r2;
    int kp = 0, pslot = 0;
    long issued = 0;
    int m2p = 0, m2n = 0;
    if (tid == 0) m2n = mtab2[pq2];
    auto issue = [&]() {
        if (kp == 0) {                                       // entering plane ip: its m2 was fetched a plane ago
            m2p = m2n;
            if (++pr2 == pdiv2) { pr2 = 0; if (++pq2 == pmod2) pq2 = 0; }
            m2n = mtab2[pq2];
        }
        int cell = i0 + m2p + kp;
        if (cell >= n2) cell -= n2;
        if (cell >= n2) cell -= n2;
        mbar_expect_tx(&full[pslot], slab_bytes);
        bulk_g2s(smem_raw + pslot * slot_stride, in + ip * plane_elems + (long)cell * slab, slab_bytes, &full[pslot]);
        ++issued;
        if (++pslot == NS) pslot = 0;
        if (++kp == L) { kp = 0; ++ip; }
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < total; ++j) issue();

    double racc[C2R][O][O];
#pragma unroll
    for (int a = 0; a < C2R; ++a)
#pragma unroll
        for (int b = 0; b < O; ++b)
#pragma unroll
            for (int d = 0; d < O; ++d) racc[a][b][d] = 0.0;

    int slot = 0;
    uint32_t phase = 0;
    T *dst_plane = out + p0 * plane_elems + (long)i0 * slab + (long)c1 * O;
    for (long pl = p0; pl < p1; ++pl) {
        const int buf = (int)((pl - p0) & 1);
        T A1[O * O], B1[O * O], A2[O * O], B2[O * O];
#pragma unroll
        for (int e = 0; e < O * O; ++e) {
            A1[e] = s_co[buf][e]; B1[e] = s_co[buf][O * O + e];
            A2[e] = s_co[buf][2 * O * O + e]; B2[e] = s_co[buf][3 * O * O + e];
        }
        const int m1 = s_m1[buf];
        const double wv = s_wv[buf];
        // next plane's coefficients: loads issued now, stored to the other buffer before the plane's last barrier
        if (++r1 == pdiv1) { r1 = 0; if (++q1 == pmod1) q1 = 0; }
        if (++r2 == pdiv2) { r2 = 0; if (++q2 == pmod2) q2 = 0; }
        const bool more = pl + 1 < p1;
        T pre = T(0);
        int pre_m = 0;
        double pre_w = 0.0;
        if (more) {
            if (tid < NCO) pre = fetch_coef(tid, q1, q2);
            if (tid == 0) { pre_m = mtab1[q1]; pre_w = Wv[pl + 1]; }
        }
        int sa1 = (active ? c1 : 0) + m1; if (sa1 >= n1) sa1 -= n1;
        int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
        const int oa = sa1 * O, ob = sb1 * O;
        T acc[O][O];                                         // A-half of the k2 rule on the older cell
#pragma unroll
        for (int k = 0; k <= C2R; ++k) {
            if (k < L) {
                mbar_wait(&full[slot], phase);
                T w[O][O];                                   // k1-swept values of this thread's cell, w[l2][j1]
                if (active) {
                    const T *sl = reinterpret_cast<const T *>(smem_raw + slot * slot_stride);
#pragma unroll
                    for (int l2 = 0; l2 < O; ++l2) {
                        T r0[O], r1v[O];
                        load_cell<T, O>(sl + l2 * N1 + oa, r0);
                        load_cell<T, O>(sl + l2 * N1 + ob, r1v);
#pragma unroll
                        for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0, r1v);
                    }
                }
                if (k == L - 1 && more) {                    // hand the next plane's coefficients over
                    if (tid < NCO) s_co[buf ^ 1][tid] = pre;
                    if constexpr (NCO > 32) {                // blocks may be as small as one warp
                        for (int e = tid + blockDim.x; e < NCO; e += blockDim.x) s_co[buf ^ 1][e] = fetch_coef(e, q1, q2);
                    }
                    if (tid == 0) { s_m1[buf ^ 1] = pre_m; s_wv[buf ^ 1] = pre_w; }
                }
                __syncthreads();                             // slab consumed: refill the slot before the k2 rule
                if (tid == 0 && issued < total) issue();
                if (++slot == NS) { slot = 0; phase ^= 1u; }
                if (active) {
                    if (k > 0) {                             // B-half, store, rho
                        T *dst = dst_plane + (long)(k - 1) * slab;
#pragma unroll
                        for (int j2 = 0; j2 < O; ++j2) {
                            T res[O];
#pragma unroll
                            for (int j1 = 0; j1 < O; ++j1) {
                                T a = acc[j2][j1];
#pragma unroll
                                for (int l = 0; l < O; ++l) a = fma_t<T>(B2[j2 * O + l], w[l][j1], a);
                                res[j1] = a;
                                racc[k > 0 ? k - 1 : 0][j2][j1] += wv * (double)a;
                            }
                            T *p = dst + (long)j2 * N1;
                            if constexpr (O % 2 == 0) {
                                using V2 = Vec<T, 2>;
#pragma unroll
                                for (int j1 = 0; j1 < O; j1 += 2) {
                                    V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                                    *reinterpret_cast<V2 *>(p + j1) = vv;
                                }
                            } else {
#pragma unroll
                                for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
                            }
                        }
                    }
                    if (k < C2R) {                           // A-half for the next cell
#pragma unroll
                        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                            for (int j1 = 0; j1 < O; ++j1) {
                                T a = mul_t<T>(A2[j2 * O], w[0][j1]);
#pragma unroll
                                for (int l = 1; l < O; ++l) a = fma_t<T>(A2[j2 * O + l], w[l][j1], a);
                                acc[j2][j1] = a;
                            }
                    }
                }
            }
        }
        dst_plane += plane_elems;
    }
    if (active) {
        double *pr = part + chunk * plane_elems;             // row `chunk` of [nchunk][X], X = n2 * slab
#pragma unroll
        for (int k = 0; k < C2R; ++k)
            if (k < ncell)
#pragma unroll
                for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1)
                        pr[((long)(i0 + k) * O + j2) * N1 + (long)c1 * O + j1] = racc[k][j2][j1];
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// x_1 x_2 x_3 triple + rho for d_x = 3 with a small x-grid (the 3+3 D step): sweep_xtriple_plane_kernel with
// the v-sum inside.  A block owns a range of C3R x_3-cells (group g) and walks a contiguous chunk of
// velocity nodes; per node it streams the C3R + 1 slabs (x_3-cells, each one contiguous O * N2 * N1 values)
// its outputs need through the cp.async.bulk ring.  The accumulators -- C3R * O^3 fp64 per thread -- do not
// fit the register file next to the O^3 window and the six A,B matrices, so they live in SHARED memory, each
// word owned by exactly one thread (no atomics, fixed order: ascending v).  One wave of equal blocks; the
// partials part[chunk][x] are chunks / V of one write of f.  f is bit-identical to the three sweeps.
// ------------------------------------------------------------------------------------------
template <typename T, int O, int C3R, int NS>
__global__ void __launch_bounds__(512, 1)
sweep_xtriple_rho_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int n3, long nv, int nchunk,
                         const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                         const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                         const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3,
                         const double *__restrict__ Wv, double *__restrict__ part) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full[NS];
    const long N1 = (long)n1 * O, N2 = (long)n2 * O;
    const long slab = O * N2 * N1;                           // elements per k3-cell
    const size_t slab_bytes = (size_t)slab * sizeof(T);
    const size_t slot_stride = (slab_bytes + 127) & ~(size_t)127;
    double *racc = reinterpret_cast<double *>(smem_raw + NS * slot_stride);   // [C3R][slab]
    const int G = (n3 + C3R - 1) / C3R;
    const int g = blockIdx.x % G;
    const long chunk = blockIdx.x / G;
    const long v0 = chunk * nv / nchunk, v1 = (chunk + 1) * nv / nchunk;
    const int i0 = g * C3R;
    const int ncell = (n3 - i0 < C3R) ? n3 - i0 : C3R;
    const int L = ncell + 1;
    const long total = (v1 - v0) * L;
    const int tid = threadIdx.x;
    const int c1 = tid % n1, c2 = tid / n1;
    const bool active = c2 < n2;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    for (long e = tid; e < (long)C3R * slab; e += blockDim.x) racc[e] = 0.0;
    __syncthreads();
    long ip = v0;
    int kp = 0, m3p = 0, m3n = 0;
    long issued = 0;
    if (tid == 0 && v0 < v1) m3n = mtab3[((v0 * n3 * slab) / qdiv3) % qmod3];
    auto issue = [&]() {
        if (kp == 0) {                                       // m3 of node ip was fetched a node ago
            m3p = m3n;
            m3n = mtab3[(((ip + 1 < nv ? ip + 1 : ip) * n3 * slab) / qdiv3) % qmod3];
        }
        int cell = i0 + m3p + kp;
        if (cell >= n3) cell -= n3;
        if (cell >= n3) cell -= n3;
        const int slot = (int)(issued % NS);
        mbar_expect_tx(&full[slot], (uint32_t)slab_bytes);
        bulk_g2s(smem_raw + slot * slot_stride, in + (ip * n3 + cell) * slab, (uint32_t)slab_bytes, &full[slot]);
        ++issued;
        if (++kp == L) { kp = 0; ++ip; }
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < total; ++j) issue();

    int slot = 0;
    uint32_t phase = 0;
    for (long v = v0; v < v1; ++v) {
        const long base = v * (long)n3 * slab;
        const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2, q3 = (base / qdiv3) % qmod3;
        T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
        for (int e = 0; e < O * O; ++e) {
            A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
            A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
            A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
        }
        const int m1 = mtab1[q1], m2 = mtab2[q2];
        const double wv = Wv[v];
        int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
        int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
        int sa2 = (active ? c2 : 0) + m2; if (sa2 >= n2) sa2 -= n2;
        int sb2 = sa2 + 1; if (sb2 == n2) sb2 = 0;
        const int off[2][2] = {{(int)(sa2 * O * N1 + sa1 * O), (int)(sa2 * O * N1 + sb1 * O)},
                               {(int)(sb2 * O * N1 + sa1 * O), (int)(sb2 * O * N1 + sb1 * O)}};
        T acc[O][O][O];                                      // A-half of the k3 rule on the older cell
#pragma unroll 1
        for (int k = 0; k < L; ++k) {
            mbar_wait(&full[slot], phase);
            T w[O][O][O];                                    // (k1,k2)-swept values of this thread's cell pair
            if (active) {
                const T *sl = reinterpret_cast<const T *>(smem_raw + slot * slot_stride);
#pragma unroll
                for (int l3 = 0; l3 < O; ++l3) {
                    T tk[2][O][O];
#pragma unroll
                    for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                        for (int l2 = 0; l2 < O; ++l2) {
                            T r0[O], r1[O];
                            load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][0] + l2 * N1, r0);
                            load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][1] + l2 * N1, r1);
#pragma unroll
                            for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                        }
#pragma unroll
                    for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                        for (int j1 = 0; j1 < O; ++j1) {
                            T a0[O], a1[O];
#pragma unroll
                            for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                            w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                        }
                }
            }
            __syncthreads();                                 // slab consumed: refill the slot before the k3 rule
            if (tid == 0 && issued < total) issue();
            if (++slot == NS) { slot = 0; phase ^= 1u; }
            if (active) {
                if (k > 0) {                                 // B-half, store, rho
                    const long cell_off = (long)c2 * O * N1 + (long)c1 * O;
                    T *dst = out + base + (long)(i0 + k - 1) * slab + cell_off;
                    double *ra = racc + (long)(k - 1) * slab + cell_off;
#pragma unroll
                    for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
                        for (int j2 = 0; j2 < O; ++j2) {
                            T res[O];
#pragma unroll
                            for (int j1 = 0; j1 < O; ++j1) {
                                T a = acc[j3][j2][j1];
#pragma unroll
                                for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                                res[j1] = a;
                            }
                            const long ro = (long)j3 * N2 * N1 + (long)j2 * N1;
                            T *p = dst + ro;
                            double *pa = ra + ro;
                            if constexpr (O % 2 == 0) {
                                using V2 = Vec<T, 2>;
                                using D2 = Vec<double, 2>;
#pragma unroll
                                for (int j1 = 0; j1 < O; j1 += 2) {
                                    V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                                    *reinterpret_cast<V2 *>(p + j1) = vv;
                                    D2 r = *reinterpret_cast<D2 *>(pa + j1);
                                    r.v[0] += wv * (double)res[j1]; r.v[1] += wv * (double)res[j1 + 1];
                                    *reinterpret_cast<D2 *>(pa + j1) = r;
                                }
                            } else {
#pragma unroll
                                for (int j1 = 0; j1 < O; ++j1) { p[j1] = res[j1]; pa[j1] += wv * (double)res[j1]; }
                            }
                        }
                }
                if (k + 1 < L) {                             // A-half for the next cell
#pragma unroll
                    for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
                        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                            for (int j1 = 0; j1 < O; ++j1) {
                                T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                                for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                                acc[j3][j2][j1] = a;
                            }
                }
            }
        }
    }
    __syncthreads();
    double *pr = part + chunk * (long)n3 * slab + (long)i0 * slab;     // row `chunk` of [nchunk][X], X = n3 * slab
    for (long e = tid; e < (long)ncell * slab; e += blockDim.x) pr[e] = racc[e];
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// The x-group applied TWICE in one pass over f.  Consecutive Strang steps end and begin with the same
// x half-step, and nothing separates the two when no invariant is written in between: x(tau) x(tau) is
// then one read and one write of f instead of two of each.  NOT x(2 tau): each application is the full O7 chain
// of the single sweeps, so the result is bit-identical to calling the x-group twice (sldg_step_n relies on it).
//
// x_1 x_2 pair, one block per (x_1,x_2) plane as sweep_xpair_plane_kernel: the first application's output cell
// (O x O values per thread) goes to a slab-sized shared-memory buffer instead of global memory; after a barrier
// every thread reads its two x_1 source cells of it and runs the second application with a second window.  The
// shifts, A and B are those of the first application (same tau, same v).  Output cells leave in the order the
// second window closes them: cell (i - 1 - m2) mod n2 when the first application has produced its cell i.
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(256)
sweep_xpair_plane2_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2,
                          const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                          const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 4;                                   // ring depth
    __shared__ __align__(8) uint64_t full[NS];
    const long N1 = (long)n1 * O;
    const long slab = O * N1;                                // elements per k2-cell of one plane
    const size_t slab_bytes = (size_t)slab * sizeof(T);
    const size_t slot_stride = (slab_bytes + 127) & ~(size_t)127;
    T *tbuf = reinterpret_cast<T *>(smem_raw + NS * slot_stride);   // the first application's current output cell
    const long base = (long)blockIdx.x * n2 * slab;          // planes are contiguous
    const int tid = threadIdx.x;
    const int c1 = tid;
    const bool active = c1 < n1;

    const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2];
    int sa1 = (active ? c1 : 0) + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    __syncthreads();
    auto issue = [&](int j) {                                // slab j <-> source k2-cell (m2 + j) mod n2
        int cell = m2 + j;
        if (cell >= n2) cell -= n2;
        const int slot = j % NS;
        mbar_expect_tx(&full[slot], (uint32_t)slab_bytes);
        bulk_g2s(smem_raw + slot * slot_stride, in + base + (long)cell * slab, (uint32_t)slab_bytes, &full[slot]);
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n2; ++j) issue(j);

    auto k1_from = [&](const T *sl, T (&w)[O][O]) {          // w[l2][j1]: k1 rule on this thread's two source cells
#pragma unroll
        for (int l2 = 0; l2 < O; ++l2) {
            T r0[O], r1[O];
            load_cell<T, O>(sl + l2 * N1 + (long)sa1 * O, r0);
            load_cell<T, O>(sl + l2 * N1 + (long)sb1 * O, r1);
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) w[l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
        }
    };
    auto a_half = [&](const T (&w)[O][O], T (&acc)[O][O]) {  // k2 rule, A row on the older cell
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a = mul_t<T>(A2[j2 * O], w[0][j1]);
#pragma unroll
                for (int l = 1; l < O; ++l) a = fma_t<T>(A2[j2 * O + l], w[l][j1], a);
                acc[j2][j1] = a;
            }
    };
    auto b_half = [&](const T (&acc)[O][O], const T (&w)[O][O], T (&res)[O][O]) {   // ... B row on the newer one
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a = acc[j2][j1];
#pragma unroll
                for (int l = 0; l < O; ++l) a = fma_t<T>(B2[j2 * O + l], w[l][j1], a);
                res[j2][j1] = a;
            }
    };
    auto put = [&](T *dst_cell, long row_stride, const T (&res)[O][O]) {           // O rows of O values
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2) {
            T *p = dst_cell + (long)j2 * row_stride;
            if constexpr (O % 2 == 0) {
                using V2 = Vec<T, 2>;
#pragma unroll
                for (int j1 = 0; j1 < O; j1 += 2) {
                    V2 vv; vv.v[0] = res[j2][j1]; vv.v[1] = res[j2][j1 + 1];
                    *reinterpret_cast<V2 *>(p + j1) = vv;
                }
            } else {
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j2][j1];
            }
        }
    };

    T wfirst[O][O], acc1[O][O], bfirst[O][O], acc2[O][O];
    // second application on the first one's output cell i (in tbuf, visible to all threads)
    auto second = [&](int i) {
        if (!active) return;
        T b[O][O];
        k1_from(tbuf, b);
        if (i == 0) {
#pragma unroll
            for (int a = 0; a < O; ++a)
#pragma unroll
                for (int d = 0; d < O; ++d) bfirst[a][d] = b[a][d];
        } else {
            T res[O][O];
            b_half(acc2, b, res);
            int cell = i - 1 - m2;
            if (cell < 0) cell += n2;
            put(out + base + (long)cell * slab + (long)c1 * O, N1, res);
        }
        a_half(b, acc2);
    };

    for (int j = 0; j < n2; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        T w[O][O];
        if (active) k1_from(reinterpret_cast<const T *>(smem_raw + slot * slot_stride), w);
        __syncthreads();                                     // slab consumed (and tbuf no longer read)
        if (tid == 0 && j + NS < n2) issue(j + NS);
        if (j == 0) {
            if (active) {
#pragma unroll
                for (int a = 0; a < O; ++a)
#pragma unroll
                    for (int d = 0; d < O; ++d) wfirst[a][d] = w[a][d];
                a_half(w, acc1);
            }
        } else {
            if (active) {
                T res[O][O];
                b_half(acc1, w, res);                        // first application, cell j - 1
                a_half(w, acc1);
                put(tbuf + (long)c1 * O, N1, res);
            }
            __syncthreads();
            second(j - 1);
        }
    }
    __syncthreads();                                         // tbuf no longer read
    if (active) {
        T res[O][O];
        b_half(acc1, wfirst, res);                           // first application, cell n2 - 1 (closes the line)
        put(tbuf + (long)c1 * O, N1, res);
    }
    __syncthreads();
    second(n2 - 1);
    if (active) {
        T res[O][O];
        b_half(acc2, bfirst, res);                           // second application closes its line
        int cell = n2 - 1 - m2;
        if (cell < 0) cell += n2;
        put(out + base + (long)cell * slab + (long)c1 * O, N1, res);
    }
}

// x_1 x_2 x_3 triple applied twice, one block per velocity node as sweep_xtriple_plane_kernel.  The two windows'
// first cells (needed only to close the periodic lines at the very end) are parked in shared memory, so the
// register budget is that of the single application.
template <typename T, int O>
__global__ void __launch_bounds__(512, 1)
sweep_xtriple_plane2_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int n3, int tpr,
                            const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                            const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                            const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 3;
    constexpr int O3 = O * O * O;
    __shared__ __align__(8) uint64_t full[NS], tbar[2];
    const long N1 = (long)n1 * O, N2 = (long)n2 * O;
    const long slab = O * N2 * N1;                           // elements per k3-cell
    const size_t slab_bytes = (size_t)slab * sizeof(T);
    const size_t slot_stride = (slab_bytes + 127) & ~(size_t)127;
    // the first application's output cells, double-buffered: cell i is written during iteration i + 1 and read
    // during iteration i + 2, so the barrier between the two (an mbarrier counted in threads: arrive after the
    // write, wait before the read) has a whole iteration to complete and nobody stalls at it
    T *tbuf0 = reinterpret_cast<T *>(smem_raw + NS * slot_stride);
    T *park = reinterpret_cast<T *>(smem_raw + (NS + 2) * slot_stride);   // [2][O3][blockDim]
    const long v = blockIdx.x;
    const long base = v * (long)n3 * slab;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int c1r = tid % tpr, c2 = tid / tpr;               // tpr threads per row, n1 active (bank conflicts, see above)
    const bool active = c2 < n2 && c1r < n1;
    const int c1 = c1r < n1 ? c1r : 0;

    const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2, q3 = (base / qdiv3) % qmod3;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    int sa2 = (active ? c2 : 0) + m2; if (sa2 >= n2) sa2 -= n2;
    int sb2 = sa2 + 1; if (sb2 == n2) sb2 = 0;
    const int off[2][2] = {{(int)(sa2 * O * N1 + sa1 * O), (int)(sa2 * O * N1 + sb1 * O)},
                           {(int)(sb2 * O * N1 + sa1 * O), (int)(sb2 * O * N1 + sb1 * O)}};
    const long cell_off = (long)c2 * O * N1 + (long)c1 * O;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        mbar_init(&tbar[0], nthr);
        mbar_init(&tbar[1], nthr);
    }
    __syncthreads();
    auto issue = [&](int j) {                                // slab j <-> source k3-cell (m3 + j) mod n3
        int cell = m3 + j;
        if (cell >= n3) cell -= n3;
        const int slot = j % NS;
        mbar_expect_tx(&full[slot], (uint32_t)slab_bytes);
        bulk_g2s(smem_raw + slot * slot_stride, in + base + (long)cell * slab, (uint32_t)slab_bytes, &full[slot]);
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n3; ++j) issue(j);

    auto k12_from = [&](const T *sl, T (&w)[O][O][O]) {      // (k1,k2)-swept values of this thread's cell pair
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[2][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    T r0[O], r1[O];
                    load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][0] + l2 * N1, r0);
                    load_cell<T, O>(sl + l3 * N2 * N1 + off[e2][1] + l2 * N1, r1);
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };
    auto a_half = [&](const T (&w)[O][O][O], T (&acc)[O][O][O]) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                    for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                    acc[j3][j2][j1] = a;
                }
    };
    // B-half of the k3 rule and the O^3 results written as O^2 rows of O values at dst (row pitches N1, N2*N1)
    auto b_half_put = [&](const T (&acc)[O][O][O], const T (&w)[O][O][O], T *dst) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2) {
                T res[O];
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = acc[j3][j2][j1];
#pragma unroll
                    for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                    res[j1] = a;
                }
                T *p = dst + (long)j3 * N2 * N1 + (long)j2 * N1;
                if constexpr (O % 2 == 0) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j1 = 0; j1 < O; j1 += 2) {
                        V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                        *reinterpret_cast<V2 *>(p + j1) = vv;
                    }
                } else {
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
                }
            }
    };
    auto park_put = [&](int which, const T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) park[((which * O3) + (a * O + b) * O + d) * nthr + tid] = w[a][b][d];
    };
    auto park_get = [&](int which, T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) w[a][b][d] = park[((which * O3) + (a * O + b) * O + d) * nthr + tid];
    };

    T acc1[O][O][O], acc2[O][O][O];
    auto tb = [&](int i) -> T * { return tbuf0 + (size_t)(i & 1) * (slot_stride / sizeof(T)); };
    auto second = [&](int i) {                               // second application on the first one's cell i
        mbar_wait(&tbar[i & 1], (uint32_t)((i >> 1) & 1));   // every thread has written its part of cell i
        if (!active) return;
        T b[O][O][O];
        k12_from(tb(i), b);
        if (i == 0) {
            park_put(1, b);
        } else {
            int cell = i - 1 - m3;
            if (cell < 0) cell += n3;
            b_half_put(acc2, b, out + base + (long)cell * slab + cell_off);
        }
        a_half(b, acc2);
    };

    for (int j = 0; j < n3; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        T w[O][O][O];
        if (active) k12_from(reinterpret_cast<const T *>(smem_raw + slot * slot_stride), w);
        __syncthreads();                                     // slab consumed; everybody is through iteration j - 1
        if (tid == 0 && j + NS < n3) issue(j + NS);
        if (j == 0) {
            if (active) { park_put(0, w); a_half(w, acc1); }
        } else {
            if (active) {
                b_half_put(acc1, w, tb(j - 1) + cell_off);   // first application, cell j - 1
                a_half(w, acc1);
            }
            mbar_arrive(&tbar[(j - 1) & 1]);
            if (j >= 2) second(j - 2);
        }
    }
    __syncthreads();
    if (active) {
        T wf[O][O][O];
        park_get(0, wf);
        b_half_put(acc1, wf, tb(n3 - 1) + cell_off);         // first application closes its line
    }
    mbar_arrive(&tbar[(n3 - 1) & 1]);
    second(n3 - 2);
    second(n3 - 1);
    if (active) {
        T bf[O][O][O];
        park_get(1, bf);
        int cell = n3 - 1 - m3;
        if (cell < 0) cell += n3;
        b_half_put(acc2, bf, out + base + (long)cell * slab + cell_off);
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// x_1 x_2 x_3 triple (APPS = 1) or the triple applied twice (APPS = 2), one block per velocity node AND per
// RANGE of x_2-cells (nb2 blocks per node).  The whole-plane kernels above keep one block of ~13 warps per SM,
// all in the same phase (shared-memory loads, then FMA chains, then the barrier): the LSU and the fp64 pipe are
// each busy about half of the time and their phases add up (ncu, profiles/ncu_twice_r2.md).  Half the plane per
// block halves threads and shared memory, two blocks are resident and their phases overlap.
//
// A block owns the x_2-cells [c2_0, c2_0 + c2b) of one node v.  Its outputs need the source cells
// c2_0 + APPS m2 ... c2_0 + APPS m2 + c2b + APPS - 1 (periodic): per x_3-cell (slab) and x_3-node one contiguous
// piece of rows of the (x_1,x_2)-plane, two when it wraps, brought in by cp.async.bulk; the extra cells are the
// x_2 neighbours (L2 hits for the block next door).  With APPS = 2 the first application is computed for
// c2b + 1 cells (one redundantly), staged in shared memory, and the second runs on it as in
// sweep_xtriple_plane2_kernel.  Bit-identical to the single sweeps.
// ------------------------------------------------------------------------------------------
template <typename T, int O, int APPS>
__global__ void __launch_bounds__(256, 2)
sweep_xtriple_part_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int n3, int c2b, int nb2,
                          const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                          const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                          const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = (APPS == 1) ? 4 : 3;
    constexpr int O3 = O * O * O;
    __shared__ __align__(8) uint64_t full[NS], tbar[2];
    const long N1 = (long)n1 * O, N2 = (long)n2 * O;
    const long slab = O * N2 * N1;                           // elements per x_3-cell of one node (global)
    const int RC = c2b + APPS;                               // staged x_2-cells
    const int nT = c2b + APPS - 1;                           // cells the first application is computed for
    const long PR = (long)RC * O;                            // staged rows per x_3-node
    const long lslab = O * PR * N1;                          // elements of a staged slab
    const size_t slot_stride = ((size_t)lslab * sizeof(T) + 127) & ~(size_t)127;
    const long TR = (long)nT * O;                            // rows per x_3-node of the first application's cell
    const size_t tb_stride = ((size_t)O * TR * N1 * sizeof(T) + 127) & ~(size_t)127;
    T *tbuf0 = reinterpret_cast<T *>(smem_raw + NS * slot_stride);
    T *park = reinterpret_cast<T *>(smem_raw + NS * slot_stride + (APPS == 2 ? 2 * tb_stride : 0));   // [APPS][O3][blockDim]
    const long v = blockIdx.x / nb2;
    const int c2_0 = (int)(blockIdx.x % nb2) * c2b;
    const long base = v * (long)n3 * slab;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int c1 = tid % n1, t2 = tid / n1;
    const bool act1 = t2 < nT;                               // computes a cell of the first application
    const bool act2 = t2 < c2b;                              // computes an output cell

    const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2, q3 = (base / qdiv3) % qmod3;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    const int t2c = act1 ? t2 : 0;
    // offsets of the 2 x 2 source cells in a staged slab / in the first application's cell: local rows t2, t2 + 1
    const int off[2][2] = {{(int)(t2c * O * N1 + sa1 * O), (int)(t2c * O * N1 + sb1 * O)},
                           {(int)((t2c + 1) * O * N1 + sa1 * O), (int)((t2c + 1) * O * N1 + sb1 * O)}};
    int rs = c2_0 + APPS * m2;                               // first staged x_2-cell (global index)
    rs %= n2;
    const int first_cells = (rs + RC <= n2) ? RC : n2 - rs;  // cells before the periodic wrap

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        mbar_init(&tbar[0], nthr);
        mbar_init(&tbar[1], nthr);
    }
    __syncthreads();
    auto issue = [&](int j) {                                // slab j <-> source x_3-cell (m3 + j) mod n3
        int cell = m3 + j;
        if (cell >= n3) cell -= n3;
        const int slot = j % NS;
        T *dst = reinterpret_cast<T *>(smem_raw + slot * slot_stride);
        mbar_expect_tx(&full[slot], (uint32_t)((size_t)lslab * sizeof(T)));
        const T *src = in + base + (long)cell * slab;
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            const uint32_t b1 = (uint32_t)((size_t)first_cells * O * N1 * sizeof(T));
            bulk_g2s(dst + l3 * PR * N1, src + l3 * N2 * N1 + (long)rs * O * N1, b1, &full[slot]);
            if (first_cells < RC)
                bulk_g2s(dst + l3 * PR * N1 + (long)first_cells * O * N1, src + l3 * N2 * N1,
                         (uint32_t)((size_t)(RC - first_cells) * O * N1 * sizeof(T)), &full[slot]);
        }
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n3; ++j) issue(j);

    // (k1,k2)-swept values of this thread's cell from a staged array with `rows` rows per x_3-node
    auto k12_from = [&](const T *sl, long rows, T (&w)[O][O][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[2][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 2; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    T r0[O], r1[O];
                    load_cell<T, O>(sl + l3 * rows * N1 + off[e2][0] + l2 * N1, r0);
                    load_cell<T, O>(sl + l3 * rows * N1 + off[e2][1] + l2 * N1, r1);
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; }
                    w[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                }
        }
    };
    auto a_half = [&](const T (&w)[O][O][O], T (&acc)[O][O][O]) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                    for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                    acc[j3][j2][j1] = a;
                }
    };
    // B-half of the k3 rule; the O^3 results go to dst as O^2 rows of O values (row pitch N1, x_3-node pitch p3)
    auto b_half_put = [&](const T (&acc)[O][O][O], const T (&w)[O][O][O], T *dst, long p3) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2) {
                T res[O];
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = acc[j3][j2][j1];
#pragma unroll
                    for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                    res[j1] = a;
                }
                T *p = dst + (long)j3 * p3 + (long)j2 * N1;
                if constexpr (O % 2 == 0) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j1 = 0; j1 < O; j1 += 2) {
                        V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                        *reinterpret_cast<V2 *>(p + j1) = vv;
                    }
                } else {
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
                }
            }
    };
    auto park_put = [&](int which, const T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) park[((which * O3) + (a * O + b) * O + d) * nthr + tid] = w[a][b][d];
    };
    auto park_get = [&](int which, T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) w[a][b][d] = park[((which * O3) + (a * O + b) * O + d) * nthr + tid];
    };
    const long own_t = (long)t2c * O * N1 + (long)c1 * O;                    // this thread's cell in a T buffer
    const long own_g = (long)(c2_0 + (act2 ? t2 : 0)) * O * N1 + (long)c1 * O;   // ... in a global slab
    auto tb = [&](int i) -> T * { return tbuf0 + (size_t)(i & 1) * (tb_stride / sizeof(T)); };

    T acc1[O][O][O], acc2[O][O][O];
    auto out_cell = [&](int i) {                             // output x_3-cell closed when first-application cell i arrives
        int cell = i - 1 - (APPS == 2 ? m3 : 0);
        if (cell < 0) cell += n3;
        return cell;
    };
    auto second = [&](int i) {                               // APPS == 2: second application on the first one's cell i
        mbar_wait(&tbar[i & 1], (uint32_t)((i >> 1) & 1));
        if (!act2) return;
        T b[O][O][O];
        k12_from(tb(i), TR, b);
        if (i == 0) park_put(1, b);
        else b_half_put(acc2, b, out + base + (long)out_cell(i) * slab + own_g, N2 * N1);
        a_half(b, acc2);
    };

    for (int j = 0; j < n3; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        T w[O][O][O];
        if (act1) k12_from(reinterpret_cast<const T *>(smem_raw + slot * slot_stride), PR, w);
        __syncthreads();                                     // slab consumed; everybody is through iteration j - 1
        if (tid == 0 && j + NS < n3) issue(j + NS);
        if (j == 0) {
            if (act1) { park_put(0, w); a_half(w, acc1); }
        } else if constexpr (APPS == 1) {
            if (act1) {
                b_half_put(acc1, w, out + base + (long)(j - 1) * slab + own_g, N2 * N1);
                a_half(w, acc1);
            }
        } else {
            if (act1) {
                b_half_put(acc1, w, tb(j - 1) + own_t, TR * N1);   // first application, cell j - 1
                a_half(w, acc1);
            }
            mbar_arrive(&tbar[(j - 1) & 1]);
            if (j >= 2) second(j - 2);
        }
    }
    if constexpr (APPS == 1) {
        if (act1) {
            T wf[O][O][O];
            park_get(0, wf);
            b_half_put(acc1, wf, out + base + (long)(n3 - 1) * slab + own_g, N2 * N1);   // closes the periodic line
        }
    } else {
        __syncthreads();
        if (act1) {
            T wf[O][O][O];
            park_get(0, wf);
            b_half_put(acc1, wf, tb(n3 - 1) + own_t, TR * N1);   // first application closes its line
        }
        mbar_arrive(&tbar[(n3 - 1) & 1]);
        second(n3 - 2);
        second(n3 - 1);
        if (act2) {
            T bf[O][O][O];
            park_get(1, bf);
            b_half_put(acc2, bf, out + base + (long)out_cell(n3) * slab + own_g, N2 * N1);
        }
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// sweep_xtriple_part_kernel<T, O, 1> with TWO adjacent x_2-cells per thread.  The k1-swept values of the x_2
// source cell shared by the two output cells are computed once instead of twice: 12 instead of 16 shared-memory
// loads and 28 instead of 32 FMA chains per output cell (the plane kernels are bound by exactly these two units,
// and under the power cap every instruction saved is clock gained).  c2b must be even.  Same arithmetic per
// value, bit-identical to the single sweeps.
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(128, 3)
sweep_xtriple_part2_kernel(const T *__restrict__ in, T *__restrict__ out, int n1, int n2, int n3, int c2b, int nb2,
                           const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                           const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                           const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    constexpr int NS = 4;
    constexpr int O3 = O * O * O;
    __shared__ __align__(8) uint64_t full[NS];
    const long N1 = (long)n1 * O, N2 = (long)n2 * O;
    const long slab = O * N2 * N1;                           // elements per x_3-cell of one node (global)
    const int RC = c2b + 1;                                  // staged x_2-cells
    const long PR = (long)RC * O;                            // staged rows per x_3-node
    const long lslab = O * PR * N1;
    const size_t slot_stride = ((size_t)lslab * sizeof(T) + 127) & ~(size_t)127;
    T *park = reinterpret_cast<T *>(smem_raw + NS * slot_stride);   // [2][O3][blockDim]: the two windows' first cells
    const long v = blockIdx.x / nb2;
    const int c2_0 = (int)(blockIdx.x % nb2) * c2b;
    const long base = v * (long)n3 * slab;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int c1 = tid % n1, tp = tid / n1;                  // tp: pair of x_2-cells 2 tp, 2 tp + 1 (local)
    const bool active = 2 * tp < c2b;

    const long q1 = (base / qdiv1) % qmod1, q2 = (base / qdiv2) % qmod2, q3 = (base / qdiv3) % qmod3;
    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    const int t2 = active ? 2 * tp : 0;
    const int offa = (int)(t2 * O * N1 + sa1 * O), offb = (int)(t2 * O * N1 + sb1 * O);   // first of the 3 source cells
    int rs = (c2_0 + m2) % n2;                               // first staged x_2-cell (global index)
    const int first_cells = (rs + RC <= n2) ? RC : n2 - rs;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    __syncthreads();
    auto issue = [&](int j) {                                // slab j <-> source x_3-cell (m3 + j) mod n3
        int cell = m3 + j;
        if (cell >= n3) cell -= n3;
        const int slot = j % NS;
        T *dst = reinterpret_cast<T *>(smem_raw + slot * slot_stride);
        mbar_expect_tx(&full[slot], (uint32_t)((size_t)lslab * sizeof(T)));
        const T *src = in + base + (long)cell * slab;
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            const uint32_t b1 = (uint32_t)((size_t)first_cells * O * N1 * sizeof(T));
            bulk_g2s(dst + l3 * PR * N1, src + l3 * N2 * N1 + (long)rs * O * N1, b1, &full[slot]);
            if (first_cells < RC)
                bulk_g2s(dst + l3 * PR * N1 + (long)first_cells * O * N1, src + l3 * N2 * N1,
                         (uint32_t)((size_t)(RC - first_cells) * O * N1 * sizeof(T)), &full[slot]);
        }
    };
    if (tid == 0)
        for (int j = 0; j < NS && j < n3; ++j) issue(j);

    // (k1,k2)-swept values of the thread's two cells: k1 rule on the three source cells, k2 rule twice
    auto k12_from = [&](const T *sl, T (&wa)[O][O][O], T (&wb)[O][O][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[3][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 3; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    T r0[O], r1[O];
                    load_cell<T, O>(sl + l3 * PR * N1 + offa + (e2 * O + l2) * N1, r0);
                    load_cell<T, O>(sl + l3 * PR * N1 + offb + (e2 * O + l2) * N1, r1);
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a0[O], a1[O], a2[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; a2[l] = tk[2][l][j1]; }
                    wa[l3][j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                    wb[l3][j2][j1] = chain<T, O>(A2, B2, j2, a1, a2);
                }
        }
    };
    auto a_half = [&](const T (&w)[O][O][O], T (&acc)[O][O][O]) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                    for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                    acc[j3][j2][j1] = a;
                }
    };
    auto b_half_put = [&](const T (&acc)[O][O][O], const T (&w)[O][O][O], T *dst) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2) {
                T res[O];
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = acc[j3][j2][j1];
#pragma unroll
                    for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                    res[j1] = a;
                }
                T *p = dst + (long)j3 * N2 * N1 + (long)j2 * N1;
                if constexpr (O % 2 == 0) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j1 = 0; j1 < O; j1 += 2) {
                        V2 vv; vv.v[0] = res[j1]; vv.v[1] = res[j1 + 1];
                        *reinterpret_cast<V2 *>(p + j1) = vv;
                    }
                } else {
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) p[j1] = res[j1];
                }
            }
    };
    auto park_put = [&](int which, const T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) park[((which * O3) + (a * O + b) * O + d) * nthr + tid] = w[a][b][d];
    };
    auto park_get = [&](int which, T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int b = 0; b < O; ++b)
#pragma unroll
                for (int d = 0; d < O; ++d) w[a][b][d] = park[((which * O3) + (a * O + b) * O + d) * nthr + tid];
    };
    const long own_a = (long)(c2_0 + t2) * O * N1 + (long)c1 * O;      // first of this thread's two cells in a global slab
    const long own_b = own_a + (long)O * N1;

    T acca[O][O][O], accb[O][O][O];
    for (int j = 0; j < n3; ++j) {
        const int slot = j % NS;
        mbar_wait(&full[slot], (uint32_t)((j / NS) & 1));
        T wa[O][O][O], wb[O][O][O];
        if (active) k12_from(reinterpret_cast<const T *>(smem_raw + slot * slot_stride), wa, wb);
        __syncthreads();                                     // slab consumed
        if (tid == 0 && j + NS < n3) issue(j + NS);
        if (active) {
            if (j == 0) {
                park_put(0, wa); park_put(1, wb);
            } else {
                T *dst = out + base + (long)(j - 1) * slab;
                b_half_put(acca, wa, dst + own_a);
                b_half_put(accb, wb, dst + own_b);
            }
            a_half(wa, acca);
            a_half(wb, accb);
        }
    }
    if (active) {                                            // closes the periodic lines
        T wf[O][O][O];
        T *dst = out + base + (long)(n3 - 1) * slab;
        park_get(0, wf);
        b_half_put(acca, wf, dst + own_a);
        park_get(1, wf);
        b_half_put(accb, wf, dst + own_b);
    }
}

}  // namespace sldg

namespace sldg {

// ------------------------------------------------------------------------------------------
// sweep_vtriple_tile_kernel with TWO adjacent k2-cells per thread (what took the x-triple from 11.5 to 9.9 ms):
// the k1-swept values of the k2 source cell shared by the two output cells are computed once; 24 instead of 32
// shared-memory loads and 28 instead of 32 FMA chains per output cell.  Block = W columns x 4 k1-cells x C2 / 2
// pairs of k2-cells; the two windows' first cells are parked in shared memory.  Same staging, same per-lane
// left/right and early/late choices, same per-block fallback; bit-identical to the three sweeps.
// ------------------------------------------------------------------------------------------
template <typename T, int O, int W, int C2, int NS, int MINB>
__global__ void __launch_bounds__(W * 2 * C2, MINB)
sweep_vtriple_tile2_kernel(const __grid_constant__ CUtensorMap tmap, const T *__restrict__ in, T *__restrict__ out,
                           long inner1, int n1, int n2, int n3, long outer3,
                           const int *__restrict__ mtab1, const T *__restrict__ ab1, long count1, long qdiv1, long qmod1,
                           const int *__restrict__ mtab2, const T *__restrict__ ab2, long count2, long qdiv2, long qmod2,
                           const int *__restrict__ mtab3, const T *__restrict__ ab3, long count3, long qdiv3, long qmod3) {
    static_assert(C2 % 2 == 0, "pairs of k2-cells");
    constexpr int C1 = 4;
    constexpr int NBOX = (C1 + 2) * (C2 + 2);
    constexpr int CELL = O * O * O * W;
    constexpr int STAGE = NBOX * CELL;
    constexpr int O3 = O * O * O;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t full[NS];
    T *ring = reinterpret_cast<T *>(smem_raw);
    T *park = ring + (size_t)NS * STAGE;                     // [2][O3][blockDim]

    const long tiles_x = inner1 / W;
    const int groups1 = n1 / C1, groups2 = n2 / C2;
    long b = blockIdx.x;
    const int g1 = (int)(b % groups1); b /= groups1;
    const int g2 = (int)(b % groups2); b /= groups2;
    const long tx = b % tiles_x;
    const long oo3 = b / tiles_x;
    const int tid = threadIdx.x, nthr = blockDim.x, col = tid % W, t1 = (tid / W) % C1, tp = tid / (W * C1);
    const int warp = tid >> 5, lane = tid & 31;
    const int c1 = g1 * C1 + t1, c2 = g2 * C2 + 2 * tp;      // first of this thread's two k2-cells
    const long ii = tx * W + col;
    const long s1 = inner1, s2 = (long)n1 * O * s1, s3 = (long)n2 * O * s2;
    const long plane = oo3 * (long)n3 * O * s3 + ii;
    const long lin0 = plane + (long)c1 * O * s1 + (long)c2 * O * s2;
    const long q1 = (lin0 / qdiv1) % qmod1, q2 = (lin0 / qdiv2) % qmod2, q3 = (lin0 / qdiv3) % qmod3;

    T A1[O * O], B1[O * O], A2[O * O], B2[O * O], A3[O * O], B3[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A1[e] = ab1[(long)e * count1 + q1]; B1[e] = ab1[(long)(O * O + e) * count1 + q1];
        A2[e] = ab2[(long)e * count2 + q2]; B2[e] = ab2[(long)(O * O + e) * count2 + q2];
        A3[e] = ab3[(long)e * count3 + q3]; B3[e] = ab3[(long)(O * O + e) * count3 + q3];
    }
    const int m1 = mtab1[q1], m2 = mtab2[q2], m3 = mtab3[q3];
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    }
    const bool small = __syncthreads_and((m1 == 0 || m1 == n1 - 1) && (m2 == 0 || m2 == n2 - 1) &&
                                         (m3 == 0 || m3 == n3 - 1)) != 0;
    int sa1 = c1 + m1; if (sa1 >= n1) sa1 -= n1;             // global path
    int sb1 = sa1 + 1; if (sb1 == n1) sb1 = 0;
    int s2c[3];
    s2c[0] = c2 + m2; if (s2c[0] >= n2) s2c[0] -= n2;
    s2c[1] = s2c[0] + 1; if (s2c[1] == n2) s2c[1] = 0;
    s2c[2] = s2c[1] + 1; if (s2c[2] == n2) s2c[2] = 0;
    const int la = t1 + (m1 == 0 ? 1 : 0), lb = 2 * tp + (m2 == 0 ? 1 : 0);   // staged path: first local source cells
    const int late = (m3 == 0) ? 1 : 0;
    const bool needL1 = __syncthreads_or(m1 != 0) != 0, needR1 = __syncthreads_or(m1 == 0) != 0;
    const bool needL2 = __syncthreads_or(m2 != 0) != 0, needR2 = __syncthreads_or(m2 == 0) != 0;
    const int nboxes = (C1 + (needL1 ? 1 : 0) + (needR1 ? 1 : 0)) * (C2 + (needL2 ? 1 : 0) + (needR2 ? 1 : 0));

    auto issue = [&](int j) {                                // stage j <-> k3-cell (j - 1) mod n3; warp 0 calls
        int cell3 = j - 1;
        if (cell3 < 0) cell3 += n3;
        if (cell3 >= n3) cell3 -= n3;
        const int slot = j % NS;
        if (lane == 0) mbar_expect_tx(&full[slot], (uint32_t)(nboxes * CELL * sizeof(T)));
        const uint64_t pol = policy_evict_first();
#pragma unroll
        for (int bx = lane; bx < NBOX; bx += 32) {
            const int ca = bx % (C1 + 2), cb = bx / (C1 + 2);
            if ((ca > 0 || needL1) && (ca < C1 + 1 || needR1) && (cb > 0 || needL2) && (cb < C2 + 1 || needR2)) {
                int cell1 = g1 * C1 - 1 + ca;
                if (cell1 < 0) cell1 += n1;
                if (cell1 >= n1) cell1 -= n1;
                int cell2 = g2 * C2 - 1 + cb;
                if (cell2 < 0) cell2 += n2;
                if (cell2 >= n2) cell2 -= n2;
                tma_load_5d_hint(ring + (size_t)slot * STAGE + (size_t)bx * CELL, &tmap, (int)(tx * W), cell1 * O,
                                 cell2 * O, cell3 * O, (int)oo3, &full[slot], pol);
            }
        }
    };
    // k2 rule twice on the k1-swept values of the three source cells
    auto k2_two = [&](const T (&tk)[3][O][O], T (&wa)[O][O], T (&wb)[O][O]) {
#pragma unroll
        for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
            for (int j1 = 0; j1 < O; ++j1) {
                T a0[O], a1[O], a2[O];
#pragma unroll
                for (int l = 0; l < O; ++l) { a0[l] = tk[0][l][j1]; a1[l] = tk[1][l][j1]; a2[l] = tk[2][l][j1]; }
                wa[j2][j1] = chain<T, O>(A2, B2, j2, a0, a1);
                wb[j2][j1] = chain<T, O>(A2, B2, j2, a1, a2);
            }
    };
    auto k12_staged = [&](int slot, T (&wa)[O][O][O], T (&wb)[O][O][O]) {
        const T *st = ring + (size_t)slot * STAGE + col;
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            T tk[3][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 3; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    const T *p0 = st + (size_t)((lb + e2) * (C1 + 2) + la) * CELL + ((l3 * O + l2) * O) * W;
                    T r0[O], r1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { r0[l] = p0[l * W]; r1[l] = p0[CELL + l * W]; }
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
            k2_two(tk, wa[l3], wb[l3]);
        }
    };
    auto k12_global = [&](int cell3, T (&wa)[O][O][O], T (&wb)[O][O][O]) {
#pragma unroll
        for (int l3 = 0; l3 < O; ++l3) {
            const T *row = in + plane + ((long)cell3 * O + l3) * s3;
            T tk[3][O][O];
#pragma unroll
            for (int e2 = 0; e2 < 3; ++e2)
#pragma unroll
                for (int l2 = 0; l2 < O; ++l2) {
                    const T *p = row + ((long)s2c[e2] * O + l2) * s2;
                    T r0[O], r1[O];
#pragma unroll
                    for (int l = 0; l < O; ++l) { r0[l] = p[((long)sa1 * O + l) * s1]; r1[l] = p[((long)sb1 * O + l) * s1]; }
#pragma unroll
                    for (int j1 = 0; j1 < O; ++j1) tk[e2][l2][j1] = chain<T, O>(A1, B1, j1, r0, r1);
                }
            k2_two(tk, wa[l3], wb[l3]);
        }
    };
    auto a_half = [&](const T (&w)[O][O][O], T (&acc)[O][O][O]) {
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = mul_t<T>(A3[j3 * O], w[0][j2][j1]);
#pragma unroll
                    for (int l = 1; l < O; ++l) a = fma_t<T>(A3[j3 * O + l], w[l][j2][j1], a);
                    acc[j3][j2][j1] = a;
                }
    };
    auto b_half_store = [&](int i3, long celloff, const T (&acc)[O][O][O], const T (&w)[O][O][O]) {
        T *dst = out + lin0 + celloff + (long)i3 * O * s3;
#pragma unroll
        for (int j3 = 0; j3 < O; ++j3)
#pragma unroll
            for (int j2 = 0; j2 < O; ++j2)
#pragma unroll
                for (int j1 = 0; j1 < O; ++j1) {
                    T a = acc[j3][j2][j1];
#pragma unroll
                    for (int l = 0; l < O; ++l) a = fma_t<T>(B3[j3 * O + l], w[l][j2][j1], a);
                    __stcs(dst + (long)j3 * s3 + (long)j2 * s2 + (long)j1 * s1, a);
                }
    };
    auto park_put = [&](int which, const T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int c = 0; c < O; ++c)
#pragma unroll
                for (int d = 0; d < O; ++d) park[((which * O3) + (a * O + c) * O + d) * nthr + tid] = w[a][c][d];
    };
    auto park_get = [&](int which, T (&w)[O][O][O]) {
#pragma unroll
        for (int a = 0; a < O; ++a)
#pragma unroll
            for (int c = 0; c < O; ++c)
#pragma unroll
                for (int d = 0; d < O; ++d) w[a][c][d] = park[((which * O3) + (a * O + c) * O + d) * nthr + tid];
    };
    const long offb = (long)O * s2;                          // the second cell of the pair

    T acca[O][O][O], accb[O][O][O], wa[O][O][O], wb[O][O][O];
    auto first = [&]() { park_put(0, wa); park_put(1, wb); a_half(wa, acca); a_half(wb, accb); };
    auto next = [&](int i3) {
        b_half_store(i3, 0, acca, wa); b_half_store(i3, offb, accb, wb);
        a_half(wa, acca); a_half(wb, accb);
    };
    auto close = [&]() {
        park_get(0, wa); b_half_store(n3 - 1, 0, acca, wa);
        park_get(1, wb); b_half_store(n3 - 1, offb, accb, wb);
    };
    if (small) {
        if (warp == 0)
            for (int j = 0; j < NS && j <= n3; ++j) issue(j);
        for (int j = 0; j <= n3 + 1; ++j) {
            const int t = j - late;
            bool fresh = false;
            if (j <= n3) {
                mbar_wait(&full[j % NS], (uint32_t)((j / NS) & 1));
                if (t >= 0 && t <= n3 - 1) { k12_staged(j % NS, wa, wb); fresh = true; }
                __syncthreads();                             // raw values read: refill the slot before the k3 rule
                if (warp == 0 && j + NS <= n3) issue(j + NS);
            }
            if (fresh) {
                if (t == 0) first();
                else next(t - 1);
            }
            if (t == n3) close();
        }
    } else {
        for (int t = 0; t <= n3; ++t) {
            int cell3 = m3 + t;
            if (cell3 >= n3) cell3 -= n3;
            if (t <= n3 - 1) {
                k12_global(cell3, wa, wb);
                if (t == 0) first();
                else next(t - 1);
            } else {
                close();
            }
        }
    }
}

}  // namespace sldg
