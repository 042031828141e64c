// sweep_tma.cuh -- the sm_100a staged variants of the translation sweep (row a-2):
// whole lines are brought into shared memory by the asynchronous copy engine (TMA), so that
//   * every byte of f is read from HBM exactly once and in full, aligned rows, whatever the
//     per-line cell offset m is (the config-4 shifts scatter m over 8 values inside a warp);
//   * the load/store units only see conflict-free shared-memory reads and coalesced stores.
// Same arithmetic contract as sweep.cuh (D:O7).
#pragma once
#include "sweep.cuh"
#include "tma.cuh"

namespace sldg {

// ------------------------------------------------------------------------------------------
// v_a sweeps (and any sweep whose shift varies along `inner`): f viewed as
// [outer][N_k][inner]; one block owns the tile [all N_k rows] x [W consecutive inner
// indices] of one `outer` index, loaded by nbox TMA boxes of box_rows rows each.
// Thread (col, seg): column `col` of the tile, cells [seg*cps, (seg+1)*cps); q = ii % X.
// The line is periodic and entirely in shared memory, so m is free per thread.
// Outputs go straight from registers to global (row-contiguous across the warp).
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__global__ void __launch_bounds__(128)
sweep_tile_tma_kernel(const __grid_constant__ CUtensorMap tmap, T *__restrict__ out, long inner, int n,
                      long tiles_per_outer, int W, int nbox, int box_rows, int cps,
                      const int *__restrict__ mtab, const T *__restrict__ ab, long count, long X) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    T *tile = reinterpret_cast<T *>(smem_raw);                  // [nbox*box_rows][W]
    // Tiles are visited in memory order (neighbouring blocks extend each row contiguously).
    // Visiting them grouped by x-tile so that the (m, A, B) table chunk stays in L2 was tried
    // and is slower (5.7 vs 6.2 TB/s at config 4): DRAM row locality matters more.  Instead the
    // table is read with an L2 evict_last policy and f with evict_first.
    const long tile_id = blockIdx.x;
    const long oo = tile_id / tiles_per_outer;
    const long col0 = (tile_id - oo * tiles_per_outer) * W;
    const uint64_t pol_keep = policy_evict_last();
    if (threadIdx.x == 0) mbar_init(&bar, 1);
    __syncthreads();
    if (threadIdx.x == 0) {
        mbar_expect_tx(&bar, (uint32_t)((size_t)nbox * box_rows * W * sizeof(T)));
        const uint64_t pol_stream = policy_evict_first();
        for (int b = 0; b < nbox; ++b)
            tma_load_3d_hint(tile + (size_t)b * box_rows * W, &tmap, (int)col0, b * box_rows, (int)oo, &bar,
                             pol_stream);
    }
    const int col = threadIdx.x % W;
    const int seg = threadIdx.x / W;
    const long ii = col0 + col;
    const bool valid = ii < inner;
    const long q = valid ? (ii % X) : 0;
    T A[O * O], B[O * O];
#pragma unroll
    for (int e = 0; e < O * O; ++e) {
        A[e] = ld_hint(ab + (long)e * count + q, pol_keep);
        B[e] = ld_hint(ab + (long)(O * O + e) * count + q, pol_keep);
    }
    const int m = ld_hint(mtab + q, pol_keep);
    mbar_wait(&bar, 0);
    const int c0 = seg * cps;
    int c1 = c0 + cps;
    if (c1 > n) c1 = n;
    if (!valid || c0 >= c1) return;

    const T *colp = tile + col;
    int is = c0 + m;
    if (is >= n) is -= n;
    T u0[O], u1[O];
#pragma unroll
    for (int l = 0; l < O; ++l) u0[l] = colp[(is * O + l) * W];
    T *dst = out + (oo * (long)n * O + (long)c0 * O) * inner + ii;
#pragma unroll 2
    for (int c = c0; c < c1; ++c) {
        if (++is == n) is = 0;
#pragma unroll
        for (int l = 0; l < O; ++l) u1[l] = colp[(is * O + l) * W];
#pragma unroll
        for (int j = 0; j < O; ++j) __stcs(dst + (long)j * inner, chain<T, O>(A, B, j, u0, u1));
#pragma unroll
        for (int l = 0; l < O; ++l) u0[l] = u1[l];
        dst += (long)O * inner;
    }
}

// ------------------------------------------------------------------------------------------
// x_1 sweep (contiguous lines): a block owns R whole consecutive lines of one shift group
// (one contiguous span of global memory): one bulk copy in, thread-per-cell arithmetic from
// shared to shared, one bulk copy out.  Cell reads have a stride of O words (conflict-free
// for O = 1..4 with 8- and 4-byte words except O = 4, which is 2-way), and the copy engine
// does all global traffic in full 128-byte lines.
// ------------------------------------------------------------------------------------------
template <typename T, int O>
__device__ __forceinline__ void load_cell(const T *p, T (&u)[O]) {
    if constexpr (O % 2 == 0) {
        using V2 = Vec<T, 2>;
#pragma unroll
        for (int l = 0; l < O; l += 2) {
            V2 t = *reinterpret_cast<const V2 *>(p + l);
            u[l] = t.v[0]; u[l + 1] = t.v[1];
        }
    } else {
#pragma unroll
        for (int l = 0; l < O; ++l) u[l] = p[l];
    }
}

// JH = outputs per thread: JH == O is one thread per cell; at O >= 5 a cell's O outputs are split over
// ceil(O / JH) threads, each holding only its JH rows of A and B (thread-per-cell needs 2 O^2 coefficient
// registers: > 200 registers and 3.7 TB/s at O = 6; thread-per-node re-reads the 2 O inputs O times: 3.4 TB/s).
// TWICE: the sweep applied twice in shared memory before the copy out (x(tau) x(tau) of two consecutive Strang
// steps, bit-identical to two launches; see sweep_xpair_plane2_kernel).
template <typename T, int O, int JH = O, bool TWICE = false>
__global__ void __launch_bounds__(256)
sweep_x1_bulk_kernel(const T *__restrict__ in, T *__restrict__ out, int n, long lines_per_group, int R,
                     int chunks_per_group, const int *__restrict__ mtab, const T *__restrict__ ab,
                     long count, long qmod, long group_stride, long line_stride) {
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    __shared__ T s_ab[2 * O * O];
    __shared__ int s_m;
    const long g = blockIdx.x / chunks_per_group;
    const int ch = blockIdx.x - (int)(g * chunks_per_group);
    const long line0 = (long)ch * R;
    int nl = R;
    if (line0 + nl > lines_per_group) nl = (int)(lines_per_group - line0);
    const int ncell = nl * n;
    const uint32_t bytes = (uint32_t)((size_t)ncell * O * sizeof(T));
    const size_t half = ((size_t)R * n * O * sizeof(T) + 127) & ~(size_t)127;
    T *s_in = reinterpret_cast<T *>(smem_raw);
    T *s_out = reinterpret_cast<T *>(smem_raw + half);
    // lines of a shift group: contiguous (d_x >= 2: line_stride == n*O, one copy for the whole chunk) or
    // strided (d_x = 1: the lines that share a v_1 node are N_v1 lines apart; one copy per line)
    const long base = g * group_stride + line0 * line_stride;
    const bool contiguous = line_stride == (long)n * O;
    const uint32_t line_bytes = (uint32_t)((size_t)n * O * sizeof(T));

    if (threadIdx.x == 0) { mbar_init(&bar, 1); mbar_expect_tx(&bar, bytes); }
    __syncthreads();
    if (contiguous) {
        if (threadIdx.x == 0) bulk_g2s(s_in, in + base, bytes, &bar);
    } else {
        for (int r = threadIdx.x; r < nl; r += blockDim.x)
            bulk_g2s(s_in + (size_t)r * n * O, in + base + r * line_stride, line_bytes, &bar);
    }
    const long q = g % qmod;
    for (int e = threadIdx.x; e < 2 * O * O; e += blockDim.x) s_ab[e] = ab[(long)e * count + q];
    if (threadIdx.x == 32) s_m = mtab[q];
    __syncthreads();
    const int m = s_m;
    if constexpr (JH == O) {
        T A[O * O], B[O * O];
#pragma unroll
        for (int e = 0; e < O * O; ++e) { A[e] = s_ab[e]; B[e] = s_ab[O * O + e]; }
        mbar_wait(&bar, 0);
        auto apply = [&](const T *src, T *dst) {
            for (int c = threadIdx.x; c < ncell; c += blockDim.x) {
                const int line = c / n;
                const int i = c - line * n;
                int is = i + m;
                if (is >= n) is -= n;
                int is1 = is + 1;
                if (is1 == n) is1 = 0;
                T u0[O], u1[O];
                load_cell<T, O>(src + (size_t)(line * n + is) * O, u0);
                load_cell<T, O>(src + (size_t)(line * n + is1) * O, u1);
                T r[O];
#pragma unroll
                for (int j = 0; j < O; ++j) r[j] = chain<T, O>(A, B, j, u0, u1);
                T *po = dst + (size_t)c * O;
                if constexpr (O % 2 == 0) {
                    using V2 = Vec<T, 2>;
#pragma unroll
                    for (int j = 0; j < O; j += 2) {
                        V2 t; t.v[0] = r[j]; t.v[1] = r[j + 1];
                        *reinterpret_cast<V2 *>(po + j) = t;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < O; ++j) po[j] = r[j];
                }
            }
        };
        apply(s_in, s_out);
        if constexpr (TWICE) {
            __syncthreads();
            apply(s_out, s_in);
        }
    } else {
        // work item = (cell, part): part p computes the outputs j = p*JH .. min(O, (p+1)*JH) - 1
        constexpr int NP = (O + JH - 1) / JH;
        const int part = threadIdx.x % NP;                    // blockDim.x is a multiple of NP
        const int jb = part * JH;
        T Ar[JH][O], Br[JH][O];                              // this thread's rows of A and B
#pragma unroll
        for (int jj = 0; jj < JH; ++jj) {
            const int j = (jb + jj < O) ? jb + jj : O - 1;
#pragma unroll
            for (int l = 0; l < O; ++l) { Ar[jj][l] = s_ab[j * O + l]; Br[jj][l] = s_ab[O * O + j * O + l]; }
        }
        mbar_wait(&bar, 0);
        auto apply = [&](const T *src, T *dst) {
            for (int c = threadIdx.x / NP; c < ncell; c += blockDim.x / NP) {
                const int line = c / n;
                const int i = c - line * n;
                int is = i + m;
                if (is >= n) is -= n;
                int is1 = is + 1;
                if (is1 == n) is1 = 0;
                T u0[O], u1[O];
                load_cell<T, O>(src + (size_t)(line * n + is) * O, u0);
                load_cell<T, O>(src + (size_t)(line * n + is1) * O, u1);
                T *po = dst + (size_t)c * O + jb;
#pragma unroll
                for (int jj = 0; jj < JH; ++jj) {
                    T acc = mul_t<T>(Ar[jj][0], u0[0]);       // the O7 chain of output jb + jj
#pragma unroll
                    for (int l = 1; l < O; ++l) acc = fma_t<T>(Ar[jj][l], u0[l], acc);
#pragma unroll
                    for (int l = 0; l < O; ++l) acc = fma_t<T>(Br[jj][l], u1[l], acc);
                    if (jb + jj < O) po[jj] = acc;
                }
            }
        };
        apply(s_in, s_out);
        if constexpr (TWICE) {
            __syncthreads();
            apply(s_out, s_in);
        }
    }
    const T *s_res = TWICE ? s_in : s_out;                   // where the result sits
    fence_proxy_async();
    __syncthreads();
    if (contiguous) {
        if (threadIdx.x == 0) {
            bulk_s2g(out + base, s_res, bytes);
            bulk_commit();
            bulk_wait_read0();
        }
    } else {
        for (int r = threadIdx.x; r < nl; r += blockDim.x) {
            bulk_s2g(out + base + r * line_stride, s_res + (size_t)r * n * O, line_bytes);
            bulk_commit();
            bulk_wait_read0();
        }
    }
}

}  // namespace sldg
