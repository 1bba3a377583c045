// leaf32_kernel.cuh -- the 128 x 128 diagonal-block factorisation of the blocked Cholesky as a
// BLOCKED kernel: four 32 x 32 sub-block steps, each
//   P1  the diagonal sub-block factored by ONE WARP in registers (lane = row), the pivot row broadcast with
//       __shfl_sync -- a dependent step costs a shuffle and a reciprocal, not a CTA barrier plus a shared-memory
//       broadcast (the 128-step rank-1 sweep of potrf_leaf_kernel: ~415 cycles per step, profiles/r01f_leaf_ncu.md);
//   P2  the 32-row panel right of it solved by substitution, one thread per column, while another warp inverts
//       the sub-block;
//   P3  the rank-32 trailing update of the remaining sub-blocks on the FP64 tensor pipe (mma.sync m8n8k4, operands
//       read straight from the shared image);
// then W = U^-1 is assembled from the inverted 32 x 32 diagonal sub-blocks by two doubling levels, again on DMMA.
// Same contract as potrf_leaf_kernel: U_kk in place (upper triangle), W = U_kk^-1 to Winv (identity-padded), a pivot
// that is not > 0 (or NaN) recorded as info = 1-based global index.
//
// Shared image: S(r, c) at r + c * P32, P32 = 132 (columns 16-byte aligned for 16-byte cp.async; 2 * 132 mod 32 = 8
// makes the DMMA fragment loads -- four consecutive rows x eight columns, or the transpose of that -- hit every
// bank at most twice, the minimum for 64-bit accesses).  The upper triangle holds A -> U; the strictly-lower triangle
// receives W TRANSPOSED (W(i, c) at S(c, i)), its diagonal lives in dinv[]: both factors in one 128 x 132 image.
#pragma once
#include <cuda_runtime.h>

#include "leaf_kernels.cuh"
#include "ptx.cuh"

namespace gs {

constexpr int P32 = 132;                 // pitch of the shared image (doubles)
constexpr int PT32 = 68;                 // pitch of the 64 x 64 temporary of the inverse assembly
constexpr int kLeaf32Threads = 256;
constexpr int kLeaf32SmemBytes = (LB * P32 + 64 * PT32 + LB + 64) * 8 + 64;   // image + temporary + dinv + pivot rows + flags

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// (the pivot rows are addressed through their 32-bit shared-memory address: explicit ld / st.shared)
__device__ __forceinline__ double lds64(uint32_t addr)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}

// 1 / d to ~1 ulp without the IEEE-rounding division sequence: the hardware seed (MUFU.RCP64H, ~20 bits) and two
// Newton steps.  The reciprocal of the pivot sits on the dependent chain of every elimination step.
__device__ __forceinline__ double leaf32_rcp(double d)
{
    double x;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
    const double e = fma(-d, x, 1.0);      // 1 - d x0
    const double x1 = fma(x, e, x);        // x0 (1 + e)
    const double e2 = e * e;               // 1 - d x1 = e^2 exactly: formed beside x1, not behind it
    return fma(x1, e2, x1);
}

// ---- P1: 32 x 32 diagonal sub-block at (b0, b0): A = L D L^T, then U = D^1/2 L^T.  FOUR warps, lane = row, warp w holds
// columns 8 w .. 8 w + 7 of every row in registers (the whole symmetric Schur complement is kept).  Per pivot J: lane J
// of every warp publishes its eight entries of the pivot row in a double-buffered shared row, one 128-thread named
// barrier, then every lane reads its multiplier A(J, lane) = A(lane, J) and its warp's eight pivot-row entries back.
// The running diagonal of every row is carried redundantly by the four warps, so the next pivot is one __shfl_sync and
// its reciprocal starts one FMA behind the previous one.  (One warp doing the whole row update alone spends 280 of its
// 530 cycles per pivot on the shared-memory round trip of 24 values and 75 on 32 FMAs: profiles/r02_leaf32.md.)
// Returns the local index of the first pivot that is not > 0, or -1 (the same value in all four warps).
__device__ __forceinline__ int leaf32_potrf_4warps(double* S, double* dinv, uint32_t rowbuf, int b0, int lane, int w)
{
    double a[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int c = 8 * w + u;
        const int lo = c < lane ? c : lane, hi = c < lane ? lane : c;
        a[u] = S[(b0 + lo) + (b0 + hi) * P32];                   // A(min, max): the upper triangle holds the block
    }
    int bad = -1;
    double dr = 1.0;                                             // this lane's own pivot d(lane)
    double dii = S[(b0 + lane) + (b0 + lane) * P32];
    double d = __shfl_sync(0xffffffffu, dii, 0);
    double inv = leaf32_rcp(d);
#pragma unroll 1
    for (int J = 0; J < 32; ++J) {
        const uint32_t rb = rowbuf + (J & 1) * 256;
        if (lane == J) {
#pragma unroll
            for (int u = 0; u < 8; u += 2)
                asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"(rb + 8 * (8 * w + u)), "d"(a[u]), "d"(a[u + 1]) : "memory");
        }
        named_bar_sync(2, 128);
        if (!(d > 0.0)) { if (bad < 0) bad = J; }              // uniform: every thread holds the same d
        if (lane == J) dr = d;
        const double aj = lds64(rb + 8 * lane);                  // A(J, lane) = A(lane, J)
        const double l = (lane > J) ? aj * inv : 0.0;            // multiplier; 0: row not updated
        dii = fma(-l, aj, dii);
        const double dn = __shfl_sync(0xffffffffu, dii, (J + 1) & 31);
        const double invn = leaf32_rcp(dn);
#pragma unroll
        for (int u = 0; u < 8; u += 2) {
            const double2 p = lds128(rb + 8 * (8 * w + u));
            a[u] = fma(-l, p.x, a[u]);          // (columns <= J are dead: updating them too costs less than sparing them)
            a[u + 1] = fma(-l, p.y, a[u + 1]);
        }
        d = dn;
        inv = invn;
    }
    if (bad >= 0) return bad;
    // row `lane` of D L^T -> row of U = D^1/2 L^T
    const double s = 1.0 / sqrt(dr);
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        const int c = 8 * w + u;
        if (c > lane) S[(b0 + lane) + (b0 + c) * P32] = a[u] * s;
        else if (c == lane) S[(b0 + lane) + (b0 + c) * P32] = dr * s;
    }
    if (w == 0) dinv[b0 + lane] = s;
    return -1;
}

// The two substitutions below are template recursions over the step index: with `#pragma unroll` alone nvcc gives up on
// the 32 x 31 / 2 triangular nests and keeps the column in local memory behind a dynamically indexed loop.

// ---- P2a: column cg of the panel right of the sub-block: x = U_bb^-T a (right-looking substitution), one thread ----
template <int I>
__device__ __forceinline__ void leaf32_trsm_step(double (&r)[32], const double* S, const double* dinv, int b0)
{
    const double x = r[I] * dinv[b0 + I];
    r[I] = x;
#pragma unroll
    for (int m = I + 1; m < 32; ++m) r[m] = fma(-S[(b0 + I) + (b0 + m) * P32], x, r[m]);   // U(I, m): same address in every thread
    if constexpr (I + 1 < 32) leaf32_trsm_step<I + 1>(r, S, dinv, b0);
}

__device__ __forceinline__ void leaf32_trsm_column(double* S, const double* dinv, int b0, int cg)
{
    double r[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) r[i] = S[(b0 + i) + cg * P32];
    leaf32_trsm_step<0>(r, S, dinv, b0);
#pragma unroll
    for (int i = 0; i < 32; ++i) S[(b0 + i) + cg * P32] = r[i];
}

// ---- P2b: W_bb = U_bb^-1, lane = column c, stored transposed below the diagonal: S(b0 + c, b0 + i) = W(i, c), i < c ----
template <int I>
__device__ __forceinline__ void leaf32_invert_step(double (&r)[32], const double* S, const double* dinv, int b0)
{
    const double w = r[I] * dinv[b0 + I];                       // (zero for I > lane)
    r[I] = w;
#pragma unroll
    for (int m = 0; m < I; ++m) r[m] = fma(-S[(b0 + m) + (b0 + I) * P32], w, r[m]);
    if constexpr (I > 0) leaf32_invert_step<I - 1>(r, S, dinv, b0);
}

__device__ __forceinline__ void leaf32_invert_warp(double* S, const double* dinv, int b0, int lane)
{
    double r[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) r[i] = (i == lane) ? 1.0 : 0.0;
    leaf32_invert_step<31>(r, S, dinv, b0);
#pragma unroll
    for (int i = 0; i < 32; ++i)
        if (i < lane) S[(b0 + lane) + (b0 + i) * P32] = r[i];
}

// ---- P3: one 16 x 32 unit of the trailing update: S(r0:r0+16, c0:c0+32) -= P^T P, P = rows b0 .. b0+31 ----
// All 48 operand fragments are loaded before the first DMMA: with one or two warps per sub-partition nothing else
// hides the shared-memory latency, and a load -> DMMA -> load -> DMMA sequence costs ~275 cycles per k-step.
__device__ __forceinline__ void leaf32_update_unit(double* S, int b0, int r0, int c0, int lane)
{
    const int g = lane >> 2, q = lane & 3;
    double acc[2][4][2];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) { acc[mi][ni][0] = 0.0; acc[mi][ni][1] = 0.0; }
    double af[8][2], bf[8][4];
#pragma unroll
    for (int ks = 0; ks < 8; ++ks) {
        const int kr = b0 + 4 * ks + q;
#pragma unroll
        for (int mi = 0; mi < 2; ++mi) af[ks][mi] = S[kr + (r0 + 8 * mi + g) * P32];
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) bf[ks][ni] = S[kr + (c0 + 8 * ni + g) * P32];
    }
#pragma unroll
    for (int ks = 0; ks < 8; ++ks)
#pragma unroll
        for (int mi = 0; mi < 2; ++mi)
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], af[ks][mi], bf[ks][ni]);
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                double* p = &S[(r0 + 8 * mi + g) + (c0 + 8 * ni + 2 * q + e) * P32];
                *p -= acc[mi][ni][e];
            }
}

// W(gk, gn) of the partly assembled inverse: above the diagonal from the transposed image, dinv on it, zero below
__device__ __forceinline__ double leaf32_w(const double* S, const double* dinv, int gk, int gn)
{
    return gk < gn ? S[gn + gk * P32] : (gk == gn ? dinv[gk] : 0.0);
}

// ---- inverse assembly, unit 16 x 32 of T = U12 W22 (s x s blocks at (o, o+s) and (o+s, o+s)); k runs to the unit's last column ----
// k in chunks of 32 (8 k-steps), the fragments of a chunk loaded before its DMMAs (see leaf32_update_unit).  W22 is upper
// triangular: the chunk k0 = n0 is the diagonal 32-block (diagonal from dinv, zeros below), the chunks before it are plain.
__device__ __forceinline__ void leaf32_t_unit(const double* S, const double* dinv, double* T, int o, int s, int m0, int n0, int lane)
{
    const int g = lane >> 2, q = lane & 3;
    double acc[2][4][2];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) { acc[mi][ni][0] = 0.0; acc[mi][ni][1] = 0.0; }
#pragma unroll 1
    for (int k0 = 0; k0 <= n0; k0 += 32) {
        double af[8][2], bf[8][4];
        const bool diag = k0 == n0;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const int k = k0 + 4 * ks + q;
#pragma unroll
            for (int mi = 0; mi < 2; ++mi) af[ks][mi] = S[(o + m0 + 8 * mi + g) + (o + s + k) * P32];
#pragma unroll
            for (int ni = 0; ni < 4; ++ni)
                bf[ks][ni] = diag ? leaf32_w(S, dinv, o + s + k, o + s + n0 + 8 * ni + g) : S[(o + s + n0 + 8 * ni + g) + (o + s + k) * P32];
        }
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)
#pragma unroll
            for (int mi = 0; mi < 2; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], af[ks][mi], bf[ks][ni]);
    }
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
            for (int e = 0; e < 2; ++e) T[(m0 + 8 * mi + g) + (n0 + 8 * ni + 2 * q + e) * PT32] = acc[mi][ni][e];
}

// ---- unit 16 x 32 of W12 = -W11 T, stored transposed: S(o + s + n, o + m) = W12(m, n); k runs from the unit's first row ----
// W11 is upper triangular: k >= m.  Chunks of 32 from the 32-block that holds row m0 (masked loads) to s (plain loads).
__device__ __forceinline__ void leaf32_x_unit(double* S, const double* dinv, const double* T, int o, int s, int m0, int n0, int lane)
{
    const int g = lane >> 2, q = lane & 3;
    double acc[2][4][2];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) { acc[mi][ni][0] = 0.0; acc[mi][ni][1] = 0.0; }
    const int kfirst = m0 & ~31;
#pragma unroll 1
    for (int k0 = kfirst; k0 < s; k0 += 32) {
        double af[8][2], bf[8][4];
        const bool diag = k0 == kfirst;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
            const int k = k0 + 4 * ks + q;
#pragma unroll
            for (int mi = 0; mi < 2; ++mi)
                af[ks][mi] = diag ? leaf32_w(S, dinv, o + m0 + 8 * mi + g, o + k) : S[(o + k) + (o + m0 + 8 * mi + g) * P32];
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) bf[ks][ni] = T[k + (n0 + 8 * ni + g) * PT32];
        }
#pragma unroll
        for (int ks = 0; ks < 8; ++ks)
#pragma unroll
            for (int mi = 0; mi < 2; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], af[ks][mi], bf[ks][ni]);
    }
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni)
#pragma unroll
            for (int e = 0; e < 2; ++e)
                S[(o + s + n0 + 8 * ni + 2 * q + e) + (o + m0 + 8 * mi + g) * P32] = -acc[mi][ni][e];
}

// rows r0 .. r0+31 of U (all 128 columns: the upper part from the image, zeros below the diagonal) to global memory,
// by 128 threads (tt = 0 .. 127): 32 consecutive rows of a column per warp instruction
__device__ __forceinline__ void leaf32_store_u_rows(const double* S, double* blk, long long ld, int nb, int r0, int tt)
{
#pragma unroll 8
    for (int idx = tt; idx < 32 * LB; idx += 128) {
        const int r = r0 + (idx & 31), c = idx >> 5;
        if (r < nb && c < nb) blk[r + (long long)c * ld] = (r <= c) ? S[r + c * P32] : 0.0;
    }
}

#ifdef LEAF32_PROF
__device__ long long g_leaf32_prof[32];
#define LEAF32_STAMP(i) do { if (threadIdx.x == 0) g_leaf32_prof[i] = clock64(); } while (0)
#else
#define LEAF32_STAMP(i) do { } while (0)
#endif

__global__ void __launch_bounds__(kLeaf32Threads, 1)
potrf_leaf32_kernel(double* __restrict__ Sg, long long ld, int N, int j0, double* __restrict__ Winv, long long ldw, int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    double* S = reinterpret_cast<double*>(leaf_raw);
    double* T = S + LB * P32;
    double* dinv = T + 64 * PT32;
    double* rowbuf = dinv + LB;
    int* s_fail = reinterpret_cast<int*>(rowbuf + 64);
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int nb = min(LB, N - j0);
    double* blk = Sg + j0 + (long long)j0 * ld;
    if (t == 0) *s_fail = -1;
    LEAF32_STAMP(0);

    // ---- load the upper triangle (16-byte cp.async when the columns are 16-byte aligned, i.e. even ld) ----
    if ((ld & 1) == 0 && nb == LB) {
        const uint32_t s0 = smem_u32(S);
        for (int ch = t; ch < LB * (LB / 2); ch += kLeaf32Threads) {   // 16-byte chunk = rows 2 rr, 2 rr + 1 of column c
            const int c = ch >> 6, rr = ch & 63;
            if (2 * rr <= c) cp_async16(s0 + (2 * rr + c * P32) * 8, blk + 2 * rr + (long long)c * ld);
        }
        cp_async_wait_all();
    } else {
        for (int idx = t; idx < LB * LB; idx += kLeaf32Threads) {
            const int r = idx & (LB - 1), c = idx >> 7;
            if (r <= c) S[r + c * P32] = (c < nb) ? blk[r + (long long)c * ld] : (r == c ? 1.0 : 0.0);   // identity padding
        }
    }
    __syncthreads();
    LEAF32_STAMP(1);

#pragma unroll 1
    for (int kb = 0; kb < 4; ++kb) {
        const int b0 = 32 * kb;
        if (warp < 4) {
            const int bad = leaf32_potrf_4warps(S, dinv, smem_u32(rowbuf), b0, lane, warp);
            if (bad >= 0 && t == 0) *s_fail = b0 + bad;
        } else if (kb > 0) {
            leaf32_store_u_rows(S, blk, ld, nb, b0 - 32, t - 128);      // rows of the previous step are final: the idle warps store them
        }
        __syncthreads();
        LEAF32_STAMP(2 + 3 * kb);
        if (*s_fail >= 0) {
            if (t == 0) atomicCAS(info, 0, j0 + *s_fail + 1);
            return;
        }
        const int ncols = LB - b0 - 32;
        if (t < ncols) leaf32_trsm_column(S, dinv, b0, b0 + 32 + t);
        else if (warp == 7) leaf32_invert_warp(S, dinv, b0, lane);      // (ncols <= 96: warps 3 .. 7 have no columns)
        __syncthreads();
        LEAF32_STAMP(3 + 3 * kb);
        // trailing update: sub-block pairs (i, j), kb < i <= j <= 3, in 16 x 32 units
        const int nsub = 3 - kb;
        const int nunits = nsub * (nsub + 1);                            // pairs * 2
        for (int u = warp; u < nunits; u += 8) {
            const int pair = u >> 1, h = u & 1;
            int i = 0, rem = pair;                                       // pair -> (i, j), i <= j over nsub sub-blocks
            while (rem >= nsub - i) { rem -= nsub - i; ++i; }
            const int j = i + rem;
            leaf32_update_unit(S, b0, b0 + 32 + 32 * i + 16 * h, b0 + 32 + 32 * j, lane);
        }
        __syncthreads();
        LEAF32_STAMP(4 + 3 * kb);
    }

    LEAF32_STAMP(14);
    // ---- W = U^-1: the diagonal 32-blocks are inverted; two doubling levels, [A B; 0 D]^-1 = [A^-1, -A^-1 B D^-1; 0, D^-1] ----
    // level 1: pairs (0,1) and (2,3), s = 32: 2 units per pair; warps 0..3
    if (warp < 4) leaf32_t_unit(S, dinv, T + (warp >> 1) * 32 * PT32, (warp >> 1) * 64, 32, 16 * (warp & 1), 0, lane);
    else leaf32_store_u_rows(S, blk, ld, nb, 96, t - 128);            // the last 32 rows of U, beside the level-1 products
    __syncthreads();
    if (warp < 4) leaf32_x_unit(S, dinv, T + (warp >> 1) * 32 * PT32, (warp >> 1) * 64, 32, 16 * (warp & 1), 0, lane);
    __syncthreads();
    // level 2: the pair of 64-blocks, s = 64: 8 units (4 row halves x 2 column halves), one per warp
    leaf32_t_unit(S, dinv, T, 0, 64, 16 * (warp & 3), 32 * (warp >> 2), lane);
    __syncthreads();
    leaf32_x_unit(S, dinv, T, 0, 64, 16 * (warp & 3), 32 * (warp >> 2), lane);
    __syncthreads();
    LEAF32_STAMP(15);

    // ---- write W (upper triangle from the transposed image, dinv on the diagonal, zeros below; identity-padded) ----
#pragma unroll 8
    for (int idx = t; idx < LB * LB; idx += kLeaf32Threads) {
        const int r = idx & (LB - 1), c = idx >> 7;
        Winv[r + (long long)c * ldw] = leaf32_w(S, dinv, r, c);
    }
    LEAF32_STAMP(16);
}

}  // namespace gs
