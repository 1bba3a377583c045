// leaf_kernels.cuh -- latency-bound 128 x 128 diagonal-block kernels of the blocked factorisations.
//
//   potrf_leaf_kernel : factor one diagonal block S_kk = U_kk^T U_kk in place and also
//                       emit W_kk = U_kk^-1, which turns the panel solve U_k,: = U_kk^-T S_k,: into a
//                       tensor-core product.
//   trtri_leaf_kernel : invert every diagonal block of U, one CTA per block.
//
// One CTA of 256 threads = a 16 x 16 grid of threads.  The block is distributed 2-D CYCLICALLY:
// thread (ty,tx) keeps the 64 elements (ty + 16 r, tx + 16 c), r,c = 0..7, in registers, so the
// shrinking active region of a right-looking sweep stays spread over all threads and whole
// register rows / columns drop out of the (unrolled) update statically.  Factorisation and inversion
// are rank-1 sweeps: the pivot row is broadcast through a double-buffered shared-memory row (one
// __syncthreads per step); potrf_leaf_kernel forms U_kk and U_kk^-1 in ONE sweep (see there).  Global traffic goes through a
// padded shared-memory image of the block so that loads and stores are coalesced.  Blocks shorter
// than 128 (ragged last block) are padded with the identity, which factors / inverts to itself.
#pragma once
#include <cuda_runtime.h>

#include "ptx.cuh"

namespace gs {

constexpr int LB = 128;                 // leaf block order
constexpr int LP = LB + 1;              // padded shared-memory pitch (doubles)
constexpr int kLeafThreads = 256;
constexpr int kLeafSmemBytes = (LB * LP + 2 * LB + LB + LB) * 8 + 16;   // Usm + rowbuf[2] + dvec + dinv + flag

struct LeafSmem {
    double* U;        // LB x LB column-major, pitch LP
    double* rowbuf;   // 2 x LB
    double* dvec;     // LB
    double* dinv;     // LB : 1 / U(m,m)
    int* flag;
};

__device__ __forceinline__ LeafSmem leaf_smem(unsigned char* raw)
{
    LeafSmem s;
    s.U = reinterpret_cast<double*>(raw);
    s.rowbuf = s.U + LB * LP;
    s.dvec = s.rowbuf + 2 * LB;
    s.dinv = s.dvec + LB;
    s.flag = reinterpret_cast<int*>(s.dinv + LB);
    return s;
}

// Coalesced load of the upper triangle of a diagonal block into the padded shared image
// (identity-padded beyond nb, zero below the diagonal).
__device__ __forceinline__ void leaf_load_upper(const LeafSmem& s, const double* blk, long long ld, int nb, int t)
{
    // batches of 8 independent (predicated) loads in flight per thread: the one-at-a-time loop spent ~19k
    // cycles (15 % of the kernel) waiting on global latency (profiles/r01g_sharded.md, leaf notes)
    constexpr int kBatch = 8;
#pragma unroll 1
    for (int base = t; base < LB * LB; base += kLeafThreads * kBatch) {
        double v[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * kLeafThreads;
            const int row = idx & (LB - 1), col = idx >> 7;
            v[u] = (row == col) ? 1.0 : 0.0;
            if (row <= col && col < nb) v[u] = blk[row + (long long)col * ld];
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * kLeafThreads;
            s.U[(idx & (LB - 1)) + (idx >> 7) * LP] = v[u];
        }
    }
}

// Coalesced store of the whole shared image (rows, cols < nb) to a column-major destination.
__device__ __forceinline__ void leaf_store_all(const LeafSmem& s, double* dst, long long ld, int nb, int t)
{
    for (int idx = t; idx < LB * LB; idx += kLeafThreads) {
        const int row = idx & (LB - 1), col = idx >> 7;
        if (row < nb && col < nb) dst[row + (long long)col * ld] = s.U[row + col * LP];
    }
}

// V = U^-1 (upper) for the U held in s.U (pitch LP) with s.dinv[m] = 1 / U(m,m).  On return the
// shared image holds V (upper = inverse, strictly lower = 0).  Right-looking, backwards:
//   for m = LB-1 .. 0:  V(m,:) = acc(m,:) * dinv(m);  acc(k,:) -= U(k,m) V(m,:)  for k < m.
__device__ __forceinline__ void leaf_invert_upper(const LeafSmem& s, int tx, int ty)
{
    double v[8][8];
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) v[r][c] = (r == c && ty == tx) ? 1.0 : 0.0;

#pragma unroll
    for (int mr = 7; mr >= 0; --mr) {
#pragma unroll 1
        for (int mo = 15; mo >= 0; --mo) {
            const int m = mr * 16 + mo;
            double* rb = s.rowbuf + (m & 1) * LB;
            if (ty == mo) {
                const double inv = s.dinv[m];
#pragma unroll
                for (int c = mr; c < 8; ++c) {
                    v[mr][c] *= inv;
                    rb[tx + 16 * c] = v[mr][c];
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r <= mr; ++r) {
                const bool rowact = (r < mr) || (ty < mo);
                const double uk = s.U[ty + 16 * r + m * LP];
#pragma unroll
                for (int c = mr; c < 8; ++c) {
                    const bool colact = (c > mr) || (tx >= mo);
                    if (rowact && colact) v[r][c] = fma(-uk, rb[tx + 16 * c], v[r][c]);
                }
            }
        }
    }
    __syncthreads();   // every thread is done reading U before it is overwritten
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            s.U[row + col * LP] = (row <= col) ? v[r][c] : 0.0;
        }
    __syncthreads();
}

// One register row group r of the fused factor-and-invert step (potrf_leaf_kernel) for pivot j = 16 jr + jo:
// x(i,c) -= ri * pivot_row(c) for the columns that are live: Y (c <= j) and the Schur complement (c >= i).
// jr and r are compile-time constants after unrolling, so the register indices are static.
__device__ __forceinline__ void leaf_update_row(double (&a)[8][8], int jr, int r, const double* rb, double ri, double pj,
                                                bool rowact, int tx, int ty, int jo)
{
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        if (c < jr) {                    // Y, columns left of group jr
            if (rowact) a[r][c] = fma(-ri, rb[tx + 16 * c], a[r][c]);
        } else if (c == jr) {            // Y for columns <= j; on the diagonal register block also the upper part
            if (rowact && ((tx <= jo) || (r == jr && tx >= ty))) a[r][c] = fma(-ri, pj, a[r][c]);
        } else if (c >= r) {             // Schur complement, upper part
            if (rowact && ((c > r) || (tx >= ty))) a[r][c] = fma(-ri, rb[tx + 16 * c], a[r][c]);
        }
    }
}

// S: N x N column-major (ld), block starts at (j0, j0), order nb = min(LB, N - j0).
// Winv: LB x LB column-major block (leading dimension ldw) receiving U_kk^-1 (identity-padded).
// info: device flag; set (if still 0) to j0 + j + 1 when pivot j is not > 0.
__global__ void __launch_bounds__(kLeafThreads, 1)
potrf_leaf_kernel(double* __restrict__ S, long long ld, int N, int j0, double* __restrict__ Winv, long long ldw, int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const LeafSmem s = leaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int nb = min(LB, N - j0);
    double* blk = S + j0 + (long long)j0 * ld;

    leaf_load_upper(s, blk, ld, nb, t);
    __syncthreads();
    double a[8][8];
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) a[r][c] = s.U[ty + 16 * r + (tx + 16 * c) * LP];

    // Right-looking factorisation without square roots inside the sweep, with the inverse formed by the
    // SAME sweep (elimination applied to the identity):  S = L D L^T, U = D^1/2 L^T, and the row
    // operations that eliminate column j, applied to I, leave Y = L^-1 (unit lower), so that
    // U^-1 = Y^T D^-1/2.  The strictly-lower register positions (row > col), unused by the symmetric
    // factorisation, hold Y; its unit diagonal is implicit.
    //   step j: d_j = a(j,j), l_i = a(j,i) / d_j for i > j;
    //           a(i,c) -= l_i a(j,c)  (c >= i: Schur complement),
    //           Y(i,c) -= l_i Y(j,c)  (c <  j),   Y(i,j) = -l_i.
    // One pass of 128 dependent steps instead of two (the latency of a step -- barrier, broadcast,
    // reciprocal -- is paid once).
#pragma unroll
    for (int jr = 0; jr < 8; ++jr) {
#pragma unroll 1
        for (int jo = 0; jo < 16; ++jo) {
            const int j = jr * 16 + jo;
            double* rb = s.rowbuf + (j & 1) * LB;
            if (ty == jo) {   // the whole pivot row: Y(j, <j), d_j, a(j, >j)
#pragma unroll
                for (int c = 0; c < 8; ++c) rb[tx + 16 * c] = a[jr][c];
            }
            __syncthreads();
            const double d = rb[j];
            if (!(d > 0.0)) {   // uniform: every thread reads the same value
                if (t == 0) atomicCAS(info, 0, j0 + j + 1);
                return;
            }
            if (t == 0) s.dvec[j] = d;
            const double invd = 1.0 / d;
            const double pj = (tx == jo) ? 1.0 : rb[tx + 16 * jr];   // column group jr of the pivot row, Y(j,j) = 1
#pragma unroll
            for (int r = jr; r < 8; ++r)
                leaf_update_row(a, jr, r, rb, rb[ty + 16 * r] * invd, pj, (r > jr) || (ty > jo), tx, ty, jo);
        }
    }
    __syncthreads();
    if (t < LB) s.dinv[t] = 1.0 / sqrt(s.dvec[t]);
    __syncthreads();

    // scale rows; shared image = U (upper) with zeros below; write it out
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            double u = 0.0;
            if (row == col) u = sqrt(s.dvec[row]);
            else if (row < col) u = a[r][c] * s.dinv[row];
            s.U[row + col * LP] = u;
        }
    __syncthreads();
    leaf_store_all(s, blk, ld, nb, t);
    __syncthreads();   // the image is rewritten next

    // W = U^-1 = Y^T D^-1/2: the register at (row, col), row > col, is W(col, row) / dinv[row]
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            double w = 0.0;
            if (row == col) w = s.dinv[row];
            else if (row > col) w = a[r][c] * s.dinv[row];
            s.U[col + row * LP] = w;
        }
    __syncthreads();
    leaf_store_all(s, Winv, ldw, LB, t);
}

// ------------------------------------------------------------------------------------------------
// potrf_leaf4_kernel: the same result as potrf_leaf_kernel (U_kk in place, W = U_kk^-1 out) by a
// BLOCKED sweep over 32 panels of 4 rows.  The step of the rank-1 sweep is a latency chain (barrier,
// broadcast, reciprocal: ~940 cycles, profiles/r01f_leaf_ncu.md); here a panel costs two barriers, and
// its 4 x 4 diagonal block is factored by EVERY thread redundantly in registers (no communication
// inside the four dependent pivots), followed by one rank-4 update.
//
// The register image Z (thread (ty,tx) holds Z(ty + 16 r, tx + 16 c)) is the elimination applied to
// [S | I] at once: positions row <= col hold the Schur complement / finished rows of U, positions
// row > col hold Y = rows of U^-T as they form (W(col,row) at the end).  Panel p = rows 4p .. 4p+3
// (register row group r = p / 4, threads ty = 4 (p % 4) + q):
//   A  the owners publish the panel rows Z(K, :)                                            -> barrier
//   B  every thread: LDL^T of the 4 x 4 diagonal block with Y_KK formed by the same row operations
//   C  the owners finish their rows: R = U_KK^-T Z(K, :) = dinv (Z + Y_KK Z) over all columns, and publish
//      R (in-panel columns: the Y part)                                                      -> barrier
//   D  rank-4 update of every row below the panel: Z(i, c) -= sum_k R(k, i) R(k, c) over the live
//      columns (Y part: c <= panel end; Schur part: c >= i)
// ------------------------------------------------------------------------------------------------
constexpr int LQ = 4;                   // panel rows

// Panels 4r .. 4r+3 (r is a template parameter so that every register index is static).
// Returns false (in every thread alike) when a pivot is not positive.
template <int r>
__device__ __forceinline__ bool leaf4_group(double (&a)[8][8], double* Zp, double* Rb, int tx, int ty, int t, int j0, int* info)
{
#pragma unroll 1
    for (int sgrp = 0; sgrp < 4; ++sgrp) {
        const int p0 = 16 * r + 4 * sgrp;          // first row / column of the panel
        const bool owner = (ty >> 2) == sgrp;
        const int q = ty & 3;
        // ---- A
        if (owner) {
#pragma unroll
            for (int c = 0; c < 8; ++c) Zp[q * LB + tx + 16 * c] = a[r][c];
        }
        __syncthreads();
        // ---- B: 4 x 4 diagonal block, every thread alike (upper part from the image; Y starts as the identity)
        double z[LQ][LQ];
#pragma unroll
        for (int i = 0; i < LQ; ++i)
#pragma unroll
            for (int c = 0; c < LQ; ++c) z[i][c] = (c >= i) ? Zp[i * LB + p0 + c] : 0.0;
        double dinv[LQ];
#pragma unroll
        for (int j = 0; j < LQ; ++j) {
            const double d = z[j][j];
            if (!(d > 0.0)) {   // the same in every thread: uniform exit
                if (t == 0) atomicCAS(info, 0, j0 + p0 + j + 1);
                return false;
            }
            const double invd = 1.0 / d;
            dinv[j] = 1.0 / sqrt(d);
#pragma unroll
            for (int i = j + 1; i < LQ; ++i) {
                const double li = z[j][i] * invd;
#pragma unroll
                for (int c = 0; c < LQ; ++c) {
                    if (c >= i || c < j) z[i][c] = fma(-li, z[j][c], z[i][c]);
                    else if (c == j) z[i][c] = -li;              // Y(i,j): the pivot row's Y(j,j) is 1
                }
            }
        }
        // ---- C: the owners finish row q of the panel
        if (owner) {
            double yq[LQ - 1], dq = dinv[0], zqq = z[0][0];
#pragma unroll
            for (int k = 0; k < LQ - 1; ++k) yq[k] = 0.0;
#pragma unroll
            for (int i = 1; i < LQ; ++i)
                if (q == i) {
                    dq = dinv[i]; zqq = z[i][i];
#pragma unroll
                    for (int k = 0; k < LQ - 1; ++k) yq[k] = (k < i) ? z[i][k] : 0.0;
                }
            double acc[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                acc[c] = Zp[q * LB + tx + 16 * c];
#pragma unroll
                for (int k = 0; k < LQ - 1; ++k) acc[c] = fma(yq[k], Zp[k * LB + tx + 16 * c], acc[c]);   // yq[k] = 0 for k >= q
                acc[c] *= dq;
            }
            double pub = acc[r];
            const int qc = tx - 4 * sgrp;             // column inside the panel (c == r only)
            if (qc >= 0 && qc < LQ) {
                // row q of the factored block: z[q][qc] (static indexing through selects)
                double zq = 0.0;
#pragma unroll
                for (int i = 0; i < LQ; ++i)
#pragma unroll
                    for (int c = 0; c < LQ; ++c)
                        if (i == q && c == qc) zq = z[i][c];
                if (qc > q) { acc[r] = zq * dq; pub = 0.0; }              // U(q,qc)    | Y part above the diagonal is 0
                else if (qc == q) { acc[r] = zqq * dq; pub = dq; }         // U(k,k)     | W(k,k)
                else { acc[r] = zq * dq; pub = acc[r]; }                   // W(qc,q)
            }
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                a[r][c] = acc[c];
                Rb[q * LB + tx + 16 * c] = (c == r) ? pub : acc[c];
            }
        }
        __syncthreads();
        // ---- D: rank-4 update of the rows below the panel
        const bool ylive = tx <= 4 * sgrp + 3;        // column group r: Y part (columns up to the panel's end)
        const bool upper = tx >= ty;                  // diagonal register blocks: Schur part
        const bool rowact = ty >= 4 * sgrp + 4;       // row group r: rows below the panel
#pragma unroll
        for (int k = 0; k < LQ; ++k) {
            double cv[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) cv[c] = Rb[k * LB + tx + 16 * c];
            {   // rows of the panel's own group
                const double u = rowact ? -Rb[k * LB + ty + 16 * r] : 0.0;
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    if (c < r || c > r) a[r][c] = fma(u, cv[c], a[r][c]);
                    else if (ylive || upper) a[r][c] = fma(u, cv[c], a[r][c]);
                }
            }
#pragma unroll
            for (int rr = r + 1; rr < 8; ++rr) {
                const double u = -Rb[k * LB + ty + 16 * rr];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    if (c < r || c > rr) a[rr][c] = fma(u, cv[c], a[rr][c]);
                    else if (c == r) { if (ylive) a[rr][c] = fma(u, cv[c], a[rr][c]); }
                    else if (c == rr) { if (upper) a[rr][c] = fma(u, cv[c], a[rr][c]); }
                }
            }
        }
        // (the next panel's step A writes Zp, which nobody reads after step C; Rb is rewritten after the next barrier)
    }
    return true;
}

__global__ void __launch_bounds__(kLeafThreads, 1)
potrf_leaf4_kernel(double* __restrict__ S, long long ld, int N, int j0, double* __restrict__ Winv, long long ldw, int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const LeafSmem s = leaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int nb = min(LB, N - j0);
    double* blk = S + j0 + (long long)j0 * ld;

    leaf_load_upper(s, blk, ld, nb, t);
    __syncthreads();
    double a[8][8];
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) a[r][c] = s.U[ty + 16 * r + (tx + 16 * c) * LP];
    __syncthreads();   // the image is free now: the panel buffers live in it
    double* Zp = s.U;                        // [4][128] panel rows as published
    double* Rb = s.U + LQ * LB;              // [4][128] finished panel rows (in-panel columns: Y part)

    if (!leaf4_group<0>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<1>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<2>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<3>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<4>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<5>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<6>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    if (!leaf4_group<7>(a, Zp, Rb, tx, ty, t, j0, info)) return;
    __syncthreads();

    // shared image = U (upper) with zeros below; write it out
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            s.U[row + col * LP] = (row <= col) ? a[r][c] : 0.0;
        }
    __syncthreads();
    leaf_store_all(s, blk, ld, nb, t);
    __syncthreads();
    // W = U^-1: the register at (row, col), row > col, is W(col, row); W(k,k) = 1 / U(k,k)
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            double w = 0.0;
            if (row == col) w = 1.0 / a[r][c];
            else if (row > col) w = a[r][c];
            s.U[col + row * LP] = w;
        }
    __syncthreads();
    leaf_store_all(s, Winv, ldw, LB, t);
}

// One CTA per diagonal block b: V_bb = U_bb^-1.  Reads only the upper triangle of U_bb; writes the
// whole diagonal block of V (upper = inverse, strictly lower = 0).  A zero diagonal entry sets
// info = -(index+1) (reported as GS_ERR_SINGULAR).
__global__ void __launch_bounds__(kLeafThreads, 1)
trtri_leaf_kernel(const double* __restrict__ U, double* __restrict__ V, long long ld, int N, int* info)
{
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const LeafSmem s = leaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int j0 = blockIdx.x * LB;
    const int nb = min(LB, N - j0);
    const double* ub = U + j0 + (long long)j0 * ld;
    double* vb = V + j0 + (long long)j0 * ld;
    if (t == 0) *s.flag = 0;
    leaf_load_upper(s, ub, ld, nb, t);
    __syncthreads();
    if (t < LB) {
        const double u = s.U[t + t * LP];
        if (u == 0.0) atomicMax(s.flag, t + 1);
        s.dinv[t] = 1.0 / u;
    }
    __syncthreads();
    if (*s.flag != 0) {
        if (t == 0) {
            int first = LB;   // report the FIRST zero diagonal entry
            for (int i = LB - 1; i >= 0; --i)
                if (s.U[i + i * LP] == 0.0) first = i;
            atomicCAS(info, 0, -(j0 + first + 1));
        }
        return;
    }
    leaf_invert_upper(s, tx, ty);
    leaf_store_all(s, vb, ld, nb, t);
}

// Scans the first n diagonal entries of U (one CTA) and records the FIRST exact zero as info = -(index + 1)
// (GS_ERR_SINGULAR).  The leaf kernels find zeros too, but one CTA per block in no particular order: which
// block reports first would be a race, and "the first bad pivot" (include/gs.h) must not be.
template <typename T>
__global__ void __launch_bounds__(1024, 1) check_diagonal_kernel(const T* __restrict__ U, long long ld, int n, int* info)
{
    if (*info != 0) return;
    __shared__ int first;
    if (threadIdx.x == 0) first = n;
    __syncthreads();
    int mine = n;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const T u = U[i + (long long)i * ld];
        bool zero;
        if constexpr (sizeof(T) == 16) zero = (u.x == 0.0 && u.y == 0.0); else zero = (u == 0.0);
        if (zero && i < mine) mine = i;
    }
    if (mine < n) atomicMin(&first, mine);
    __syncthreads();
    if (threadIdx.x == 0 && first < n) atomicCAS(info, 0, -(first + 1));
}

// Zero the strictly-lower part of an N x N column-major matrix outside its 128 x 128 diagonal
// blocks (those are written whole by the leaf kernels): the "strictly-lower part is zero" contract
// of U and U^-1 (include/gs.h).
template <typename T, int kLB>
__global__ void zero_lower_blocks_kernel(T* __restrict__ X, long long ld, int N, const int* info)
{
    if (*info != 0) return;
    const int col = blockIdx.x;                // columns on grid.x (gridDim.y stops at 65535, N does not)
    const int first = (col / kLB + 1) * kLB;   // first row below the diagonal block of this column
    for (int row = first + blockIdx.y * blockDim.x + threadIdx.x; row < N; row += gridDim.y * blockDim.x)
        X[row + (long long)col * ld] = T{};
}

// Fused-exchange helper of the column-range inversion: copies, for every column c of [col0, col0 + ncols),
// the rows of the diagonal band it lies in (rows [band * floor(c / band), + band), clipped to N) from src to
// each of the n push targets (same layout).  That band -- the inverted diagonal panel blocks -- is the only
// part of a rank's U^-1 slab that the tile engine's own push (EngineParams::peer) does not carry.
struct PushTargets {
    void* ptr[8];
    int n;
};
template <typename T>
__global__ void push_band_kernel(const T* __restrict__ src, PushTargets dst, long long ld, int N, int col0, int band, const int* info)
{
    if (*info != 0) return;
    const int col = col0 + blockIdx.x;
    const int r0 = (col / band) * band;
    const int r1 = min(r0 + band, N);
    for (int row = r0 + blockIdx.y * blockDim.x + threadIdx.x; row < r1; row += gridDim.y * blockDim.x) {
        const long long off = row + (long long)col * ld;
        const T v = src[off];
        for (int d = 0; d < dst.n; ++d) static_cast<T*>(dst.ptr[d])[off] = v;
    }
}

// dst_d[drow0 + r, dcol0 + c] = src[srow0 + r, scol0 + c] for r < rows, c = blockIdx.x, for each of the n targets
// (all with leading dimension ldd): the pieces of the sharded factorisation (gs_cholesky_sharded) that no engine
// epilogue carries -- a finished row-panel piece, copied out of the workspace into the rank's own S and into every
// peer's S; the factored diagonal block and its inverse.  upper_only: only rows r <= c (a triangular block).
template <typename T>
__global__ void copy_block_push_kernel(const T* __restrict__ src, long long lds, int srow0, int scol0, PushTargets dst, long long ldd,
                                       int drow0, int dcol0, int rows, int upper_only, const int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    const int c = blockIdx.x;
    const int r = blockIdx.y * blockDim.x + threadIdx.x;
    if (r < rows && (!upper_only || r <= c)) {
        const T v = src[srow0 + r + (long long)(scol0 + c) * lds];
        const long long off = drow0 + r + (long long)(dcol0 + c) * ldd;
        for (int d = 0; d < dst.n; ++d) static_cast<T*>(dst.ptr[d])[off] = v;
    }
}

// dst[row0 + r, col0 + c] = src[row0 + r, col0 + c] for r < rows; one grid column (blockIdx.x) per column c.
template <typename T>
__global__ void copy_block_kernel(const T* __restrict__ src, T* __restrict__ dst, long long ld, int row0, int rows,
                                  int col0, const int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    const int r = blockIdx.y * blockDim.x + threadIdx.x;
    if (r < rows) {
        const long long off = row0 + r + (long long)(col0 + blockIdx.x) * ld;
        dst[off] = src[off];
    }
}

// X[l + i * ldx] = sqrt(f[l]) * C[i + l * ldc]  for i < N, l < nev: the occupation-weighted, transposed
// eigenvector block of gs_density_matrix (P_ij = sum_l f_l c*_li c_lj).  32 x 32 tiles
// through shared memory so that both the read (along i) and the write (along l) are coalesced.
template <typename T>
__global__ void transpose_scale_kernel(const T* __restrict__ C, long long ldc, const double* __restrict__ f, T* __restrict__ X,
                                       long long ldx, int N, int nev, const int* info)
{
    if (*info != 0) return;
    __shared__ T tile[32][33];
    const int i0 = blockIdx.x * 32, l0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int i = i0 + threadIdx.x, l = l0 + r;
        if (i < N && l < nev) tile[r][threadIdx.x] = C[i + (long long)l * ldc];
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int l = l0 + threadIdx.x, i = i0 + r;
        if (i < N && l < nev) {
            const double w = sqrt(f[l]);
            T v = tile[threadIdx.x][r];
            if constexpr (sizeof(T) == 16) { v.x *= w; v.y *= w; } else { v *= w; }
            X[l + (long long)i * ldx] = v;
        }
    }
}

}  // namespace gs
