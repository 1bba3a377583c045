// leaf_kernels.cuh -- latency-bound 128 x 128 diagonal-block kernels of the blocked factorisations.
//
//   potrf_leaf_kernel : factor one diagonal block S_kk = U_kk^T U_kk in place and also
//                       emit W_kk = U_kk^-1, which turns the panel solve U_k,: = U_kk^-T S_k,: into a
//                       tensor-core product.
//   trtri_leaf_kernel : invert every diagonal block of U, one CTA per block.
//
// One CTA of 256 threads = a 16 x 16 grid of threads, thread (ty,tx) keeps the 8 x 8 sub-block
// rows 8ty.., cols 8tx.. in registers.  Both factorisation and inversion are right-looking rank-1
// sweeps: the pivot row is broadcast through a double-buffered shared-memory row (one
// __syncthreads per step), the update is 64 register FMAs per thread.  Blocks shorter than 128
// (ragged last block) are padded with the identity, which factors / inverts to itself.
#pragma once
#include <cuda_runtime.h>

namespace gs {

constexpr int LB = 128;                 // leaf block order
constexpr int kLeafThreads = 256;
constexpr int kLeafSmemBytes = LB * LB * 8 + 2 * LB * 8 + LB * 8 + 16;   // Usm + rowbuf[2] + dvec + flag

struct LeafSmem {
    double* U;        // LB x LB column-major, pitch LB
    double* rowbuf;   // 2 x LB
    double* dvec;     // LB
    int* flag;
};

__device__ __forceinline__ LeafSmem leaf_smem(unsigned char* raw)
{
    LeafSmem s;
    s.U = reinterpret_cast<double*>(raw);
    s.rowbuf = s.U + LB * LB;
    s.dvec = s.rowbuf + 2 * LB;
    s.flag = reinterpret_cast<int*>(s.dvec + LB);
    return s;
}

// V = Usm^-1 (upper), result left in registers v[r][c] of the upper thread blocks (ty <= tx).
// Right-looking: for m = LB-1 .. 0: V(m,:) = acc(m,:) / U(m,m); acc(k,:) -= U(k,m) V(m,:) for k < m.
__device__ __forceinline__ void invert_upper_from_smem(const LeafSmem& s, double (&v)[8][8], int tx, int ty)
{
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int c = 0; c < 8; ++c) v[r][c] = (ty == tx && r == c) ? 1.0 : 0.0;

    for (int m = LB - 1; m >= 0; --m) {
        const int mb = m >> 3, mr = m & 7;
        double* rb = s.rowbuf + (m & 1) * LB;
        if (ty == mb && tx >= mb) {
            const double inv = 1.0 / s.U[m + m * LB];
#pragma unroll
            for (int r = 0; r < 8; ++r)
                if (r == mr) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) { v[r][c] *= inv; rb[8 * tx + c] = v[r][c]; }
                }
        }
        __syncthreads();
        if (ty <= mb && tx >= mb && tx >= ty) {
            double rc[8], uk[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) rc[c] = rb[8 * tx + c];
#pragma unroll
            for (int r = 0; r < 8; ++r) uk[r] = (8 * ty + r < m) ? s.U[8 * ty + r + m * LB] : 0.0;
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int c = 0; c < 8; ++c) v[r][c] = fma(-uk[r], rc[c], v[r][c]);
        }
    }
}

// S: N x N column-major (ld), block starts at (j0, j0), order nb = min(LB, N - j0).
// Winv: dense LB x LB column-major slot receiving U_kk^-1 (identity-padded).
// info: device flag; set (if still 0) to j0 + j + 1 when pivot j is not > 0.
__global__ void __launch_bounds__(kLeafThreads, 1)
potrf_leaf_kernel(double* __restrict__ S, long long ld, int N, int j0, double* __restrict__ Winv, int* info)
{
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const LeafSmem s = leaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int nb = min(LB, N - j0);
    double* blk = S + j0 + (long long)j0 * ld;

    double a[8][8];
    if (ty <= tx) {
#pragma unroll
        for (int c = 0; c < 8; ++c)
#pragma unroll
            for (int r = 0; r < 8; ++r) {
                const int row = 8 * ty + r, col = 8 * tx + c;
                a[r][c] = (row < nb && col < nb) ? blk[row + (long long)col * ld] : (row == col ? 1.0 : 0.0);
            }
    }
    if (t == 0) *s.flag = 0;
    __syncthreads();

    // right-looking factorisation without square roots inside the sweep:
    //   step j: d_j = a(j,j);  a(i,c) -= a(j,i) a(j,c) / d_j  (j < i <= c);  U(j,c) = a(j,c) / sqrt(d_j) afterwards
    for (int j = 0; j < LB; ++j) {
        const int jb = j >> 3, jr = j & 7;
        double* rb = s.rowbuf + (j & 1) * LB;
        if (ty == jb && tx >= jb) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
                if (r == jr) {
#pragma unroll
                    for (int c = 0; c < 8; ++c) rb[8 * tx + c] = a[r][c];
                }
        }
        __syncthreads();
        const double d = rb[j];
        if (!(d > 0.0)) {   // uniform: every thread reads the same value
            if (t == 0) atomicCAS(info, 0, j0 + j + 1);
            return;
        }
        if (t == 0) s.dvec[j] = d;
        if (ty >= jb && tx >= ty) {
            const double invd = 1.0 / d;
            double rc[8], ri[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) rc[c] = rb[8 * tx + c];
#pragma unroll
            for (int r = 0; r < 8; ++r) ri[r] = (8 * ty + r > j) ? rb[8 * ty + r] * invd : 0.0;
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int c = 0; c < 8; ++c) a[r][c] = fma(-ri[r], rc[c], a[r][c]);
        }
    }
    __syncthreads();

    // scale rows, write U to global (whole block: upper = U, strictly lower = 0) and to shared memory
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = 8 * ty + r, col = 8 * tx + c;
            double u = 0.0;
            if (ty <= tx && row <= col) {
                const double sd = sqrt(s.dvec[row]);
                u = (row == col) ? sd : a[r][c] / sd;
            }
            s.U[row + col * LB] = u;
            if (row < nb && col < nb) blk[row + (long long)col * ld] = u;
        }
    __syncthreads();

    double v[8][8];
    invert_upper_from_smem(s, v, tx, ty);
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = 8 * ty + r, col = 8 * tx + c;
            Winv[row + col * LB] = (ty <= tx && row <= col) ? v[r][c] : 0.0;
        }
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
    __syncthreads();
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = 8 * ty + r, col = 8 * tx + c;
            double u = (row == col) ? 1.0 : 0.0;
            if (row <= col && col < nb) u = ub[row + (long long)col * ld];
            if (row == col && u == 0.0) *s.flag = row + 1;
            s.U[row + col * LB] = u;
        }
    __syncthreads();
    if (*s.flag != 0) {
        if (t == 0) atomicCAS(info, 0, -(j0 + *s.flag));
        return;
    }
    double v[8][8];
    invert_upper_from_smem(s, v, tx, ty);
#pragma unroll
    for (int c = 0; c < 8; ++c)
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const int row = 8 * ty + r, col = 8 * tx + c;
            if (row < nb && col < nb) vb[row + (long long)col * ld] = (ty <= tx && row <= col) ? v[r][c] : 0.0;
        }
}

// Zero the strictly-lower part of an N x N column-major matrix outside its 128 x 128 diagonal
// blocks (those are written whole by the leaf kernels): the "strictly-lower part is zero" contract
// of U and U^-1 (include/gs.h).
__global__ void zero_lower_blocks_kernel(double* __restrict__ X, long long ld, int N, const int* info)
{
    if (*info != 0) return;
    const int col = blockIdx.y;
    const int first = (col / LB + 1) * LB;   // first row below the diagonal block of this column
    const int row = first + blockIdx.x * blockDim.x + threadIdx.x;
    if (row < N) X[row + (long long)col * ld] = 0.0;
}

}  // namespace gs
