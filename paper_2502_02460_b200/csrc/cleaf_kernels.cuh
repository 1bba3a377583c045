// cleaf_kernels.cuh -- complex128 diagonal-block kernels (Hermitian path), 64 x 64 complex blocks.
//
//   potrf_cleaf_kernel : S_kk = U_kk^H U_kk in place (conjugate transpose per
//                        PAPER.md:67), real positive diagonal; also emits W_kk = U_kk^-1.
//   trtri_cleaf_kernel : invert every diagonal block of U, one CTA per block.
//
// Same scheme as leaf_kernels.cuh: 256 threads = 16 x 16, block distributed 2-D cyclically (thread
// (ty,tx) keeps elements (ty + 16 r, tx + 16 c), r,c = 0..3), rank-1 sweeps with the pivot row
// broadcast through a double-buffered shared row, coalesced global traffic through a padded shared
// image.  Only the real part of a diagonal entry of S is used (as in the oracle's definition).
#pragma once
#include <cuda_runtime.h>

#include "ptx.cuh"

namespace gs {

constexpr int CLB = 64;                  // complex leaf block order
constexpr int CLP = CLB + 1;             // padded shared pitch (complex elements)
constexpr int kCLeafThreads = 256;
constexpr int kCLeafSmemBytes = (CLB * CLP + 2 * CLB + CLB) * 16 + CLB * 8 + 16;   // U + rowbuf[2] + dinv + dvec + flag

struct CLeafSmem {
    double2* U;        // CLB x CLB column-major, pitch CLP
    double2* rowbuf;   // 2 x CLB
    double2* dinv;     // CLB : 1 / U(m,m)
    double* dvec;      // CLB
    int* flag;
};

__device__ __forceinline__ CLeafSmem cleaf_smem(unsigned char* raw)
{
    CLeafSmem s;
    s.U = reinterpret_cast<double2*>(raw);
    s.rowbuf = s.U + CLB * CLP;
    s.dinv = s.rowbuf + 2 * CLB;
    s.dvec = reinterpret_cast<double*>(s.dinv + CLB);
    s.flag = reinterpret_cast<int*>(s.dvec + CLB);
    return s;
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b)
{
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// a -= x * y
__device__ __forceinline__ void cfnma(double2& a, double2 x, double2 y)
{
    a.x = fma(-x.x, y.x, a.x);
    a.x = fma(x.y, y.y, a.x);
    a.y = fma(-x.x, y.y, a.y);
    a.y = fma(-x.y, y.x, a.y);
}

__device__ __forceinline__ void cleaf_load_upper(const CLeafSmem& s, const double2* blk, long long ld, int nb, int t)
{
    constexpr int kBatch = 8;   // independent loads in flight per thread (leaf_kernels.cuh: leaf_load_upper)
#pragma unroll 1
    for (int base = t; base < CLB * CLB; base += kCLeafThreads * kBatch) {
        double2 v[kBatch];
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * kCLeafThreads;
            const int row = idx & (CLB - 1), col = idx >> 6;
            v[u] = make_double2((row == col) ? 1.0 : 0.0, 0.0);
            if (row <= col && col < nb) v[u] = blk[row + (long long)col * ld];
        }
#pragma unroll
        for (int u = 0; u < kBatch; ++u) {
            const int idx = base + u * kCLeafThreads;
            s.U[(idx & (CLB - 1)) + (idx >> 6) * CLP] = v[u];
        }
    }
}

__device__ __forceinline__ void cleaf_store_all(const CLeafSmem& s, double2* dst, long long ld, int nb, int t)
{
    for (int idx = t; idx < CLB * CLB; idx += kCLeafThreads) {
        const int row = idx & (CLB - 1), col = idx >> 6;
        if (row < nb && col < nb) dst[row + (long long)col * ld] = s.U[row + col * CLP];
    }
}

// V = U^-1 (upper) for the U held in s.U with s.dinv[m] = 1 / U(m,m); result left in s.U.
__device__ __forceinline__ void cleaf_invert_upper(const CLeafSmem& s, int tx, int ty)
{
    double2 v[4][4];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) v[r][c] = make_double2((r == c && ty == tx) ? 1.0 : 0.0, 0.0);

#pragma unroll
    for (int mr = 3; mr >= 0; --mr) {
#pragma unroll 1
        for (int mo = 15; mo >= 0; --mo) {
            const int m = mr * 16 + mo;
            double2* rb = s.rowbuf + (m & 1) * CLB;
            if (ty == mo) {
                const double2 inv = s.dinv[m];
#pragma unroll
                for (int c = mr; c < 4; ++c) {
                    v[mr][c] = cmul(v[mr][c], inv);
                    rb[tx + 16 * c] = v[mr][c];
                }
            }
            __syncthreads();
#pragma unroll
            for (int r = 0; r <= mr; ++r) {
                const bool rowact = (r < mr) || (ty < mo);
                const double2 uk = s.U[ty + 16 * r + m * CLP];
#pragma unroll
                for (int c = mr; c < 4; ++c) {
                    const bool colact = (c > mr) || (tx >= mo);
                    if (rowact && colact) cfnma(v[r][c], uk, rb[tx + 16 * c]);
                }
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            s.U[row + col * CLP] = (row <= col) ? v[r][c] : make_double2(0.0, 0.0);
        }
    __syncthreads();
}

// One register row group of the fused factor-and-invert step (see leaf_update_row in leaf_kernels.cuh);
// rr = a(j,row) as published, the multiplier is conj(rr) / d.
__device__ __forceinline__ void cleaf_update_row(double2 (&a)[4][4], int jr, int r, const double2* rb, double2 rr, double invd,
                                                 double2 pj, bool rowact, int tx, int ty, int jo)
{
    const double2 ri = make_double2(rr.x * invd, -rr.y * invd);
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        if (c < jr) {
            if (rowact) cfnma(a[r][c], ri, rb[tx + 16 * c]);
        } else if (c == jr) {
            if (rowact && ((tx <= jo) || (r == jr && tx >= ty))) cfnma(a[r][c], ri, pj);
        } else if (c >= r) {
            if (rowact && ((c > r) || (tx >= ty))) cfnma(a[r][c], ri, rb[tx + 16 * c]);
        }
    }
}

__global__ void __launch_bounds__(kCLeafThreads, 1)
potrf_cleaf_kernel(double2* __restrict__ S, long long ld, int N, int j0, double2* __restrict__ Winv, long long ldw, int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const CLeafSmem s = cleaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int nb = min(CLB, N - j0);
    double2* blk = S + j0 + (long long)j0 * ld;

    cleaf_load_upper(s, blk, ld, nb, t);
    __syncthreads();
    double2 a[4][4];
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) a[r][c] = s.U[ty + 16 * r + (tx + 16 * c) * CLP];

    // One sweep forms U_kk and U_kk^-1 (leaf_kernels.cuh, potrf_leaf_kernel): S = L D L^H, U = D^1/2 L^H,
    // Y = L^-1 (unit lower, kept in the strictly-lower register positions), U^-1 = Y^H D^-1/2.
    //   step j: d_j = Re a(j,j), l_i = conj(a(j,i)) / d_j for i > j;
    //           a(i,c) -= l_i a(j,c) (c >= i);  Y(i,c) -= l_i Y(j,c) (c < j);  Y(i,j) = -l_i.
#pragma unroll
    for (int jr = 0; jr < 4; ++jr) {
#pragma unroll 1
        for (int jo = 0; jo < 16; ++jo) {
            const int j = jr * 16 + jo;
            double2* rb = s.rowbuf + (j & 1) * CLB;
            if (ty == jo) {
#pragma unroll
                for (int c = 0; c < 4; ++c) rb[tx + 16 * c] = a[jr][c];
            }
            __syncthreads();
            const double d = rb[j].x;
            if (!(d > 0.0)) {   // uniform
                if (t == 0) atomicCAS(info, 0, j0 + j + 1);
                return;
            }
            if (t == 0) s.dvec[j] = d;
            const double invd = 1.0 / d;
            const double2 pj = (tx == jo) ? make_double2(1.0, 0.0) : rb[tx + 16 * jr];
#pragma unroll
            for (int r = jr; r < 4; ++r)
                cleaf_update_row(a, jr, r, rb, rb[ty + 16 * r], invd, pj, (r > jr) || (ty > jo), tx, ty, jo);
        }
    }
    __syncthreads();
    if (t < CLB) {
        const double sd = sqrt(s.dvec[t]);
        s.dinv[t] = make_double2(1.0 / sd, 0.0);
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            double2 u = make_double2(0.0, 0.0);
            if (row == col) u.x = sqrt(s.dvec[row]);
            else if (row < col) { const double sc = s.dinv[row].x; u = make_double2(a[r][c].x * sc, a[r][c].y * sc); }
            s.U[row + col * CLP] = u;
        }
    __syncthreads();
    cleaf_store_all(s, blk, ld, nb, t);
    __syncthreads();   // the image is rewritten next

    // W = U^-1 = Y^H D^-1/2: the register at (row, col), row > col, is conj(W(col, row)) / dinv[row]
#pragma unroll
    for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int row = ty + 16 * r, col = tx + 16 * c;
            double2 w = make_double2(0.0, 0.0);
            if (row == col) w.x = s.dinv[row].x;
            else if (row > col) { const double sc = s.dinv[row].x; w = make_double2(a[r][c].x * sc, -a[r][c].y * sc); }
            s.U[col + row * CLP] = w;
        }
    __syncthreads();
    cleaf_store_all(s, Winv, ldw, CLB, t);
}

__global__ void __launch_bounds__(kCLeafThreads, 1)
trtri_cleaf_kernel(const double2* __restrict__ U, double2* __restrict__ V, long long ld, int N, int* info)
{
    if (*info != 0) return;
    extern __shared__ __align__(16) unsigned char leaf_raw[];
    const CLeafSmem s = cleaf_smem(leaf_raw);
    const int t = threadIdx.x, tx = t & 15, ty = t >> 4;
    const int j0 = blockIdx.x * CLB;
    const int nb = min(CLB, N - j0);
    const double2* ub = U + j0 + (long long)j0 * ld;
    double2* vb = V + j0 + (long long)j0 * ld;
    if (t == 0) *s.flag = 0;
    cleaf_load_upper(s, ub, ld, nb, t);
    __syncthreads();
    if (t < CLB) {
        const double2 u = s.U[t + t * CLP];
        const double n2 = u.x * u.x + u.y * u.y;
        if (n2 == 0.0) atomicMax(s.flag, t + 1);
        s.dinv[t] = make_double2(u.x / n2, -u.y / n2);
    }
    __syncthreads();
    if (*s.flag != 0) {
        if (t == 0) {
            int first = CLB;
            for (int i = CLB - 1; i >= 0; --i) {
                const double2 u = s.U[i + i * CLP];
                if (u.x == 0.0 && u.y == 0.0) first = i;
            }
            atomicCAS(info, 0, -(j0 + first + 1));
        }
        return;
    }
    cleaf_invert_upper(s, tx, ty);
    cleaf_store_all(s, vb, ld, nb, t);
}

}  // namespace gs
