// evp_dc.cuh -- kernels of the tridiagonal eigensolver (NEXT-4: the "Solve" stage of the standard eigenproblem,
// PAPER.md:126-133 Table 1 column "Solve"; "the solve step of the tridiagonal matrix"):
// Cuppen's divide and conquer with Gu / Eisenstat's stable eigenvector formula -- the method of LAPACK's xSTEDC
// and of ELPA's solve step, restated here for the GPU (nothing is copied from either).
//
//   T = diag(T1, T2) + beta (e_a e_b^T + e_b e_a^T) = diag(T1', T2') + |beta| w w^T,  w = e_a + sign(beta) e_b,
//   T1' = T1 - |beta| e_a e_a^T, T2' = T2 - |beta| e_b e_b^T.  With T1' = Q1 D1 Q1^T, T2' = Q2 D2 Q2^T:
//   T = Q (D + rho z z^T) Q^T,  Q = diag(Q1, Q2),  z = Q^T w / sqrt2,  rho = 2 |beta|.
//   * deflation: entries with rho |z_j| tiny, and pairs of (nearly) equal d rotated so that one z vanishes, are
//     eigenpairs already;
//   * the other k eigenvalues are the roots of  1 + rho sum_i z_i^2 / (d_i - lambda) = 0, one per interval
//     (d_j, d_j+1): found in mu = lambda - d_origin with the origin at the NEARER pole, so that every difference
//     d_i - lambda_j = (d_i - d_origin) - mu is formed without cancellation (a bracket shrunk until it cannot be halved:
//     regula falsi on f |mu| with a bisection safeguard, dc_secular_kernel);
//   * z is replaced by the z^ for which the computed lambda are the EXACT eigenvalues (Loewner's formula): the
//     eigenvectors x_j = (D - lambda_j)^-1 z^ / ||.|| are then orthogonal to working precision;
//   * the new eigenvector block is  Q X: two GEMMs on the FP64 tensor-core tile engine (top rows use only the
//     columns that come from Q1 or were mixed by a deflation rotation, bottom rows likewise) -- all the O(N^3) work.
// Leaves (kDcLeaf x kDcLeaf = 64 x 64) are solved by the implicit QL iteration, one CTA each.
//
// Eigenvalues of a solved block are kept sorted through an index (dcur ascending, idx -> physical column of Q),
// so no column is ever moved for the sake of ordering.  All arrays below are indexed by GLOBAL position
// (block offset + local index).
#pragma once
#include <cuda_runtime.h>

#include <cfloat>

namespace gs {
namespace evp {

constexpr int kDcLeaf = 64;       // (128: the leaves' QL iteration is 6 ms at any N; 32: one more level of small GEMMs costs more than the leaves gain from N = 8192 on)
constexpr int kDcLeafSmemBytes = kDcLeaf * kDcLeaf * 8;     // the leaf's Q block

struct MergeDesc {
    int off, n1, n2;     // block [off, off + n1 + n2): children [off, off + n1), [off + n1, off + n1 + n2)
    int k;               // number of non-deflated eigenvalues (device -> host)
    int c1, c2, c3;      // of those: columns from Q1 only / mixed by a rotation / from Q2 only (grouped order)
    int nrot;            // deflation rotations recorded
    int r;               // roots whose eigenVECTORS are wanted (host -> device; k except at the top level)
    int fail;
    double rho;
    double pad;
};

struct DcArrays {
    double* Qcur; double* Qnew; double* G; long long ldq;   // eigenvector blocks (block diagonal), gather buffer
    double* dcur; int* idx;        // solved blocks: eigenvalues ascending, physical column of each
    double* dnew; int* idxnew;     // the same for the level being formed
    double* dm; double* zs; int* srcm; int* typ;      // merged (sorted) D, z, source column, type 1 / 2 / 3
    double* dlam; double* wz; int* gsrc; int* gpos; int* gtyp;   // non-deflated: sorted d, z, source column, grouped position, type
    double* dval; int* dsrc; int* dtyp;                // deflated eigenvalues, their columns and types
    double* mu; int* org;          // roots: lambda_j = dlam[org_j] + mu_j
    double* zhat;
    int* rota; int* rotb; int* rotta; int* rottb; double* rotc; double* rots;   // rotations: columns, prior types, c, s
    MergeDesc* desc;
    int* info;                     // plan's failure flag
};

// ---------------------------------------------------------------------------------------------------------
// d(b-1) -= |e(b-1)|, d(b) -= |e(b-1)| at every leaf boundary b (all of them are cut points of some level)
// ---------------------------------------------------------------------------------------------------------
__global__ void dc_cut_kernel(double* d, const double* e, int N)
{
    const int b = (blockIdx.x * blockDim.x + threadIdx.x + 1) * kDcLeaf;
    if (b < N) {
        const double a = fabs(e[b - 1]);
        d[b - 1] -= a;
        d[b] -= a;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Leaf: all eigenpairs of the n x n (n <= kDcLeaf) tridiagonal block at offset off by the implicit QL iteration with
// Wilkinson shifts (EISPACK tql2 / LAPACK xSTEQR scheme).  Thread 0 runs the scalar recurrences of one sweep and
// leaves its rotations in shared memory; then every thread applies them to its own ROW of Q, which lives in dynamic
// shared memory (kDcLeaf^2 x 8 B = 32 KB per leaf; with 128 x 128 leaves in global memory every rotation was an L2 round trip: 7.75 -> see profiles/) and is
// written out once at the end.  Result: dcur ascending, idx = physical column.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kDcLeaf) dc_leaf_kernel(const double* __restrict__ dd, const double* __restrict__ ee, int N, DcArrays a)
{
    if (*a.info != 0) return;
    const int off = blockIdx.x * kDcLeaf;
    const int n = min(kDcLeaf, N - off);
    const int t = threadIdx.x;
    __shared__ double d[kDcLeaf], e[kDcLeaf], cs[kDcLeaf], sn[kDcLeaf];
    __shared__ int s_l, s_m, s_cnt, s_fail;
    extern __shared__ double dc_leaf_q[];        // the leaf's Q block (kDcLeaf x kDcLeaf, column-major): every sweep rewrites it
    if (t < n) { d[t] = dd[off + t]; e[t] = (t + 1 < n) ? ee[off + t] : 0.0; }
    double* Q = dc_leaf_q;
    constexpr long long ldq = kDcLeaf;
    for (int c = 0; c < n; ++c)
        if (t < n) Q[t + (long long)c * ldq] = (t == c) ? 1.0 : 0.0;
    if (t == 0) { s_fail = 0; }
    __syncthreads();
    for (int l = 0; l < n; ++l) {
        int iter = 0;
        while (true) {
            if (t == 0) {
                int m = l;
                for (; m < n - 1; ++m) {
                    const double ds = fabs(d[m]) + fabs(d[m + 1]);
                    if (fabs(e[m]) <= DBL_EPSILON * 0.5 * ds) break;
                }
                s_m = m;
                s_cnt = 0;
                if (m != l) {
                    if (iter == 60) s_fail = 1;
                    double g = (d[l + 1] - d[l]) / (2.0 * e[l]);
                    double r = hypot(g, 1.0);
                    g = d[m] - d[l] + e[l] / (g + copysign(r, g));
                    double s = 1.0, c = 1.0, p = 0.0;
                    int i = m - 1;
                    bool early = false;
                    for (; i >= l; --i) {
                        double f = s * e[i];
                        const double b = c * e[i];
                        // (this single-thread recurrence is the leaf's critical path: a plain square root and one
                        // reciprocal where they are safe, hypot and the divisions where f^2 + g^2 leaves the normal range)
                        const double q2 = f * f + g * g;
                        const bool plain = q2 > 1e-280 && q2 < 1e280;
                        r = plain ? sqrt(q2) : hypot(f, g);
                        e[i + 1] = r;
                        if (r == 0.0) { d[i + 1] -= p; e[m] = 0.0; early = true; break; }
                        if (plain) { const double rr = 1.0 / r; s = f * rr; c = g * rr; }
                        else { s = f / r; c = g / r; }
                        g = d[i + 1] - p;
                        r = (d[i] - g) * s + 2.0 * c * b;
                        p = s * r;
                        d[i + 1] = g + p;
                        g = c * r - b;
                        cs[i] = c; sn[i] = s;          // rotation of columns (i, i+1)
                    }
                    s_l = early ? i + 1 : l;           // rotations recorded for i = m-1 .. s_l
                    s_cnt = (m - 1) - s_l + 1;
                    if (!early) { d[l] -= p; e[l] = g; e[m] = 0.0; }
                }
            }
            __syncthreads();
            const int m = s_m;
            if (s_fail) break;
            if (m == l) break;
            // apply the sweep's rotations, i = m-1 down to s_l, to row t of Q
            if (t < n && s_cnt > 0) {
                const int lo = s_l;
                double hi_val = Q[t + (long long)m * ldq];            // z(t, i+1)
                for (int i = m - 1; i >= lo; --i) {
                    const double zi = Q[t + (long long)i * ldq];
                    const double c = cs[i], s = sn[i];
                    Q[t + (long long)(i + 1) * ldq] = s * zi + c * hi_val;
                    hi_val = c * zi - s * hi_val;
                }
                Q[t + (long long)lo * ldq] = hi_val;
            }
            ++iter;
            __syncthreads();
        }
        if (s_fail) break;
    }
    __syncthreads();
    if (s_fail) { if (t == 0) atomicCAS(a.info, 0, -(1 << 30)); return; }
    {   // the eigenvector block goes out once (rows over the threads: coalesced)
        double* Qg = a.Qcur + off + (long long)off * a.ldq;
        for (int c = 0; c < n; ++c)
            if (t < n) Qg[t + (long long)c * a.ldq] = Q[t + (long long)c * ldq];
    }
    // ascending order through an index (rank sort, ties by position)
    if (t < n) {
        const double v = d[t];
        int rank = 0;
        for (int j = 0; j < n; ++j) rank += (d[j] < v || (d[j] == v && j < t)) ? 1 : 0;
        a.dcur[off + rank] = v;
        a.idx[off + rank] = off + t;
    }
}

// ---------------------------------------------------------------------------------------------------------
// Eigenvalues only ("If the eigenvectors are needed, one has to perform the backtransformation", PAPER.md:67 -- and if
// they are not, neither they nor the divide and conquer are needed): the k-th smallest eigenvalue of tridiag(e, d, e),
// k < nev, by bisection on the Sturm count (Sylvester's inertia of T - x I = L D L^T: q_0 = d_0 - x,
// q_i = d_i - x - e_{i-1}^2 / q_{i-1}, count = number of negative q_i; the method of xSTEBZ), from the Gershgorin
// interval until the interval cannot be halved in FP64.  One thread per eigenvalue: the recurrence is a dependent
// chain of N rows per count, ~60 counts per eigenvalue, all eigenvalues side by side (49 ms for 4096 eigenvalues at N = 16384).
// ---------------------------------------------------------------------------------------------------------
constexpr int kBisectThreads = 32;      // one warp per CTA: the counts are bound by the FP64 pipe, which the warps of an SM share
__global__ void __launch_bounds__(kBisectThreads) tridiag_bisect_kernel(const double* __restrict__ d, const double* __restrict__ e, int N, int nev,
                                                             double* __restrict__ eps, const int* info)
{
    if (*info != 0) return;
    constexpr int kWarps = kBisectThreads / 32;
    __shared__ double s_lo[kWarps], s_hi[kWarps];
    const int t = threadIdx.x;
    double lo = d[0], hi = d[0];
    for (int i = t; i < N; i += kBisectThreads) {
        const double r = (i > 0 ? fabs(e[i - 1]) : 0.0) + (i + 1 < N ? fabs(e[i]) : 0.0);
        lo = fmin(lo, d[i] - r);
        hi = fmax(hi, d[i] + r);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((t & 31) == 0) { s_lo[t >> 5] = lo; s_hi[t >> 5] = hi; }
    __syncthreads();
    lo = s_lo[0];
    hi = s_hi[0];
#pragma unroll
    for (int w = 1; w < kWarps; ++w) {
        lo = fmin(lo, s_lo[w]);
        hi = fmax(hi, s_hi[w]);
    }
    const double pad = 2.0 * DBL_EPSILON * fmax(fabs(lo), fabs(hi)) * double(N) + 1e-300;
    lo -= pad;
    hi += pad;
    const int k = blockIdx.x * kBisectThreads + t;
    if (k >= nev) return;
    // The count in its product form: p_i = (d_i - x) p_{i-1} - e_{i-1}^2 p_{i-2} (the leading principal minors of T - x I;
    // q_i = p_i / p_{i-1}), count = number of sign changes, a zero taking the sign opposite to its predecessor's (q_i = 0
    // counts as negative).  Two dependent FMAs per row instead of a division; the pair (p_{i-1}, p_i) is rescaled by a power
    // of two whenever it leaves [2^-300, 2^300], and the matrix is scaled to unit size so that a step cannot jump the range.
    const double inv_sigma = 1.0 / fmax(fmax(fabs(lo), fabs(hi)), 1e-300);
    for (int it = 0; it < 2000; ++it) {
        const double mid = lo + 0.5 * (hi - lo);
        if (!(mid > lo && mid < hi)) break;
        int count = 0;
        double p0 = 0.0, p1 = 1.0;          // p_{i-2}, p_{i-1}
        bool neg = false;                   // sign of p_{i-1}
#pragma unroll 8
        for (int i = 0; i < N; ++i) {
            const double a = (d[i] - mid) * inv_sigma;
            const double b = (i == 0) ? 0.0 : e[i - 1] * inv_sigma;
            if (b == 0.0) p1 = neg ? -1.0 : 1.0;        // a new diagonal block starts: q_i = d_i - x, whatever the minors before
            const double pn = fma(a, p1, -(b * b) * p0);
            const bool nneg = pn < 0.0 || (pn == 0.0 && !neg);
            count += nneg != neg ? 1 : 0;
            neg = nneg;
            p0 = p1;
            p1 = pn;
            const double ap = fabs(pn);
            if (!(ap <= 0x1p300 && ap >= 0x1p-300) && ap != 0.0) {      // rare
                const double sc = ap > 0x1p300 ? 0x1p-300 : 0x1p300;
                p0 *= sc;
                p1 *= sc;
            }
        }
        if (count <= k) lo = mid; else hi = mid;
    }
    eps[k] = lo + 0.5 * (hi - lo);
}

// ---------------------------------------------------------------------------------------------------------
// M1: z = Q^T w / sqrt2 and the merge of the two sorted eigenvalue lists of a pair of children.
// grid.x = merge, 256 threads.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_setup_kernel(const double* __restrict__ e, DcArrays a)
{
    if (*a.info != 0) return;
    MergeDesc& ds = a.desc[blockIdx.x];
    const int off = ds.off, n1 = ds.n1, n2 = ds.n2, n = n1 + n2;
    const double beta = e[off + n1 - 1];
    const double sgn = beta < 0.0 ? -1.0 : 1.0;
    if (threadIdx.x == 0) ds.rho = 2.0 * fabs(beta);
    const double is2 = 0.70710678118654752440;
    const double* d1 = a.dcur + off;
    const double* d2 = a.dcur + off + n1;
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        double dv, zv;
        int col, rank, ty;
        if (j < n1) {
            dv = d1[j]; col = a.idx[off + j]; ty = 1;
            zv = a.Qcur[(off + n1 - 1) + (long long)col * a.ldq] * is2;            // last row of Q1
            int lo = 0, hi = n2;                                                    // # of d2 < dv
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (d2[mid] < dv) lo = mid + 1; else hi = mid; }
            rank = j + lo;
        } else {
            const int j2 = j - n1;
            dv = d2[j2]; col = a.idx[off + j]; ty = 3;
            zv = sgn * a.Qcur[(off + n1) + (long long)col * a.ldq] * is2;          // first row of Q2
            int lo = 0, hi = n1;                                                    // # of d1 <= dv
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (d1[mid] <= dv) lo = mid + 1; else hi = mid; }
            rank = j2 + lo;
        }
        a.dm[off + rank] = dv; a.zs[off + rank] = zv; a.srcm[off + rank] = col; a.typ[off + rank] = ty;
    }
}

// ---------------------------------------------------------------------------------------------------------
// M2: deflation scan, one CTA per merge.  The scan is sequential in the sorted order (an entry is compared with the
// last survivor, which a rotation may have changed), so one thread runs it -- but out of shared memory, which all
// threads fill in chunks, with the survivor's entry in registers (448 -> ~40 ns per entry: the loop used to be a chain
// of global-memory round trips), and with the hypot and the two divisions of the rotation test only where the test is
// not decided by a factor of two without them.  The grouped order of the survivors is then formed by all threads.
// ---------------------------------------------------------------------------------------------------------
constexpr int kDeflChunk = 1024;
__global__ void __launch_bounds__(256) dc_deflate_kernel(DcArrays a)
{
    if (*a.info != 0) return;
    MergeDesc& ds = a.desc[blockIdx.x];
    const int off = ds.off, n = ds.n1 + ds.n2;
    const int t = threadIdx.x;
    __shared__ double s_max[256];
    __shared__ double s_dm[kDeflChunk], s_z[kDeflChunk];
    __shared__ int s_src[kDeflChunk], s_typ[kDeflChunk];
    __shared__ int s_c[3][256];
    __shared__ int s_k;
    double mx = 0.0;
    for (int j = t; j < n; j += 256) mx = fmax(mx, fmax(fabs(a.dm[off + j]), fabs(a.zs[off + j])));
    s_max[t] = mx;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) s_max[t] = fmax(s_max[t], s_max[t + o]);
        __syncthreads();
    }
    const double tol = 8.0 * (DBL_EPSILON * 0.5) * s_max[0];
    const double rho = ds.rho;
    // thread 0: k survivors (compacted into dlam, wz, gsrc, gtyp), ndef deflated entries (dval, dsrc, dtyp), nrot rotations;
    // (p_*) = the last survivor so far, not yet written out
    int k = 0, ndef = 0, nrot = 0;
    bool have = false;
    double p_dm = 0.0, p_z = 0.0;
    int p_src = 0, p_typ = 0;
    auto defl = [&](double dv, int sv, int tv) { a.dval[off + ndef] = dv; a.dsrc[off + ndef] = sv; a.dtyp[off + ndef] = tv; ++ndef; };
    auto keep = [&](double dv, double zv, int sv, int tv) { a.dlam[off + k] = dv; a.wz[off + k] = zv; a.gsrc[off + k] = sv; a.gtyp[off + k] = tv; ++k; };
    for (int c0 = 0; c0 < n; c0 += kDeflChunk) {
        const int cn = min(kDeflChunk, n - c0);
        for (int i = t; i < cn; i += 256) {
            s_dm[i] = a.dm[off + c0 + i]; s_z[i] = a.zs[off + c0 + i]; s_src[i] = a.srcm[off + c0 + i]; s_typ[i] = a.typ[off + c0 + i];
        }
        __syncthreads();
        if (t == 0) {
            for (int jj = 0; jj < cn; ++jj) {
                const double dj = s_dm[jj], zj = s_z[jj];
                const int sj = s_src[jj], tj = s_typ[jj];
                if (rho * fabs(zj) <= tol) { defl(dj, sj, tj); continue; }
                if (!have) { have = true; p_dm = dj; p_z = zj; p_src = sj; p_typ = tj; continue; }
                const double tdiff = dj - p_dm;
                // |tdiff c s| = |tdiff| |z_j z_p| / (z_j^2 + z_p^2): beyond twice the tolerance the rotation test below fails for sure
                bool rotate = false;
                double c = zj, sn = p_z, tau = 0.0;
                if (!(fabs(tdiff) * fabs(zj * p_z) > 2.0 * tol * fma(zj, zj, p_z * p_z))) {
                    tau = hypot(c, sn);
                    c /= tau;
                    sn = -sn / tau;
                    rotate = fabs(tdiff * c * sn) <= tol;
                }
                if (rotate) {
                    a.rota[off + nrot] = p_src; a.rotb[off + nrot] = sj;
                    a.rotta[off + nrot] = p_typ; a.rottb[off + nrot] = tj;
                    a.rotc[off + nrot] = c; a.rots[off + nrot] = sn;
                    ++nrot;
                    const int ty = (p_typ != tj) ? 2 : tj;
                    const double tt = p_dm * c * c + dj * sn * sn;
                    const double dn = p_dm * sn * sn + dj * c * c;
                    defl(tt, p_src, ty);
                    p_dm = dn; p_z = tau; p_src = sj; p_typ = ty;
                } else {
                    keep(p_dm, p_z, p_src, p_typ);
                    p_dm = dj; p_z = zj; p_src = sj; p_typ = tj;
                }
            }
        }
        __syncthreads();
    }
    if (t == 0) {
        if (have) keep(p_dm, p_z, p_src, p_typ);
        s_k = k;
    }
    __syncthreads();
    // grouped order of the non-deflated columns: [from Q1 only | mixed | from Q2 only]; thread t owns a run of them
    k = s_k;
    const int len = (k + 255) / 256, q0 = min(t * len, k), q1 = min(q0 + len, k);
    int n1 = 0, n2 = 0, n3 = 0;
    for (int q = q0; q < q1; ++q) { const int ty = a.gtyp[off + q]; n1 += ty == 1; n2 += ty == 2; n3 += ty == 3; }
    s_c[0][t] = n1; s_c[1][t] = n2; s_c[2][t] = n3;
    __syncthreads();
    int c1 = 0, c2 = 0, c3 = 0, b1 = 0, b2 = 0, b3 = 0;       // totals, and the counts of the runs before this thread's
    for (int u = 0; u < 256; ++u) {
        const int v1 = s_c[0][u], v2 = s_c[1][u], v3 = s_c[2][u];
        if (u < t) { b1 += v1; b2 += v2; b3 += v3; }
        c1 += v1; c2 += v2; c3 += v3;
    }
    int p1 = b1, p2 = c1 + b2, p3 = c1 + c2 + b3;
    for (int q = q0; q < q1; ++q) {
        const int ty = a.gtyp[off + q];
        a.gpos[off + q] = ty == 1 ? p1++ : ty == 2 ? p2++ : p3++;
    }
    if (t == 0) { ds.k = k; ds.c1 = c1; ds.c2 = c2; ds.c3 = c3; ds.nrot = nrot; ds.fail = 0; }
}

// ---------------------------------------------------------------------------------------------------------
// M3: the deflation rotations applied to the columns of Q, one thread per row of the merged block.  A column
// that still belongs to one child only is zero outside that child's rows (the storage there is not read).
// grid = (row chunks, merges).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_rotate_kernel(DcArrays a)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, n1 = ds.n1, n = ds.n1 + ds.n2;
    const int lr = blockIdx.x * 256 + threadIdx.x;
    if (lr >= n || ds.nrot == 0) return;
    const bool top = lr < n1;
    double* Qr = a.Qcur + off + lr;
    for (int q = 0; q < ds.nrot; ++q) {
        const int ca = a.rota[off + q], cb = a.rotb[off + q];
        const int ta = a.rotta[off + q], tb = a.rottb[off + q];
        const double c = a.rotc[off + q], s = a.rots[off + q];
        const bool ina = ta == 2 || (ta == 1) == top, inb = tb == 2 || (tb == 1) == top;
        const double x = ina ? Qr[(long long)ca * a.ldq] : 0.0;
        const double y = inb ? Qr[(long long)cb * a.ldq] : 0.0;
        if (ta == tb && ta != 2 && !ina) continue;            // both columns are zero in this row and stay so
        Qr[(long long)ca * a.ldq] = c * x + s * y;
        Qr[(long long)cb * a.ldq] = c * y - s * x;
    }
}

// ---------------------------------------------------------------------------------------------------------
// M4: gather.  Non-deflated column q -> G[:, off + gpos(q)]; deflated column q' -> Qnew[:, off + k + q'].  All rows
// are written, zeros outside the column's support (the k-range of the bottom GEMM may start one column early,
// inside the columns that come from Q1 only: a TMA box of FP64 elements must start at an even row of X).
// grid = (columns of the block, merges), 256 threads stride over the rows.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_gather_kernel(DcArrays a)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, n1 = ds.n1, n = ds.n1 + ds.n2, k = ds.k;
    const int q = blockIdx.x;
    if (q >= n) return;
    int src, ty;
    double* dst;
    bool nondefl = q < k;
    if (nondefl) { src = a.gsrc[off + q]; ty = a.gtyp[off + q]; dst = a.G + off + (long long)(off + a.gpos[off + q]) * a.ldq; }
    else { src = a.dsrc[off + q - k]; ty = a.dtyp[off + q - k]; dst = a.Qnew + off + (long long)(off + q) * a.ldq; }
    const double* s = a.Qcur + off + (long long)src * a.ldq;
    for (int r = threadIdx.x; r < n; r += 256) {
        const bool in = ty == 2 || (ty == 1) == (r < n1);
        dst[r] = in ? s[r] : 0.0;
    }
}

// ---------------------------------------------------------------------------------------------------------
// M5: secular equation f(mu) = 1 + rho sum_i w_i^2 / ((d_i - d_origin) - mu) = 0, mu = lambda - d_origin with the origin
// at the nearer pole.  One warp per root j of every merge; a bracket [lo, hi] with f(lo) < 0 <= f(hi), one end of it the
// origin itself (mu = 0), is shrunk until it cannot be halved in FP64.  Plain bisection needs 55 - 70 evaluations of the
// O(k) sum per root; here the next point is the regula-falsi point of g(mu) = f(mu) |mu| -- the origin's pole removed:
// g = -+rho w_origin^2 + mu h(mu) with h smooth on the bracket, the other poles being at least half a gap away -- with the
// Illinois rule (the value at an end that survives twice is halved), and a bisection step whenever three such steps
// have not halved the bracket: 8 - 15 evaluations, the same stopping rule, the same sign decisions (those of f).
// grid = (ceil(maxk / 8), merges), 256 threads.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double secular_f(const double* __restrict__ dl, const double* __restrict__ w, int k, double dorg, double mu, double rho, int lane)
{
    double s = 0.0;
    for (int i = lane; i < k; i += 32) {
        const double wi = w[i];
        s += wi * wi / ((dl[i] - dorg) - mu);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    return 1.0 + rho * s;
}

__global__ void __launch_bounds__(256) dc_secular_kernel(DcArrays a)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, k = ds.k;
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (j >= k) return;
    const double* dl = a.dlam + off;
    const double* w = a.wz + off;
    const double rho = ds.rho;
    int org;
    double lo, hi, glo, ghi;                 // the bracket and g = f |mu| at its ends (the limit at the origin)
    if (j < k - 1) {
        const double gap = dl[j + 1] - dl[j];
        const double fm = secular_f(dl, w, k, dl[j], 0.5 * gap, rho, lane);
        if (fm >= 0.0) { org = j; lo = 0.0; hi = 0.5 * gap; glo = -rho * w[j] * w[j]; ghi = fm * hi; }                    // root in the left half: origin d_j
        else { org = j + 1; lo = -0.5 * gap; hi = 0.0; glo = fm * (0.5 * gap); ghi = rho * w[j + 1] * w[j + 1]; }         // right half: origin d_j+1
    } else {
        double w2 = 0.0;
        for (int i = lane; i < k; i += 32) w2 += w[i] * w[i];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) w2 += __shfl_xor_sync(0xffffffffu, w2, o);
        org = j; lo = 0.0; hi = rho * w2 * (1.0 + 4.0 * DBL_EPSILON);
        if (!(hi > 0.0)) hi = DBL_MIN;
        glo = -rho * w[j] * w[j];
        ghi = fmax(secular_f(dl, w, k, dl[j], hi, rho, lane) * hi, DBL_MIN);
    }
    const double dorg = dl[org];
    int since = 0, side = 0;                 // regula-falsi steps since the bracket last halved; the end moved last
    double wref = hi - lo;
    for (int it = 0; it < 1200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (!(mid > lo && mid < hi)) break;
        double x = mid;
        if (since < 3) {
            const double xs = lo - glo * ((hi - lo) / (ghi - glo));
            if (xs > lo && xs < hi) x = xs;
        }
        const double f = secular_f(dl, w, k, dorg, x, rho, lane);
        const double g = f * fabs(x);
        if (f >= 0.0) { hi = x; ghi = g; if (side > 0) glo *= 0.5; side = 1; }
        else { lo = x; glo = g; if (side < 0) ghi *= 0.5; side = -1; }
        if (since >= 3 || (++since == 3 && hi - lo <= 0.5 * wref)) { since = 0; wref = hi - lo; }
    }
    double mu = 0.5 * (lo + hi);
    if (mu == 0.0) mu = (org == j) ? hi : lo;          // never on the pole itself
    if (lane == 0) { a.mu[off + j] = mu; a.org[off + j] = org; }
}

// d_i - lambda_j from the shifted representation
__device__ __forceinline__ double dc_diff(const double* __restrict__ dl, const double* __restrict__ mu, const int* __restrict__ org, int i, int j)
{
    return (dl[i] - dl[org[j]]) - mu[j];
}

// ---------------------------------------------------------------------------------------------------------
// M6: z^_i (Loewner / Gu-Eisenstat), one warp per i:
//   z^_i^2 = (lambda_{k-1} - d_i) / rho * prod_{j<i} (d_i - lambda_j)/(d_i - d_j) * prod_{j>i} (lambda_{j-1} - d_i)/(d_j - d_i)
// every factor is positive by interlacing; sign taken from z_i.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_zhat_kernel(DcArrays a)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, k = ds.k;
    const int i = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (i >= k) return;
    const double* dl = a.dlam + off;
    const double* mu = a.mu + off;
    const int* org = a.org + off;
    double prod = 1.0;
    const double di = dl[i];
    for (int j = lane; j < k; j += 32) {
        if (j < i) prod *= dc_diff(dl, mu, org, i, j) / (di - dl[j]);
        else if (j > i) prod *= -dc_diff(dl, mu, org, i, j - 1) / (dl[j] - di);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) prod *= __shfl_xor_sync(0xffffffffu, prod, o);
    if (lane == 0) {
        const double last = -dc_diff(dl, mu, org, i, k - 1);        // lambda_{k-1} - d_i > 0
        const double z2 = prod * last / ds.rho;
        a.zhat[off + i] = copysign(sqrt(fmax(z2, 0.0)), a.wz[off + i]);
    }
}

// ---------------------------------------------------------------------------------------------------------
// M7: eigenvector x_j = (D - lambda_j)^-1 z^, normalised, written with its rows in the grouped order of the
// gathered columns: X[off + gpos(i), off + j].  One warp per root j < r.
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_xcols_kernel(DcArrays a, double* __restrict__ X)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, k = ds.k;
    const int j = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (j >= ds.r) return;
    const double* dl = a.dlam + off;
    const double* mu = a.mu + off;
    const int* org = a.org + off;
    double n2 = 0.0;
    for (int i = lane; i < k; i += 32) {
        const double x = a.zhat[off + i] / dc_diff(dl, mu, org, i, j);
        n2 += x * x;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) n2 += __shfl_xor_sync(0xffffffffu, n2, o);
    const double inv = 1.0 / sqrt(n2);
    double* col = X + off + (long long)(off + j) * a.ldq;
    for (int i = lane; i < k; i += 32) col[a.gpos[off + i]] = a.zhat[off + i] / dc_diff(dl, mu, org, i, j) * inv;
}

// ---------------------------------------------------------------------------------------------------------
// M8: eigenvalues of the merged block (roots, then deflated values) and their ascending index.
// Root j lives in column off + j of Qnew (j < r; no column otherwise: idx = -1), deflated q in column off + k + q.
// grid = (ceil(n / 256), merges).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dc_values_kernel(DcArrays a, double* __restrict__ val)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, n = ds.n1 + ds.n2, k = ds.k;
    const int x = blockIdx.x * 256 + threadIdx.x;
    if (x >= n) return;
    val[off + x] = x < k ? a.dlam[off + a.org[off + x]] + a.mu[off + x] : a.dval[off + x - k];
}

__global__ void __launch_bounds__(256) dc_rank_kernel(DcArrays a, const double* __restrict__ val)
{
    if (*a.info != 0) return;
    const MergeDesc ds = a.desc[blockIdx.y];
    const int off = ds.off, n = ds.n1 + ds.n2, k = ds.k;
    const int x = blockIdx.x * 256 + threadIdx.x;
    if (x >= n) return;
    const double v = val[off + x];
    int rank = 0;
    for (int y = 0; y < n; ++y) {
        const double vy = val[off + y];
        rank += (vy < v || (vy == v && y < x)) ? 1 : 0;
    }
    a.dnew[off + rank] = v;
    a.idxnew[off + rank] = (x < k && x >= ds.r) ? -1 : off + x;
}

// a block without a partner at this level passes through: its columns are copied to the other Q buffer
__global__ void __launch_bounds__(256) dc_copy_block_kernel(const double* __restrict__ src, double* __restrict__ dst, long long ld, int off, int n)
{
    const int c = blockIdx.x;
    for (int r = threadIdx.x; r < n; r += 256) dst[off + r + (long long)(off + c) * ld] = src[off + r + (long long)(off + c) * ld];
}

// Z(:, c) = Q(:, idx(c)), eps(c) = d(c) for the lowest nev pairs
__global__ void __launch_bounds__(256) dc_output_kernel(const double* __restrict__ Q, long long ldq, const double* __restrict__ d, const int* __restrict__ idx,
                                                        int N, int nev, double* __restrict__ eps, double* __restrict__ Z, long long ldz, int* info)
{
    if (*info != 0) return;
    const int c = blockIdx.x;
    if (c >= nev) return;
    const int src = idx[c];
    if (src < 0) { if (threadIdx.x == 0) atomicCAS(info, 0, -(1 << 30) - 1); return; }
    if (threadIdx.x == 0) eps[c] = d[c];
    for (int r = threadIdx.x; r < N; r += 256) Z[r + (long long)c * ldz] = Q[r + (long long)src * ldq];
}

}  // namespace evp
}  // namespace gs
