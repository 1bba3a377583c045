// evp_tridiag.cuh -- kernels of the one-stage Householder tridiagonalisation  H~ = Q T Q^H  (NEXT-4: the
// "Tridiag." stage of the standard eigenproblem, "conventional one-stage diagonalization method
// (ELPA1)", Table 1 column "Tridiag."; the paper notes that on GPUs the one-stage solver is
// typically the faster one).
//
// Upper-triangle form: column i = N-1 .. 1 of the leading (unreduced) block is annihilated above the first
// superdiagonal by H(i) = I - tau v v^H, v(i-1) = 1, v(i:) = 0; Q = H(N-1) ... H(1).  Panels of nb columns are
// reduced against the STALE leading block with the usual lazy rank-2 corrections (V, W), and one HER2K-shaped
// launch of the tile engine applies  A -= V W^H + W V^H  after every panel.
//
// Half of the 4N^3/3 flop are the N matrix-vector products with the leading block: 0.5 flop per byte, i.e.
// HBM-bound (the FP64 ridge of this part is ~5.7 flop/B).  So the design goal of the step kernels is HBM
// traffic, not arithmetic: the symmetric product reads ONE triangle (4 m^2 bytes per step instead of 8 m^2:
// 4N^3/3 bytes over the whole reduction), every element feeding both y(r) += a u(c) and y(c) += conj(a) u(r).
//
// A step contains three global reductions that depend on each other (the matrix-vector product, the dot product
// w'^H v, the norm of the next column): S, C, F.  With a tensor map on A (complex, or real with even N) it is TWO
// launches -- symv_tma_kernel (S, with the F of the previous column formed inside it) and combine_kernel (C);
// finish_kernel (F) then runs only at the panel boundaries.  Without one (odd real N): symv_kernel, combine_kernel,
// finish_kernel, three launches per column.  Two identities shorten the chain:
//   * with u = the updated column a(0:i) BEFORE scaling, v = s (u - beta e_{i-1}), s = 1 / (alpha - beta): every
//     product with v is linear in u, so S multiplies by u and never waits for the norm; the scaling is applied
//     in C:  A v = s (A u - beta A(:, i-1)),  W^H v = s (W^H u - beta conj(W(i-1, :)));
//   * the part of the NEXT column's lazy update that involves the old panel columns is formed in the same pass
//     over the panels as the correction of w (C), so the panels are read once per step.
// Partial sums are combined in a fixed order (per-CTA partial buffers; the last CTA to arrive -- an atomic ticket
// -- adds them up), so the reduction is bit-reproducible.
//
// Panels are stored as conjugate transposes  Vt = V^H, Wt = W^H  (nb x N, leading dimension nb): that is the
// k-contiguous operand layout of the tile engine's HER2K-shaped launch, and it makes W^H u a plain product.
#pragma once
#include <cuda_runtime.h>

#include "ptx.cuh"

namespace gs {
namespace evp {

// ---- scalar helpers: T = double (real symmetric) or double2 (complex Hermitian, interleaved re/im) ----
__device__ __forceinline__ double zero_of(double) { return 0.0; }
__device__ __forceinline__ double2 zero_of(double2) { return make_double2(0.0, 0.0); }
__device__ __forceinline__ double cj(double a) { return a; }
__device__ __forceinline__ double2 cj(double2 a) { return make_double2(a.x, -a.y); }
__device__ __forceinline__ double re(double a) { return a; }
__device__ __forceinline__ double re(double2 a) { return a.x; }
__device__ __forceinline__ double abs2(double a) { return a * a; }
__device__ __forceinline__ double abs2(double2 a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ double mul(double a, double b) { return a * b; }
__device__ __forceinline__ double2 mul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double add(double a, double b) { return a + b; }
__device__ __forceinline__ double2 add(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double sub(double a, double b) { return a - b; }
__device__ __forceinline__ double2 sub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double rscale(double a, double r) { return a * r; }
__device__ __forceinline__ double2 rscale(double2 a, double r) { return make_double2(a.x * r, a.y * r); }
// acc + a * b
__device__ __forceinline__ double fmad(double a, double b, double acc) { return fma(a, b, acc); }
__device__ __forceinline__ double2 fmad(double2 a, double2 b, double2 acc)
{
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
    return acc;
}
// acc + conj(a) * b
__device__ __forceinline__ double cfmad(double a, double b, double acc) { return fma(a, b, acc); }
__device__ __forceinline__ double2 cfmad(double2 a, double2 b, double2 acc)
{
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(-a.y, b.x, acc.y);
    return acc;
}
__device__ __forceinline__ bool is_zero(double a) { return a == 0.0; }
__device__ __forceinline__ bool is_zero(double2 a) { return a.x == 0.0 && a.y == 0.0; }
__device__ __forceinline__ double real_only(double a) { return a; }
__device__ __forceinline__ double2 real_only(double2 a) { return make_double2(a.x, 0.0); }
__device__ __forceinline__ double from_real(double r, double) { return r; }
__device__ __forceinline__ double2 from_real(double r, double2) { return make_double2(r, 0.0); }
__device__ __forceinline__ double shfl_xor(double v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }
__device__ __forceinline__ double2 shfl_xor(double2 v, int m)
{
    return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}
__device__ __forceinline__ double ldcg(const double* p) { return __ldcg(p); }
__device__ __forceinline__ double2 ldcg(const double2* p) { return __ldcg(p); }

// Per-step scalars of the reduction, produced by the finalising CTAs and read by the next kernels.
template <typename T>
struct StepScalars {
    T tau;          // reflector scalar of the CURRENT step (H = I - tau v v^H); 0: H = I
    T s;            // 1 / (alpha - beta) (0 when tau == 0)
    T alpha2;       // -1/2 |tau|^2 (w'^H v), set by C's finaliser
    double beta;    // the new off-diagonal entry e(i-1)
    double xnorm2;  // ||x||^2 of the current column
    int pad[2];
};

// Householder scalars of a column with off-diagonal part (x, alpha):  H [x; alpha] = [0; beta]  (LAPACK xLARFG
// without the safmin rescaling loop).
__device__ __forceinline__ void householder_scalars(double alpha, double xnorm2, StepScalars<double>& sc)
{
    sc.xnorm2 = xnorm2;
    if (xnorm2 == 0.0) { sc.tau = 0.0; sc.s = 0.0; sc.beta = alpha; return; }
    const double beta = -copysign(sqrt(alpha * alpha + xnorm2), alpha);
    sc.beta = beta;
    sc.tau = (beta - alpha) / beta;
    sc.s = 1.0 / (alpha - beta);
}
__device__ __forceinline__ void householder_scalars(double2 alpha, double xnorm2, StepScalars<double2>& sc)
{
    sc.xnorm2 = xnorm2;
    if (xnorm2 == 0.0 && alpha.y == 0.0) { sc.tau = make_double2(0.0, 0.0); sc.s = make_double2(0.0, 0.0); sc.beta = alpha.x; return; }
    const double beta = -copysign(sqrt(alpha.x * alpha.x + alpha.y * alpha.y + xnorm2), alpha.x);
    sc.beta = beta;
    sc.tau = make_double2((beta - alpha.x) / beta, -alpha.y / beta);
    const double dr = alpha.x - beta, di = alpha.y, den = dr * dr + di * di;     // 1 / (alpha - beta)
    sc.s = make_double2(dr / den, -di / den);
}

// the scalars of step i live in sc[i & 1]: a launch that derives the next step's scalars (F, or S with F fused in)
// writes the other slot while its own CTAs may still be reading the current one
template <typename T> struct StepParams;
template <typename T> __device__ __forceinline__ StepScalars<T>* sc_of(const StepParams<T>& p, int step);

constexpr int kSymvThreads = 256;
constexpr int kSymvTW = 128;                        // tile width (columns): 8 warps x 16 columns
template <typename T> struct SymvGeom { static constexpr int RPT = 32 / int(sizeof(T)); static constexpr int TH = 32 * RPT; };

// Everything a step kernel needs.
template <typename T>
struct StepParams {
    T* A;                 // N x N column-major, ld = N; upper triangle of the leading m x m block is live
    long long ld;
    int N;
    int i;                // current column (S, C, F); the active block is A[0:i, 0:i]
    int jp;               // number of reflectors already in the panel (panel column of this step)
    int nb;               // panel width = leading dimension of Vt, Wt
    int itop;             // column index of panel column 0 (i = itop - jp)
    T* u;                 // N: the updated, unscaled current column a(0:i+1)
    T* wp;                // N: w' (C -> F)
    T* corr2;             // N: old-panel part of the next column's lazy update (C -> F)
    T* Vt;                // nb x N (ld nb): V^H of the panel
    T* Wt;                // nb x N (ld nb): W^H of the panel
    T* P1;                // [N][ldj] row-direction partials of y = A u: row r, column block J (the partials of a row lie side by side)
    long long ldj;
    T* P2;                // [nI][ldp] column-direction partials, indexed by row block
    long long ldp;
    T* Pt;                // [nJ][2 nb] partials of W^H u, V^H u
    T* tfin;              // 2 nb: tW' = W^H v, tV' = V^H v (scaled), final
    T* Pd;                // dot / norm partials (one per CTA)
    StepScalars<T>* sc;   // sc[0]: current step
    unsigned int* tickets;   // [4] atomic tickets (S panel-dot, C, F)
    double* d;            // N
    double* e;            // N
    T* tau;               // N
    T* R;                 // per-panel upper triangular M^H = conj(D) + striu(V^H V), block p at R + p * lb * (lb + 1), ld = lb
    int lb;               // block order of R (= nb)
    int panel;            // panel number (block of R)
    int mode;             // F: 0 = lazy next column (stale A + panel corrections), 1 = fresh (A is up to date), 2 = none
    int p2_chunk_rows;    // rows of A one P2 partial covers: TH (symv_kernel) or chunk_blocks * 128 (symv_tma_kernel)
    int fuse;             // symv_tma_kernel: the previous step's F (mode 0) is formed inside this launch (u_next_value)
    const int* info;
};

template <typename T> __device__ __forceinline__ StepScalars<T>* sc_of(const StepParams<T>& p, int step) { return p.sc + (step & 1); }

// Per-step indices of the device functions below; the step kernels take them from StepParams (step_idx).
struct StepIdx {
    int m;        // column i of this step = order of the active block
    int jp;       // its column in the panel
    int fuse;     // S: the F of the previous step is formed inside it
    int bar_id;   // 0: the callers are the whole CTA (__syncthreads); else its first nthr threads, meeting at this named barrier
    int nthr;
};
template <typename T> __device__ __forceinline__ StepIdx step_idx(const StepParams<T>& p) { return StepIdx{p.i, p.jp, p.fuse, 0, 0}; }
__device__ __forceinline__ void step_sync(const StepIdx& ix)
{
    if (ix.bar_id == 0) __syncthreads(); else named_bar_sync(ix.bar_id, ix.nthr);
}

// ---- F (mode 0) inside S: the next column, formed wherever it is needed -------------------------------------
// With io = p.i + 1 the step just combined (panel column jpo = p.jp - 1) and sc its scalars:
//   w(r) = tau w'(r) + alpha2 v(r),   u(r) = A(r, p.i) - corr2(r) - v(r) conj(w(io-1)) - w(r) conj(v(io-1)),  r <= p.i.
// Every operation is an explicit intrinsic (no contraction left to the compiler), so the CTAs that store u and
// those that only use it get the same bits.
__device__ __forceinline__ double fx_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double2 fx_mul(double2 a, double2 b)
{
    return make_double2(__fma_rn(-a.y, b.y, __dmul_rn(a.x, b.x)), __fma_rn(a.y, b.x, __dmul_rn(a.x, b.y)));
}
__device__ __forceinline__ double fx_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double2 fx_add(double2 a, double2 b) { return make_double2(__dadd_rn(a.x, b.x), __dadd_rn(a.y, b.y)); }
__device__ __forceinline__ double fx_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double2 fx_sub(double2 a, double2 b) { return make_double2(__dsub_rn(a.x, b.x), __dsub_rn(a.y, b.y)); }

template <typename T>
struct FusedF {
    T tau, alpha2, cwlast, cvlast;      // conj(w(io-1)), conj(v(io-1))
    int jpo, col;
    // alpha2_local: the caller's own copy of alpha2 of the step just combined; nullptr: read from sc
    __device__ __forceinline__ void init(const StepParams<T>& p, const StepIdx& ix, const T* alpha2_local = nullptr)
    {
        const StepScalars<T>* sc = sc_of(p, ix.m + 1);
        tau = ldcg(&sc->tau); alpha2 = alpha2_local != nullptr ? *alpha2_local : ldcg(&sc->alpha2);
        jpo = ix.jp - 1; col = ix.m;
        const T vlast = cj(p.Vt[jpo + (long long)col * p.nb]);
        const T wlast = fx_add(fx_mul(tau, p.wp[col]), fx_mul(alpha2, vlast));
        cwlast = cj(wlast); cvlast = cj(vlast);
    }
    __device__ __forceinline__ T w_of(const StepParams<T>& p, int r, T& v) const
    {
        v = cj(p.Vt[jpo + (long long)r * p.nb]);
        return fx_add(fx_mul(tau, p.wp[r]), fx_mul(alpha2, v));
    }
    __device__ __forceinline__ T u_of(const StepParams<T>& p, int r, T* w_out = nullptr) const
    {
        T v;
        const T w = w_of(p, r, v);
        T un = fx_sub(fx_sub(fx_sub(p.A[r + (long long)col * p.ld], p.corr2[r]), fx_mul(v, cwlast)), fx_mul(w, cvlast));
        if (r == col) un = real_only(un);
        if (w_out != nullptr) *w_out = w;
        return un;
    }
};

// ---------------------------------------------------------------------------------------------------------
// Panel dots of S (CTA x of nx, >= 256 threads of which the first 256 work):
//   Pt[x][c] = sum_{r in chunk x} Wt[c, r] u[r],  Pt[x][nb + c] likewise for Vt  (128-row chunks);
// the last CTA to arrive finalises tW' = s (W^H u - beta Wt[:, i-1]), tV' likewise, and the new column of
// M^H = conj(D) + striu(V^H V).  sm: 512 elements of shared memory.
// ---------------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ void panel_dots(const StepParams<T>& p, const StepIdx& ix, int x, int nx, T* sm, unsigned int* s_last,
                                           const T* alpha2_local = nullptr, int failed = 0)
{
    constexpr int TW = kSymvTW;
    const int m = ix.m, jp = ix.jp, nb = p.nb;
    const int t = threadIdx.x;
    if (jp == 0) return;
    const int r0 = x * TW, r1 = min(r0 + TW, m);
    if (ix.fuse) {
        // F of the previous step for the rows of this chunk (the last chunk also takes row m, the new diagonal entry):
        // column jp-1 of W, the next column u, the partial of ||u(0 : m-2)||^2; rows >= io of the reflector column io = 0
        FusedF<T> ff;
        ff.init(p, ix, alpha2_local);
        const int io = m + 1;
        double nrm = 0.0;
        const int r = (t < TW) ? r0 + t : ((t == TW && x == nx - 1) ? m : -1);
        if (r >= 0 && (r < r1 || r == m)) {
            T w;
            const T un = ff.u_of(p, r, &w);
            p.Wt[ff.jpo + (long long)r * nb] = cj(w);
            p.u[r] = un;
            if (r < m - 1) nrm = abs2(un);
        }
        if (failed == 0)      // (the only store of this function outside the workspace)
            for (int rz = io + x * kSymvThreads + t; rz < p.N && t < kSymvThreads; rz += nx * kSymvThreads) p.A[rz + (long long)io * p.ld] = zero_of(T{});
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
        double* sn = reinterpret_cast<double*>(sm);
        if ((t & 31) == 0) sn[t >> 5] = nrm;
        step_sync(ix);
        if (t == 0) {
            double sum = 0.0;
            for (int w = 0; w < (ix.bar_id == 0 ? int(blockDim.x) : ix.nthr) / 32; ++w) sum += sn[w];
            reinterpret_cast<double*>(p.Pd)[x] = sum;
        }
        step_sync(ix);      // the chunk's u and column jp-1 of Wt are read back below; sm is reused
    }
    const int groups = kSymvThreads / nb;            // nb = 128: 2 row groups; nb = 64: 4
    const int c = t % nb, g = t / nb;
    T aw = zero_of(T{}), av = zero_of(T{});
    if (t < kSymvThreads && c < jp) {
#pragma unroll 8
        for (int r = r0 + g; r < r1; r += groups) {
            const T ur = p.u[r];
            aw = fmad(p.Wt[c + (long long)r * nb], ur, aw);
            av = fmad(p.Vt[c + (long long)r * nb], ur, av);
        }
    }
    if (t < kSymvThreads) { sm[t] = aw; sm[kSymvThreads + t] = av; }
    step_sync(ix);
    if (t < nb) {
        T sw = zero_of(T{}), sv = zero_of(T{});
        for (int gg = 0; gg < groups; ++gg) { sw = add(sw, sm[gg * nb + t]); sv = add(sv, sm[kSymvThreads + gg * nb + t]); }
        p.Pt[(long long)x * 2 * nb + t] = sw;
        p.Pt[(long long)x * 2 * nb + nb + t] = sv;
    }
    __threadfence();
    step_sync(ix);
    if (t == 0) *s_last = (atomicAdd(&p.tickets[0], 1u) == unsigned(nx - 1)) ? 1u : 0u;
    step_sync(ix);
    if (!*s_last) return;
    __threadfence();
    if (ix.fuse) {
        // the scalars of this step from the norm of the new column (F's finaliser)
        if (t < 32) {
            double x2 = 0.0;
            for (int b = t; b < nx; b += 32) x2 += __ldcg(&reinterpret_cast<const double*>(p.Pd)[b]);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x2 += __shfl_xor_sync(0xffffffffu, x2, o);
            if (t == 0) {
                StepScalars<T> nx_sc;
                nx_sc.alpha2 = zero_of(T{});
                householder_scalars(ldcg(&p.u[m - 1]), x2, nx_sc);
                nx_sc.pad[0] = nx_sc.pad[1] = 0;
                *sc_of(p, m) = nx_sc;
            }
        }
        step_sync(ix);
    }
    // last chunk CTA: tW' = s (W^H u - beta Wt[:, i-1]),  tV' likewise;  the new column of M^H = conj(D) + striu(V^H V)
    const StepScalars<T> sc = *sc_of(p, m);   // (written by this CTA just above, or by a kernel before this one)
    if (t < 2 * nb) {
        const int cc = t % nb;
        const bool isV = t >= nb;
        T acc = zero_of(T{});
        if (cc < jp) {
            for (int xx = 0; xx < nx; ++xx) acc = add(acc, ldcg(&p.Pt[(long long)xx * 2 * nb + t]));
            const T rowv = (isV ? p.Vt : p.Wt)[cc + (long long)(m - 1) * nb];   // conj(W(i-1, c))
            acc = mul(sc.s, sub(acc, rscale(rowv, sc.beta)));
        }
        p.tfin[t] = acc;
        if (isV && cc < jp) {
            // G(a, b) = v_a^H v_b for a = itop - cc > b = i;  M^H(b - i0, a - i0) = conj(G(a, b)) with i0 = itop - lb + 1
            const int lb = p.lb, rowb = lb - 1 - jp, cola = lb - 1 - cc;
            p.R[(long long)p.panel * lb * (lb + 1) + rowb + (long long)cola * lb] = cj(acc);
        }
    }
    if (t == 0) p.tickets[0] = 0u;
}

// ---------------------------------------------------------------------------------------------------------
// S: partial sums of y = A[0:m, 0:m] u (m = i) from the UPPER triangle only, one CTA per (TH x 128) tile; the
// extra grid row (blockIdx.y == nI) forms W^H u and V^H u over 128-row chunks, and its last CTA finalises them.
// ---------------------------------------------------------------------------------------------------------
template <typename T, bool kVec>
__global__ void __launch_bounds__(kSymvThreads) symv_kernel(const StepParams<T> p)
{
    constexpr int RPT = SymvGeom<T>::RPT, TH = SymvGeom<T>::TH, TW = kSymvTW;
    grid_dep_launch();
    grid_dep_wait();
    if (*p.info != 0) return;
    const int m = p.i;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int nI = (m + TH - 1) / TH;
    __shared__ T red[8][TH];
    __shared__ unsigned int s_last;

    if (int(blockIdx.y) == nI) {
        panel_dots(p, step_idx(p), int(blockIdx.x), int(gridDim.x), &red[0][0], &s_last);
        return;
    }

    // ---- one tile of the upper triangle ----
    const int I = blockIdx.y, J = blockIdx.x;
    if (I * TH > J * TW + TW - 1 || I * TH >= m || J * TW >= m) return;
    const int r0 = I * TH + lane * RPT;
    const int c0 = J * TW + warp * 16;
    T ur[RPT], yr[RPT];
#pragma unroll
    for (int k = 0; k < RPT; ++k) {
        ur[k] = (r0 + k < m) ? p.u[r0 + k] : zero_of(T{});
        yr[k] = zero_of(T{});
    }
    const bool rows_in = r0 + RPT <= m;
#pragma unroll
    for (int cc = 0; cc < 16; cc += 8) {
        T a[8][RPT];
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int c = c0 + cc + q;
            const T* src = p.A + r0 + (long long)c * p.ld;
            // only tiles that reach the upper triangle are loaded: a thread whose rows lie below column c skips
            if (c < m && r0 <= c) {
                if (kVec && rows_in) {
                    if constexpr (sizeof(T) == 8) {
                        const double2 v0 = *reinterpret_cast<const double2*>(src);       // 16-byte aligned: even ld
                        const double2 v1 = *reinterpret_cast<const double2*>(src + 2);
                        a[q][0] = v0.x; a[q][1] = v0.y; a[q][2] = v1.x; a[q][3] = v1.y;
                    } else {
#pragma unroll
                        for (int k = 0; k < RPT; ++k) a[q][k] = src[k];
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < RPT; ++k) a[q][k] = (r0 + k < m) ? src[k] : zero_of(T{});
                }
            } else {
#pragma unroll
                for (int k = 0; k < RPT; ++k) a[q][k] = zero_of(T{});
            }
        }
#pragma unroll
        for (int q = 0; q < 8; ++q) {
            const int c = c0 + cc + q;
            const T uc = (c < m) ? p.u[c] : zero_of(T{});
            T yc = zero_of(T{});
#pragma unroll
            for (int k = 0; k < RPT; ++k) {
                const int r = r0 + k;
                T av = a[q][k];
                if (r > c || c >= m) av = zero_of(T{});          // strictly-lower part of the buffer is never used
                if (r == c) av = real_only(av);                   // Hermitian: real diagonal
                yr[k] = fmad(av, uc, yr[k]);
                if (r < c) yc = cfmad(av, ur[k], yc);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) yc = add(yc, shfl_xor(yc, o));
            if (lane == 0 && c < m) p.P2[(long long)I * p.ldp + c] = yc;
        }
    }
#pragma unroll
    for (int k = 0; k < RPT; ++k) red[warp][lane * RPT + k] = yr[k];
    __syncthreads();
    if (t < TH) {
        T s = red[0][t];
#pragma unroll
        for (int w = 1; w < 8; ++w) s = add(s, red[w][t]);
        const int r = I * TH + t;
        if (r < m) p.P1[(long long)r * p.ldj + J] = s;
    }
}

// ---------------------------------------------------------------------------------------------------------
// S, TMA form (the default whenever A admits a tensor map: complex, or real with even N).  Same partial sums as
// symv_kernel, other machinery -- the step is bound by the HBM stream of the triangle, so what matters is that
// the stream never stops and that little else is issued beside it:
//   * PERSISTENT CTAs (two per SM): a producer warp keeps a ring of 16 KB stages (TH rows x 16 columns, one TMA
//     box each) full across tile and work-item boundaries; eight consumer warps read the stages from shared
//     memory (conflict-free 16-byte loads), so no register is tied up by a load in flight.
//   * a work item is a COLUMN STRIP: chunk_blocks * 128 rows of one 128-column block.  The column sums
//     y(c) += conj(a(r,c)) u(r) stay in registers over the whole strip (a warp owns two columns of every stage,
//     a lane four rows) and are reduced across lanes once per strip by a transposing butterfly (16 shuffles
//     instead of 80); the row sums y(r) += a(r,c) u(c) of a tile are summed over the eight warps through shared
//     memory (one named barrier per tile, double-buffered).
//   * tiles strictly above the diagonal take a path without any per-element test; only the tiles that reach
//     the diagonal select (r <= c: the strictly-lower part of the buffer is never used; real diagonal).
//   Work items are dealt round-robin (item = cta, cta + G, ...): every partial has one owner and a fixed
//   summation order, so the result does not depend on scheduling.
// Leading CTAs (blockIdx.x < dot_ctas) form the panel dots instead (panel_dots).
// P1[r][J]: row sums of column block J; P2[q][c]: column sums of strip q (p2_chunk_rows = chunk_blocks * 128).
// ---------------------------------------------------------------------------------------------------------
constexpr int kSvStageBytes = 16384;                 // TH rows x 16 columns
constexpr int kSvConsumerWarps = 8;
constexpr int kSvThreads = (kSvConsumerWarps + 1) * 32;
constexpr int kSvRedBytes = 2 * kSvConsumerWarps * 1024;   // two buffers of 8 warps x TH elements
constexpr int kSvUcolBytes = 2 * kSymvTW * 16;             // u over the column block, two work items
constexpr int kSvUrowBytes = 2 * 1024;                     // u over the rows of a tile (TH elements), two tiles
// real: 16 column sums = 32 registers -> two CTAs of 5 stages per SM; complex: 64 registers -> one CTA of 10 stages
template <typename T> struct SvCfg {
    static constexpr int kStages = sizeof(T) == 8 ? 5 : 10;
    static constexpr int kCtasPerSm = sizeof(T) == 8 ? 2 : 1;
    static constexpr int kSmemBytes = kStages * kSvStageBytes + kSvRedBytes + kSvUcolBytes + kSvUrowBytes + 256 /*barriers*/ + 1024 /*alignment*/;
};

template <typename T>
struct SymvTmaParams {
    StepParams<T> s;
    CUtensorMap mapA;     // A as an (N * sizeof(T)/8) x N FP64 tensor; box = 128 doubles (TH rows) x 16 columns, no swizzle
    int chunk_blocks;     // 128-row blocks per work item (1, 2 or 4)
    int dot_ctas;         // leading CTAs that form the panel dots (0 when the panel is empty)
    int evict_first;      // the tiles of A are loaded with the L2 evict-first policy (the triangle does not fit the L2 anyway)
    int keep_blocks;      // ... except those of the column blocks below this one: the same tiles in every column of the reduction, kept in L2
};

// number of work items in the column blocks j < J:  sum_{j<J} ceil((j + 1) / K)
__host__ __device__ __forceinline__ int sv_items_before(int J, int K)
{
    const int a = J / K, b = J - a * K;
    return K * a * (a + 1) / 2 + b * (a + 1);
}
// strips of K blocks: the longest that still leaves every persistent CTA a few work items
__host__ __device__ __forceinline__ int sv_chunk_blocks(int nJ, int chunk_thresh)
{
    const long long nblocks = (long long)nJ * (nJ + 1) / 2;
    return nblocks >= chunk_thresh ? 4 : (2 * nblocks >= chunk_thresh ? 2 : 1);
}

// v[16] per lane -> the sum over the 32 lanes of v[idx], idx = bits 4..1 of the lane (both lanes of a pair hold it)
template <typename T>
__device__ __forceinline__ T sv_transpose_reduce(const T (&v)[16], int lane)
{
    T w8[8], w4[4], w2[2];
    const bool u16 = (lane & 16) != 0, u8 = (lane & 8) != 0, u4 = (lane & 4) != 0, u2 = (lane & 2) != 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) w8[i] = add(u16 ? v[i + 8] : v[i], shfl_xor(u16 ? v[i] : v[i + 8], 16));
#pragma unroll
    for (int i = 0; i < 4; ++i) w4[i] = add(u8 ? w8[i + 4] : w8[i], shfl_xor(u8 ? w8[i] : w8[i + 4], 8));
#pragma unroll
    for (int i = 0; i < 2; ++i) w2[i] = add(u4 ? w4[i + 2] : w4[i], shfl_xor(u4 ? w4[i] : w4[i + 2], 4));
    T w1 = add(u2 ? w2[1] : w2[0], shfl_xor(u2 ? w2[0] : w2[1], 2));
    return add(w1, shfl_xor(w1, 1));
}

// Shared memory of a streaming CTA and the running counters of its two roles.
template <typename T>
struct SvCta {
    unsigned char* stages;
    T *red, *ucol, *urow;
    uint32_t full0, empty0, qfull0, qempty0;
    volatile int* item_q;
    uint32_t cnt;          // stages issued (producer) / consumed (consumers)
    int nitem, ntile;      // queue slots written (producer) / read (consumers); tiles consumed
    __device__ __forceinline__ void carve(unsigned char* raw)
    {
        constexpr int kStages = SvCfg<T>::kStages;
        unsigned char* smem = raw + ((1024u - (smem_u32(raw) & 1023u)) & 1023u);
        stages = smem;
        red = reinterpret_cast<T*>(smem + kStages * kSvStageBytes);
        ucol = reinterpret_cast<T*>(smem + kStages * kSvStageBytes + kSvRedBytes);
        urow = reinterpret_cast<T*>(smem + kStages * kSvStageBytes + kSvRedBytes + kSvUcolBytes);
        uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kStages * kSvStageBytes + kSvRedBytes + kSvUcolBytes + kSvUrowBytes);
        full0 = smem_u32(bars); empty0 = smem_u32(bars + kStages); qfull0 = smem_u32(bars + 2 * kStages); qempty0 = smem_u32(bars + 2 * kStages + 4);
        item_q = reinterpret_cast<volatile int*>(bars + 2 * kStages + 8);
        cnt = 0; nitem = 0; ntile = 0;
    }
    __device__ __forceinline__ void init_barriers() const      // one thread
    {
        constexpr int kStages = SvCfg<T>::kStages;
        for (int s = 0; s < kStages; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, kSvConsumerWarps); }
        for (int s = 0; s < 4; ++s) { mbar_init(qfull0 + 8 * s, 1); mbar_init(qempty0 + 8 * s, kSvConsumerWarps); }
        mbar_fence_init();
    }
};

// item -> (column block J, first and one-past-last row tile): largest J with items_before(J) <= item
template <typename T>
__device__ __forceinline__ void sv_decode(int item, int nJ, int nI, int K, int& J, int& I0, int& I1)
{
    constexpr int R = kSymvTW / SymvGeom<T>::TH;      // row tiles per 128-row block
    int lo = 0, hi = nJ;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (sv_items_before(mid, K) <= item) lo = mid; else hi = mid;
    }
    J = lo;
    const int qq = item - sv_items_before(lo, K);
    I0 = qq * K * R;
    I1 = min(min((qq + 1) * K * R, (J + 1) * R), nI);
}

// Producer lane, one step (order of the active block m): streams every stage of every tile of the CTA's work items.
// The first item is `first` (< 0: none, the CTA starts with the counter), the others are dyn_base + the values of
// the atomic counter; every item goes to the consumers through the four-slot queue (full / empty barriers per slot),
// -1 ends the step.
template <typename T>
__device__ __forceinline__ void sv_produce_step(SvCta<T>& c, const CUtensorMap* map, int m, int K, int first, int dyn_base, unsigned int* counter,
                                                bool evict_first, int keep_blocks)
{
    const uint64_t policy = l2_policy_evict_first();
    constexpr int kStages = SvCfg<T>::kStages;
    constexpr int TH = SymvGeom<T>::TH, TW = kSymvTW, W8 = int(sizeof(T)) / 8;
    const int nJ = (m + TW - 1) / TW, nI = (m + TH - 1) / TH;
    const int nitems = sv_items_before(nJ, K);
    int item = first >= 0 ? first : dyn_base + int(atomicAdd(counter, 1u));
    for (;; ++c.nitem) {
        if (c.nitem >= 4) mbar_wait(c.qempty0 + 8 * (c.nitem & 3), ((c.nitem >> 2) - 1) & 1);   // the slot has been read
        c.item_q[c.nitem & 3] = item < nitems ? item : -1;
        mbar_arrive(c.qfull0 + 8 * (c.nitem & 3));
        if (item >= nitems) { ++c.nitem; break; }
        int J, I0, I1;
        sv_decode<T>(item, nJ, nI, K, J, I0, I1);
        for (int I = I0; I < I1; ++I) {
            for (int s = 0; s < TW / 16; ++s, ++c.cnt) {
                const uint32_t stage = c.cnt % kStages;
                if (c.cnt >= kStages) mbar_wait(c.empty0 + 8 * stage, ((c.cnt / kStages) - 1) & 1);
                mbar_arrive_expect_tx(c.full0 + 8 * stage, kSvStageBytes);
                if (evict_first && J >= keep_blocks) tma_load_2d_hint(smem_u32(c.stages + stage * kSvStageBytes), map, I * TH * W8, J * TW + 16 * s, c.full0 + 8 * stage, policy);
                else tma_load_2d(smem_u32(c.stages + stage * kSvStageBytes), map, I * TH * W8, J * TW + 16 * s, c.full0 + 8 * stage);
            }
        }
        // the next item is taken only now (the ring holds five stages of look-ahead, more than the counter's round
        // trip): a CTA that reserves its next item before streaming the current one leaves a tail of two items
        item = dyn_base + int(atomicAdd(counter, 1u));
    }
}

// Consumers (the first 256 threads), one step: warp w owns columns 2w, 2w+1 of every stage, lane l owns rows
// {l H .. l H + H-1} of each half tile; u(r) is stored by F, or (fuse) formed here from the previous step's vectors.
template <typename T>
__device__ __forceinline__ void sv_consume_step(SvCta<T>& c, const StepParams<T>& p, const StepIdx& ix, const FusedF<T>& ff, int K)
{
    constexpr int kStages = SvCfg<T>::kStages;
    constexpr int RPT = SymvGeom<T>::RPT, TH = SymvGeom<T>::TH, TW = kSymvTW, H = RPT / 2;
    constexpr int R = TW / TH;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int m = ix.m;
    const int nJ = (m + TW - 1) / TW, nI = (m + TH - 1) / TH;
    auto row_of = [&](int k) { return (k / H) * (TH / 2) + lane * H + (k % H); };
    auto u_val = [&](int r) -> T { return (r < m) ? (ix.fuse ? ff.u_of(p, r) : p.u[r]) : zero_of(T{}); };
    for (;; ++c.nitem) {
        mbar_wait(c.qfull0 + 8 * (c.nitem & 3), (c.nitem >> 2) & 1);
        const int item = c.item_q[c.nitem & 3];
        __syncwarp();
        if (lane == 0) mbar_arrive(c.qempty0 + 8 * (c.nitem & 3));
        if (item < 0) { ++c.nitem; break; }
        int J, I0, I1;
        sv_decode<T>(item, nJ, nI, K, J, I0, I1);
        T* uc = c.ucol + (c.nitem & 1) * TW;
        if (t < TW) uc[t] = u_val(J * TW + t);
        if (t < TH) c.urow[(c.ntile & 1) * TH + t] = u_val(I0 * TH + t);
        named_bar_sync(1, kSvConsumerWarps * 32);
        T yc[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) yc[i] = zero_of(T{});
        for (int I = I0; I < I1; ++I, ++c.ntile) {
            // the next tile's rows of u: loaded now, parked in shared memory before this tile's barrier
            T unext = zero_of(T{});
            const bool prefetch = (I + 1 < I1) && t < TH;
            if (prefetch) unext = u_val((I + 1) * TH + t);
            T ur[RPT];
#pragma unroll
            for (int k = 0; k < RPT; ++k) ur[k] = c.urow[(c.ntile & 1) * TH + row_of(k)];
            T yr[RPT];
#pragma unroll
            for (int k = 0; k < RPT; ++k) yr[k] = zero_of(T{});
            const bool masked = I * TH + TH - 1 >= J * TW;     // some element of the tile lies below the diagonal
#pragma unroll
            for (int s = 0; s < TW / 16; ++s) {
                const uint32_t stage = c.cnt % kStages;
                mbar_wait(c.full0 + 8 * stage, (c.cnt / kStages) & 1);
                if (c.cnt > 0) {                                 // release the previous stage (ptx.cuh: not right behind its loads)
                    __syncwarp();
                    if (lane == 0) mbar_arrive(c.empty0 + 8 * ((c.cnt - 1) % kStages));
                }
                ++c.cnt;
                const unsigned char* sp = c.stages + stage * kSvStageBytes + (2 * warp) * (TH * int(sizeof(T)));
                T a[2][RPT];
#pragma unroll
                for (int j = 0; j < 2; ++j) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const double2 v = *reinterpret_cast<const double2*>(sp + j * (TH * int(sizeof(T))) + h * (TH / 2) * int(sizeof(T)) + lane * 16);
                        if constexpr (sizeof(T) == 8) { a[j][2 * h] = v.x; a[j][2 * h + 1] = v.y; }
                        else { a[j][h] = v; }
                    }
                }
                const T u0 = uc[16 * s + 2 * warp], u1 = uc[16 * s + 2 * warp + 1];
                if (!masked) {
#pragma unroll
                    for (int k = 0; k < RPT; ++k) {
                        yr[k] = fmad(a[0][k], u0, yr[k]);
                        yr[k] = fmad(a[1][k], u1, yr[k]);
                        yc[2 * s] = cfmad(a[0][k], ur[k], yc[2 * s]);
                        yc[2 * s + 1] = cfmad(a[1][k], ur[k], yc[2 * s + 1]);
                    }
                } else {
                    const int c0 = J * TW + 16 * s + 2 * warp;
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const int cc = c0 + j;
#pragma unroll
                        for (int k = 0; k < RPT; ++k) {
                            const int r = I * TH + row_of(k);
                            T av = (r <= cc) ? a[j][k] : zero_of(T{});
                            if (r == cc) av = real_only(av);
                            yr[k] = fmad(av, j == 0 ? u0 : u1, yr[k]);
                            if (r < cc) yc[2 * s + j] = cfmad(av, ur[k], yc[2 * s + j]);
                        }
                    }
                }
            }
            // row sums of the tile over the eight warps
            T* rb = c.red + ((c.ntile & 1) * kSvConsumerWarps + warp) * TH;
#pragma unroll
            for (int k = 0; k < RPT; ++k) rb[row_of(k)] = yr[k];
            if (prefetch) c.urow[((c.ntile + 1) & 1) * TH + t] = unext;
            named_bar_sync(2, kSvConsumerWarps * 32);
            if (t < TH) {
                const T* rr = c.red + (c.ntile & 1) * kSvConsumerWarps * TH + t;
                T sum = rr[0];
#pragma unroll
                for (int w = 1; w < kSvConsumerWarps; ++w) sum = add(sum, rr[w * TH]);
                const int r = I * TH + t;
                if (r < m) p.P1[(long long)r * p.ldj + J] = sum;
            }
        }
        // column sums of the strip
        const T ysum = sv_transpose_reduce(yc, lane);
        if ((lane & 1) == 0) {
            const int idx = lane >> 1;                          // = 2 s + j
            const int cc = J * TW + 16 * (idx >> 1) + 2 * warp + (idx & 1);
            if (cc < m) p.P2[(long long)(I0 / (K * R)) * p.ldp + cc] = ysum;
        }
    }
}

// ---- Timeline of one column (trace build only: `python -m paper_2502_02460_b200.trace_tridiag`, -DGS_SV_TRACE) ----
// %globaltimer stamps of the S launches of the blocks of order trace_m and trace_m - 1, per CTA: [0] entry (before the
// grid dependency), [1] dependency resolved, [2] first work item, [3] end, [4] items, [5] tiles, [6] SM, [7] 1 = panel-dot
// CTA; of the C launches: earliest entry, earliest start after the dependency, latest end.
#ifdef GS_SV_TRACE
constexpr int kTraceCtas = 600;
__device__ unsigned long long g_sv_trace[2][kTraceCtas][8];
__device__ unsigned long long g_c_trace[2][4];
__device__ int g_sv_trace_m = -1;
__device__ __forceinline__ unsigned long long trace_time() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }
#define GS_TRACE(...) __VA_ARGS__
#else
#define GS_TRACE(...)
#endif

template <typename T>
__global__ void __launch_bounds__(kSvThreads, SvCfg<T>::kCtasPerSm) symv_tma_kernel(const __grid_constant__ SymvTmaParams<T> q)
{
    const StepParams<T>& p = q.s;
    extern __shared__ unsigned char sv_smem_raw[];
    SvCta<T> c;
    c.carve(sv_smem_raw);
    __shared__ unsigned int s_last;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    if (t == 0) {
        c.init_barriers();
        tma_prefetch_desc(&q.mapA);
    }
    __syncthreads();
    GS_TRACE(const unsigned long long tr_entry = trace_time();)
    grid_dep_launch();
    grid_dep_wait();
    // The info flag is read here and consumed only where something outside the workspace is stored (the panel-dot CTAs
    // zero a column of A): a branch on it at this point would put one more L2 round trip in front of every column.  With
    // the flag set the kernel runs on whatever the workspace holds -- fixed trip counts, stores into the workspace only.
    const int failed = *reinterpret_cast<const volatile int*>(p.info);
    const StepIdx ix = step_idx(p);
    GS_TRACE(const int tr_slot = g_sv_trace_m - ix.m;
             unsigned long long* tr = ((tr_slot == 0 || tr_slot == 1) && blockIdx.x < kTraceCtas && t == 0) ? g_sv_trace[tr_slot][blockIdx.x] : nullptr;
             if (tr) { tr[0] = tr_entry; tr[1] = trace_time(); tr[7] = int(blockIdx.x) < q.dot_ctas ? 1 : 0; })
    if (int(blockIdx.x) < q.dot_ctas) {
        panel_dots(p, ix, int(blockIdx.x), q.dot_ctas, c.red, &s_last, static_cast<const T*>(nullptr), failed);
        GS_TRACE(if (tr) tr[3] = trace_time();)
        return;
    }
    // Work items: the first one of a CTA is its own index, the rest comes from a global counter (tickets[3], reset by
    // the C kernel that follows), so the CTAs that start late (behind the panel-dot CTAs) simply take fewer items.
    const int cta = int(blockIdx.x) - q.dot_ctas, G = int(gridDim.x) - q.dot_ctas;
    if (warp == kSvConsumerWarps) {
        if (lane == 0) sv_produce_step(c, &q.mapA, ix.m, q.chunk_blocks, cta, G, p.tickets + 3, q.evict_first != 0, q.keep_blocks);
        return;
    }
    FusedF<T> ff;
    if (ix.fuse) ff.init(p, ix);
    GS_TRACE(if (tr) tr[2] = trace_time();)
    sv_consume_step(c, p, ix, ff, q.chunk_blocks);
    GS_TRACE(if (tr) { unsigned int sm; asm volatile("mov.u32 %0, %%smid;" : "=r"(sm)); tr[3] = trace_time(); tr[4] = c.nitem; tr[5] = c.ntile; tr[6] = sm; })
}

// ---------------------------------------------------------------------------------------------------------
// C: per row r < m = i (16 rows per CTA, 16 threads per row):
//   y      = sum of the partials of S
//   v(r)   = s (u(r) - beta [r == i-1])                       -> Vt[jp, r] = conj(v), A(r, i) = v   (clean reflector)
//   w'(r)  = s (y - beta A(r, i-1)) - sum_c ( V(r,c) tW'(c) + W(r,c) tV'(c) )
//   corr2  = sum_c ( V(r,c) conj(W(i-1,c)) + W(r,c) conj(V(i-1,c)) )     (old panel columns of the next lazy update)
//   partial of w'^H v; the last CTA sets alpha2 = -1/2 |tau|^2 (w'^H v) and records d(i), e(i-1), tau(i).
// ---------------------------------------------------------------------------------------------------------
// threads per row: 16 up to mid sizes; 8 for the largest blocks, where 16 would make the launch more than one wave of CTAs

// tW', tV' and row i-1 of the panels into shared memory (2 * 128 elements each), by the first nthr threads of the CTA
template <typename T>
__device__ __forceinline__ void combine_load(const StepParams<T>& p, const StepIdx& ix, T* s_t, T* s_row, int nthr)
{
    const int nb = p.nb;
    for (int c = threadIdx.x; c < 2 * nb; c += nthr) {
        const int cc = c % nb;
        s_t[c] = (cc < ix.jp) ? p.tfin[c] : zero_of(T{});
        s_row[c] = (cc < ix.jp) ? (c < nb ? p.Wt : p.Vt)[cc + (long long)(ix.m - 1) * nb] : zero_of(T{});
    }
}

// rows [g * kCombineRows, (g + 1) * kCombineRows), kCombineRows = 256 / kCombineTPR, by 256 threads; returns the thread's share of w'^H v (its row's
// term in the threads that own a row, zero elsewhere)
template <typename T, int kCombineTPR>
__device__ __forceinline__ T combine_group(const StepParams<T>& p, const StepIdx& ix, const StepScalars<T>& sc, const T* s_t, const T* s_row, int g, int failed)
{
    constexpr int TW = kSymvTW;
    constexpr int kCombineRows = 256 / kCombineTPR;
    const int m = ix.m, jp = ix.jp, nb = p.nb;
    const int t = threadIdx.x, l8 = t % kCombineTPR, rr = t / kCombineTPR;
    const int r = g * kCombineRows + rr;
    T dotp = zero_of(T{});
    T y = zero_of(T{}), c1 = zero_of(T{}), c2 = zero_of(T{});
    T ur = zero_of(T{}), acol = zero_of(T{});
    if (r < m) {
        // Every load of the row is independent of every other: they are issued in blocks of eight predicated loads
        // per array (a dependent chain of L2 round trips is what this kernel's time consists of).
        if (l8 == 0) { ur = p.u[r]; acol = p.A[r + (long long)(m - 1) * p.ld]; }
        // y(r): P1[r][J] for J >= r / TW (one contiguous run per row), P2[I][r] for I <= r / p2_chunk_rows
        const int nJ = (m + TW - 1) / TW;
        const T* p1 = p.P1 + (long long)r * p.ldj;
        for (int J0 = r / TW + l8; J0 < nJ; J0 += 8 * kCombineTPR) {
            T v8[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) { const int J = J0 + k * kCombineTPR; v8[k] = J < nJ ? p1[J] : zero_of(T{}); }
#pragma unroll
            for (int k = 0; k < 8; ++k) y = add(y, v8[k]);
        }
        const int nP2 = r / p.p2_chunk_rows + 1;
        for (int I0 = l8; I0 < nP2; I0 += 4 * kCombineTPR) {
            T v4[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) { const int I = I0 + k * kCombineTPR; v4[k] = I < nP2 ? p.P2[(long long)I * p.ldp + r] : zero_of(T{}); }
#pragma unroll
            for (int k = 0; k < 4; ++k) y = add(y, v4[k]);
        }
    }
    // The first block of the row's panel entries is loaded before the barrier that publishes s_t and s_row (staged by
    // combine_load), so that the staging and the row's own loads are one round trip to the L2, not two.
    const T* vt = p.Vt + (long long)r * nb;
    const T* wt = p.Wt + (long long)r * nb;
    T vv[8], ww[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int c = l8 + k * kCombineTPR;
        const bool in = r < m && c < jp;
        vv[k] = in ? vt[c] : zero_of(T{});
        ww[k] = in ? wt[c] : zero_of(T{});
    }
    __syncthreads();
    if (r < m) {
        for (int c0 = l8; c0 < jp; c0 += 8 * kCombineTPR) {
            if (c0 != l8) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const int c = c0 + k * kCombineTPR;
                    vv[k] = c < jp ? vt[c] : zero_of(T{});
                    ww[k] = c < jp ? wt[c] : zero_of(T{});
                }
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int c = min(c0 + k * kCombineTPR, nb - 1);   // (beyond jp: vv = ww = 0 and the entries of s_t, s_row are zero)
                const T vrc = cj(vv[k]), wrc = cj(ww[k]);             // V(r,c), W(r,c)
                c1 = fmad(vrc, s_t[c], c1);
                c1 = fmad(wrc, s_t[nb + c], c1);
                c2 = fmad(vrc, s_row[c], c2);                          // V(r,c) conj(W(i-1,c)) : s_row[c] = Wt[c, i-1] = conj(W(i-1,c))
                c2 = fmad(wrc, s_row[nb + c], c2);
            }
        }
    }
    // (all 32 lanes take part in the shuffles: a warp holds several rows, some of which may lie beyond m)
#pragma unroll
    for (int o = kCombineTPR / 2; o > 0; o >>= 1) { y = add(y, shfl_xor(y, o)); c1 = add(c1, shfl_xor(c1, o)); c2 = add(c2, shfl_xor(c2, o)); }
    if (r < m && l8 == 0) {
        T v = mul(sc.s, (r == m - 1) ? sub(ur, from_real(sc.beta, T{})) : ur);
        if (r == m - 1 && !is_zero(sc.s)) v = from_real(1.0, T{});   // (an identity reflector keeps v = 0)
        if (r == m - 1) acol = real_only(acol);
        T wpr = sub(mul(sc.s, sub(y, rscale(acol, sc.beta))), c1);
        p.Vt[jp + (long long)r * nb] = cj(v);
        if (failed == 0) p.A[r + (long long)m * p.ld] = v;          // (with d, e, tau the only stores of C outside the workspace)
        p.wp[r] = wpr;
        p.corr2[r] = c2;
        dotp = cfmad(wpr, v, dotp);
    }
    return dotp;
}

// what the finaliser of C records besides alpha2: d(i), e(i-1), tau(i) and the diagonal of M^H = conj(D) + striu(V^H V)
template <typename T>
__device__ __forceinline__ void combine_record(const StepParams<T>& p, const StepIdx& ix, const StepScalars<T>& sc)
{
    const int m = ix.m;
    p.d[m] = re(ldcg(&p.u[m]));
    p.e[m - 1] = sc.beta;
    p.tau[m] = sc.tau;
    const int lb = p.lb, pos = lb - 1 - ix.jp;                 // conj(1 / tau) (1 for an identity reflector)
    T dinv;
    if (is_zero(sc.tau)) dinv = from_real(1.0, T{});
    else { const double n2 = abs2(sc.tau); dinv = cj(rscale(cj(sc.tau), 1.0 / n2)); }   // conj(1/tau) = conj(conj(tau)/|tau|^2)
    p.R[(long long)p.panel * lb * (lb + 1) + pos + (long long)pos * lb] = dinv;
}

template <typename T, int kCombineTPR>
__global__ void __launch_bounds__(256) combine_kernel(const StepParams<T> p)
{
    GS_TRACE(const unsigned long long tr_entry = trace_time();)
    grid_dep_launch();
    grid_dep_wait();
    const int failed = *reinterpret_cast<const volatile int*>(p.info);      // consumed at the stores (symv_tma_kernel says why)
    const StepIdx ix = step_idx(p);
    const int m = ix.m;
    const int t = threadIdx.x;
    GS_TRACE(struct TraceEnd { unsigned long long* c; __device__ ~TraceEnd() { if (c) atomicMax(c + 2, trace_time()); } }
                 tr_end{((g_sv_trace_m - m == 0 || g_sv_trace_m - m == 1) && t == 0) ? g_c_trace[g_sv_trace_m - m] : nullptr};
             if (tr_end.c) { atomicMin(tr_end.c + 0, tr_entry); atomicMin(tr_end.c + 1, trace_time()); })
    if (blockIdx.x == 0 && t == 0) p.tickets[3] = 0u;      // work counter of symv_tma_kernel
    const StepScalars<T> sc = *sc_of(p, m);
    __shared__ T s_t[2 * 128];           // tW', tV'
    __shared__ T s_row[2 * 128];         // Wt[:, i-1], Vt[:, i-1]
    __shared__ T s_dot[8];
    __shared__ unsigned int s_last;
    combine_load(p, ix, s_t, s_row, 256);
    T dotp = combine_group<T, kCombineTPR>(p, ix, sc, s_t, s_row, int(blockIdx.x), failed);      // (holds the barrier for s_t, s_row)
    // block partial of w'^H v
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) dotp = add(dotp, shfl_xor(dotp, o));
    if ((t & 31) == 0) s_dot[t >> 5] = dotp;
    __syncthreads();
    if (t == 0) {
        T s = s_dot[0];
        for (int w = 1; w < 8; ++w) s = add(s, s_dot[w]);
        p.Pd[blockIdx.x] = s;
        __threadfence();
        s_last = (atomicAdd(&p.tickets[1], 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // the last CTA adds the partials up: every thread a strided share, then the fixed shuffle / warp order
    T part = zero_of(T{});
    for (int b = t; b < int(gridDim.x); b += 256) part = add(part, ldcg(&p.Pd[b]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part = add(part, shfl_xor(part, o));
    if ((t & 31) == 0) s_dot[t >> 5] = part;
    __syncthreads();
    if (t == 0) {
        T dot = s_dot[0];
        for (int w = 1; w < 8; ++w) dot = add(dot, s_dot[w]);
        sc_of(p, m)->alpha2 = rscale(dot, -0.5 * abs2(sc.tau));
        if (failed == 0) combine_record(p, ix, sc);
        p.tickets[1] = 0u;
    }
}

// ---------------------------------------------------------------------------------------------------------
// F: finishes step i and prepares column inext = i - 1.
//   mode 0 (inside a panel):   w(r) = tau w'(r) + alpha2 v(r) -> Wt[jp, r] = conj(w);
//                              u(r) = A(r, i-1) - corr2(r) - v(r) conj(w(i-1)) - w(r)       (r <= i-1; v(i-1) = 1)
//   mode 2 (last of a panel):  only w (the HER2K-shaped launch and a fresh load follow)
//   mode 1 (fresh load):       u(r) = A(r, inext), A up to date; p.i = inext + 1
//   rows >= i of column i of A are zeroed (clean reflector matrix for the back-transformation);
//   partial ||u(0 : inext-1)||^2; the last CTA derives beta, tau, s of the next step (and d(0) at the very end).
// ---------------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) finish_kernel(const StepParams<T> p)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*p.info != 0) return;
    const int i = p.i, inext = i - 1, jp = p.jp, nb = p.nb, mode = p.mode;
    const int t = threadIdx.x;
    if (blockIdx.x == 0 && t == 0) p.tickets[3] = 0u;      // work counter of symv_tma_kernel
    const StepScalars<T> sc = *sc_of(p, i);          // (mode 1: not used)
    __shared__ double s_n[8];
    __shared__ unsigned int s_last;
    T wlast = zero_of(T{}), vlast = zero_of(T{});
    if (mode != 1) {   // w(i-1) and v(i-1) (= 1, or 0 for an identity reflector): every thread forms them itself
        vlast = cj(p.Vt[jp + (long long)(i - 1) * nb]);
        wlast = add(mul(sc.tau, p.wp[i - 1]), mul(sc.alpha2, vlast));
    }
    double nrm = 0.0;
    for (int r = blockIdx.x * 256 + t; r < p.N; r += gridDim.x * 256) {
        if (mode != 1) {
            if (r < i) {
                const T v = cj(p.Vt[jp + (long long)r * nb]);
                const T w = add(mul(sc.tau, p.wp[r]), mul(sc.alpha2, v));
                p.Wt[jp + (long long)r * nb] = cj(w);
                if (mode == 0) {
                    T un = sub(sub(sub(p.A[r + (long long)inext * p.ld], p.corr2[r]), mul(v, cj(wlast))), mul(w, cj(vlast)));
                    if (r == inext) un = real_only(un);
                    p.u[r] = un;
                    if (r < inext - 1) nrm += abs2(un);
                }
            } else {
                p.A[r + (long long)i * p.ld] = zero_of(T{});
            }
        } else {
            if (r <= inext) {
                T un = p.A[r + (long long)inext * p.ld];
                if (r == inext) un = real_only(un);
                p.u[r] = un;
                if (r < inext - 1) nrm += abs2(un);
            }
            if (inext == 0) p.A[r] = zero_of(T{});      // column 0 carries no reflector: the reflector matrix has a zero column there
        }
    }
    if (mode == 2) return;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o);
    if ((t & 31) == 0) s_n[t >> 5] = nrm;
    __syncthreads();
    if (t == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += s_n[w];
        reinterpret_cast<double*>(p.Pd)[blockIdx.x] = s;
        __threadfence();
        s_last = (atomicAdd(&p.tickets[2], 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double xp = 0.0;
    for (int b = t; b < int(gridDim.x); b += 256) xp += __ldcg(&reinterpret_cast<const double*>(p.Pd)[b]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) xp += __shfl_xor_sync(0xffffffffu, xp, o);
    if ((t & 31) == 0) s_n[t >> 5] = xp;
    __syncthreads();
    if (t == 0) {
        double x2 = 0.0;
        for (int w = 0; w < 8; ++w) x2 += s_n[w];
        if (inext >= 1) {
            StepScalars<T> nx;
            nx.alpha2 = zero_of(T{});
            householder_scalars(ldcg(&p.u[inext - 1]), x2, nx);
            nx.pad[0] = nx.pad[1] = 0;
            *sc_of(p, inext) = nx;
        } else {
            p.d[0] = re(ldcg(&p.u[0]));
            p.tau[0] = zero_of(T{});
        }
        p.tickets[2] = 0u;
    }
}

// identity blocks of R (lb x lb, stride lb (lb + 1)): a partial last panel leaves part of its block unset
template <typename T>
__global__ void init_r_kernel(T* R, int lb, int npanels)
{
    const long long total = (long long)npanels * lb * (lb + 1);
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long within = idx % ((long long)lb * (lb + 1));
        const int row = int(within % lb), col = int(within / lb);
        R[idx] = (row == col && col < lb) ? from_real(1.0, T{}) : zero_of(T{});
    }
}

// out[i] = sum_s parts[s * stride + i] (s ascending: a fixed order), i < total -- the split-k partials of the
// back-transformation's Y = Vp^H C~
template <typename T>
__global__ void sum_parts_kernel(const T* __restrict__ parts, long long stride, int nparts, T* __restrict__ out, long long total, const int* info)
{
    grid_dep_launch();
    grid_dep_wait();
    if (*info != 0) return;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        T acc = parts[i];
        for (int s = 1; s < nparts; ++s) acc = add(acc, parts[(long long)s * stride + i]);
        out[i] = acc;
    }
}

// C~(r, c) = Z(r, c) as T (real -> complex widening for the Hermitian path; a plain copy for the real one)
template <typename T>
__global__ void widen_kernel(const double* __restrict__ Z, long long ldz, T* __restrict__ C, long long ldc, int rows, int cols)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= rows) return;
    for (int c = blockIdx.y; c < cols; c += gridDim.y) C[r + (long long)c * ldc] = from_real(Z[r + (long long)c * ldz], T{});
}

// Truncated-basis route: column i of X (= eigenvector D_i of S) is scaled by sigma_i^-1/2 if
// sigma_i >= delta and zeroed otherwise; *kept = number of kept directions.
template <typename T>
__global__ void truncate_scale_kernel(T* __restrict__ X, long long ld, int N, const double* __restrict__ sigma, double delta, int* kept, const int* info)
{
    if (*info != 0) return;
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
        int k = 0;
        for (int c = 0; c < N; ++c) k += (sigma[c] >= delta && sigma[c] > 0.0) ? 1 : 0;
        *kept = k;
    }
    if (r >= N) return;
    for (int c = blockIdx.y; c < N; c += gridDim.y) {
        const double s = sigma[c];
        const double f = (s >= delta && s > 0.0) ? 1.0 / sqrt(s) : 0.0;
        X[r + (long long)c * ld] = rscale(X[r + (long long)c * ld], f);
    }
}

// H_r(i,i) = 2 sqrt2 ||triu(H_r)||_F + 1 for the dropped directions i (whose rows and columns of H_r are zero): a
// value above the spectrum of H_r, so that these decoupled 1 x 1 blocks are never among the lowest eigenvalues.
template <typename T>
__global__ void __launch_bounds__(256) shift_dropped_kernel(T* __restrict__ Hr, long long ld, int N, const double* __restrict__ sigma, double delta,
                                                            double* partial, unsigned int* ticket, const int* info)
{
    if (*info != 0) return;
    __shared__ double s_n[8];
    __shared__ unsigned int s_last;
    double acc = 0.0;
    for (long long c = blockIdx.x; c < N; c += gridDim.x)
        for (int r = threadIdx.x; r <= c; r += 256) acc += abs2(Hr[r + c * ld]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) s_n[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += s_n[w];
        partial[blockIdx.x] = s;
        __threadfence();
        s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double tot = 0.0;
    for (int b = 0; b < int(gridDim.x); ++b) tot += __ldcg(&partial[b]);
    const double shift = 2.0 * sqrt(2.0 * tot) + 1.0;
    for (int c = threadIdx.x; c < N; c += 256)
        if (!(sigma[c] >= delta && sigma[c] > 0.0)) Hr[c + (long long)c * ld] = from_real(shift, T{});
    if (threadIdx.x == 0) *ticket = 0u;
}

}  // namespace evp
}  // namespace gs
