// gs.cu -- the C ABI of include/gs.h: plan management and the four stage drivers.
//
// Every stage is a short host-side schedule of launches of (a) the FP64 tile engine
// (tile_engine.cuh: TMA-staged DMMA tiles with triangular k-ranges) and (b) the 128 x 128 leaf
// kernels (leaf_kernels.cuh).  Nothing here calls cuBLAS/cuSOLVER, and there is no CPU fallback.
//
//   gs_cholesky           recursive blocked POTRF  S = U^T U
//   gs_invert_triangular  block-recursive TRTRI    V = U^-1
//   gs_to_standard        G = T V (T = triu(H,1) + diag(H)/2), H~ = V^T G + G^T V
//   gs_backtransform      C = V C~
#include "../../include/gs.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "engine_host.cuh"
#include "leaf_kernels.cuh"

using namespace gs;

// launch labels for the optional per-launch timing (gs_plan_set_timing)
enum LaunchLabel : int {
    L_POTRF_LEAF = 0, L_POTRF_TRSM, L_POTRF_GEMM, L_POTRF_SYRK, L_ZERO_LOWER,
    L_TRTRI_LEAF, L_TRTRI_W, L_TRTRI_X, L_TOSTD_G, L_TOSTD_SYR2K, L_BACK_TRMM, L_COUNT
};
static const char* const kLabelNames[L_COUNT] = {
    "potrf.leaf", "potrf.trsm_leaf", "potrf.gemm", "potrf.syrk", "zero_lower",
    "trtri.leaf", "trtri.w", "trtri.x", "to_standard.g", "to_standard.syr2k", "backtransform.trmm"};

struct TimedLaunch {
    int label;
    cudaEvent_t e0, e1;
};

struct gs_plan {
    int64_t N = 0;
    int64_t nev = 0;
    gs_dtype_t dtype = GS_REAL64;
    int nblk = 0;                    // ceil(N / 128)
    unsigned char* ws = nullptr;     // caller-owned device workspace
    size_t ws_bytes = 0;
    int64_t launches = 0;
    int timing_mode = 0;
    std::vector<TimedLaunch> timed;
    // look-ahead of the blocked factorisation: a high-priority side stream owned by the plan, forked
    // from and joined back into the caller's stream with events inside every call that uses it
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    int potrf_nb = 8;                // panel width of the look-ahead schedule, in 128-blocks
    char cuda_error[256] = {0};
};

namespace {

constexpr size_t kInfoBytes = 256;

size_t winv_bytes(const gs_plan* p) { return size_t(p->nblk) * LB * LB * sizeof(double); }
size_t big_offset(const gs_plan* p) { return kInfoBytes + ((winv_bytes(p) + 255) / 256) * 256; }
size_t workspace_bytes(const gs_plan* p) { return big_offset(p) + size_t(p->N) * size_t(p->N) * sizeof(double); }

int* info_ptr(const gs_plan* p) { return reinterpret_cast<int*>(p->ws); }
double* winv_ptr(const gs_plan* p) { return reinterpret_cast<double*>(p->ws + kInfoBytes); }
double* big_ptr(const gs_plan* p) { return reinterpret_cast<double*>(p->ws + big_offset(p)); }

gs_status_t cuda_fail(gs_plan* p, cudaError_t e)
{
    if (p != nullptr) std::snprintf(p->cuda_error, sizeof(p->cuda_error), "%s", cudaGetErrorString(e));
    return GS_ERR_CUDA;
}

// Brackets one kernel launch with CUDA events on the launching stream when timing is enabled.
struct LaunchTimer {
    gs_plan* plan;
    cudaStream_t stream;
    bool on;
    TimedLaunch t;
    LaunchTimer(gs_plan* p, int label, cudaStream_t s) : plan(p), stream(s), on(false)
    {
        if (p->timing_mode == 1 || (p->timing_mode == 2 && label == L_TOSTD_SYR2K)) {
            t.label = label;
            if (cudaEventCreate(&t.e0) == cudaSuccess && cudaEventCreate(&t.e1) == cudaSuccess) {
                on = true;
                cudaEventRecord(t.e0, stream);
            }
        }
    }
    ~LaunchTimer()
    {
        if (on) {
            cudaEventRecord(t.e1, stream);
            plan->timed.push_back(t);
        }
    }
};

void clear_timed(gs_plan* p)
{
    for (TimedLaunch& t : p->timed) {
        cudaEventDestroy(t.e0);
        cudaEventDestroy(t.e1);
    }
    p->timed.clear();
}

#define GS_CUDA(plan, call)                                   \
    do {                                                      \
        const cudaError_t e__ = (call);                       \
        if (e__ != cudaSuccess) return cuda_fail((plan), e__); \
    } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// A stage under construction: knows whether every operand can go through TMA.
struct Stage {
    gs_plan* plan;
    cudaStream_t stream;
    bool tma;
};

EngineParams blank_params(const gs_plan* plan)
{
    EngineParams p;
    std::memset(&p, 0, sizeof(p));
    p.batch = 1;
    p.alpha = 1.0;
    p.beta = 0.0;
    p.info = info_ptr(plan);
    return p;
}

// which: 0 = A, 1 = B, 2 = A2, 3 = B2.  mcontig selects the 16 x 16 box of the m-contiguous A operand.
bool set_operand(const Stage& st, EngineParams& p, int which, const MatView& m, bool mcontig)
{
    RawOperand r{m.ptr, m.ld, int(m.rows), int(m.cols)};
    CUtensorMap* map = which == 0 ? &p.mapA : which == 1 ? &p.mapB : which == 2 ? &p.mapA2 : &p.mapB2;
    (which == 0 ? p.rawA : which == 1 ? p.rawB : which == 2 ? p.rawA2 : p.rawB2) = r;
    if (!st.tma) return true;
    return make_tensor_map(map, m, mcontig ? 16 : BN);
}

gs_status_t launch(Stage& st, const EngineParams& p, bool a_nn, int label)
{
    LaunchTimer timer(st.plan, label, st.stream);
    const cudaError_t e = engine_launch(p, a_nn, st.tma, st.stream);
    if (e != cudaSuccess) return cuda_fail(st.plan, e);
    st.plan->launches += 1;
    return GS_OK;
}

#define GS_TRY(expr)                          \
    do {                                      \
        const gs_status_t s__ = (expr);       \
        if (s__ != GS_OK) return s__;         \
    } while (0)

gs_status_t check_ready(const gs_plan* plan)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    if (plan->dtype != GS_REAL64) return GS_ERR_INVALID_ARG;   // complex path: not built yet
    if (plan->ws == nullptr || plan->ws_bytes < workspace_bytes(plan)) return GS_ERR_WORKSPACE;
    return GS_OK;
}

gs_status_t zero_lower(Stage& st, double* X)
{
    const gs_plan* plan = st.plan;
    const int N = int(plan->N);
    if (N <= LB) return GS_OK;
    dim3 grid((N + 255) / 256, N);
    LaunchTimer timer(st.plan, L_ZERO_LOWER, st.stream);
    zero_lower_blocks_kernel<<<grid, 256, 0, st.stream>>>(X, plan->N, N, info_ptr(plan));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(st.plan, e);
    st.plan->launches += 1;
    return GS_OK;
}

// ------------------------------------------------------------------------------------------------
// gs_cholesky: recursive blocked POTRF on 128-blocks.
//   potrf(b0,b1): potrf(b0,mid); S12 = U11^-T S12 (trsm); S22 -= S12^T S12 (syrk, upper tiles); potrf(mid,b1)
//   trsm(r0,r1 | c0,c1): recursive on the triangular block; leaves multiply by the inverted
//   diagonal block W = U_kk^-1 produced by the leaf factorisation.
// ------------------------------------------------------------------------------------------------
struct Potrf {
    Stage st;
    double* S;
    MatView vS;
    MatView vW;   // one Winv slot viewed as 128 x (128*nblk) matrix, ld 128

    gs_status_t leaf(int b)
    {
        gs_plan* plan = st.plan;
        LaunchTimer timer(plan, L_POTRF_LEAF, st.stream);
        potrf_leaf_kernel<<<1, kLeafThreads, kLeafSmemBytes, st.stream>>>(S, plan->N, int(plan->N), b * LB,
                                                                          winv_ptr(plan) + size_t(b) * LB * LB, info_ptr(plan));
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(plan, e);
        plan->launches += 1;
        return GS_OK;
    }

    // X = W_r0^T * S[r0, c0:c1], in place (each CTA reads exactly the tile it overwrites)
    gs_status_t trsm_leaf(int r0, int c0, int c1)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vW, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = S; p.ldc = vS.ld;
        p.tiles_m = 1; p.tiles_n = c1 - c0; p.order = ORDER_COL;
        p.c_row0 = r0 * LB; p.c_col0 = c0 * LB; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = LB / BK; p.kmax = LB / BK;
        p.a.k0 = 0; p.a.x0 = r0 * LB;          // W slot r0 = columns [128 r0, 128 r0 + 128) of vW
        p.b.k0 = r0 * LB; p.b.x0 = c0 * LB;
        return launch(st, p, false, L_POTRF_TRSM);
    }

    // S[h:r1, c0:c1] -= U[r0:h, h:r1]^T * S[r0:h, c0:c1]
    gs_status_t gemm_update(int r0, int h, int r1, int c0, int c1)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vS, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = S; p.ldc = vS.ld;
        p.tiles_m = r1 - h; p.tiles_n = c1 - c0; p.order = ORDER_COL;
        p.c_row0 = h * LB; p.c_col0 = c0 * LB; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (h - r0) * (LB / BK); p.kmax = p.khi_c;
        p.a.k0 = r0 * LB; p.a.x0 = h * LB;
        p.b.k0 = r0 * LB; p.b.x0 = c0 * LB;
        p.alpha = -1.0; p.beta = 1.0;
        return launch(st, p, false, L_POTRF_GEMM);
    }

    gs_status_t trsm(int r0, int r1, int c0, int c1)
    {
        if (c1 <= c0) return GS_OK;
        if (r1 - r0 == 1) return trsm_leaf(r0, c0, c1);
        const int h = r0 + (r1 - r0 + 1) / 2;
        GS_TRY(trsm(r0, h, c0, c1));
        GS_TRY(gemm_update(r0, h, r1, c0, c1));
        return trsm(h, r1, c0, c1);
    }

    // S[c0:c1, c0:c1] -= S[k0:k1, c0:c1]^T S[k0:k1, c0:c1], upper tiles only
    gs_status_t syrk(int k0, int k1, int c0, int c1)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vS, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = S; p.ldc = vS.ld;
        p.tiles_m = c1 - c0; p.tiles_n = c1 - c0; p.order = ORDER_TRI_ROW_DESC;
        p.c_row0 = c0 * LB; p.c_col0 = c0 * LB; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (k1 - k0) * (LB / BK); p.kmax = p.khi_c;
        p.a.k0 = k0 * LB; p.a.x0 = c0 * LB;
        p.b.k0 = k0 * LB; p.b.x0 = c0 * LB;
        p.alpha = -1.0; p.beta = 1.0;
        p.flags = F_STORE_UPPER;
        return launch(st, p, false, L_POTRF_SYRK);
    }

    // Block rows [r0, r1) of the trailing update (the next panel's rows), upper trapezoid:
    // S[r0:r1, r0:n] -= S[k0:k1, r0:r1]^T S[k0:k1, r0:n]
    gs_status_t update_rows(int k0, int k1, int r0, int r1, int n)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vS, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = S; p.ldc = vS.ld;
        p.tiles_m = r1 - r0; p.tiles_n = n - r0; p.order = ORDER_TRAPEZOID;
        p.c_row0 = r0 * LB; p.c_col0 = r0 * LB; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (k1 - k0) * (LB / BK); p.kmax = p.khi_c;
        p.a.k0 = k0 * LB; p.a.x0 = r0 * LB;
        p.b.k0 = k0 * LB; p.b.x0 = r0 * LB;
        p.alpha = -1.0; p.beta = 1.0;
        p.flags = F_STORE_UPPER;
        return launch(st, p, false, L_POTRF_SYRK);
    }

    // recursive factorisation of the diagonal block [b0, b1) (touches nothing outside it)
    gs_status_t potrf(int b0, int b1)
    {
        if (b1 - b0 == 1) return leaf(b0);
        const int mid = b0 + (b1 - b0 + 1) / 2;
        GS_TRY(potrf(b0, mid));
        GS_TRY(trsm(b0, mid, mid, b1));
        GS_TRY(syrk(b0, mid, mid, b1));
        return potrf(mid, b1);
    }

    // panel = block rows [b0, b1): factor the diagonal block, then solve the row panel to its right
    gs_status_t panel(int b0, int b1, int n)
    {
        GS_TRY(potrf(b0, b1));
        return trsm(b0, b1, b1, n);
    }

    // Right-looking over panels of NB blocks with one panel of look-ahead: while the caller's
    // stream applies panel p to the trailing matrix beyond panel p+1, the plan's high-priority
    // side stream applies it to the rows of panel p+1 and factors that panel.
    gs_status_t factor(int n, int NB, cudaStream_t main_stream, cudaStream_t side, cudaEvent_t ev_fork, cudaEvent_t ev_join)
    {
        gs_plan* plan = st.plan;
        st.stream = main_stream;
        GS_TRY(panel(0, NB < n ? NB : n, n));
        for (int b0 = 0; b0 + NB < n; b0 += NB) {
            const int b1 = b0 + NB;
            const int b2 = b1 + NB < n ? b1 + NB : n;
            GS_CUDA(plan, cudaEventRecord(ev_fork, main_stream));
            GS_CUDA(plan, cudaStreamWaitEvent(side, ev_fork, 0));
            st.stream = side;
            gs_status_t rc = update_rows(b0, b1, b1, b2, n);
            if (rc == GS_OK) rc = panel(b1, b2, n);
            st.stream = main_stream;
            if (rc == GS_OK && b2 < n) rc = syrk(b0, b1, b2, n);
            // always join the side stream back, also on failure
            const cudaError_t e1 = cudaEventRecord(ev_join, side);
            const cudaError_t e2 = cudaStreamWaitEvent(main_stream, ev_join, 0);
            GS_TRY(rc);
            GS_CUDA(plan, e1);
            GS_CUDA(plan, e2);
        }
        return GS_OK;
    }
};

gs_status_t ensure_side_stream(gs_plan* plan)
{
    if (plan->side != nullptr) return GS_OK;
    int lo = 0, hi = 0;
    GS_CUDA(plan, cudaDeviceGetStreamPriorityRange(&lo, &hi));
    GS_CUDA(plan, cudaStreamCreateWithPriority(&plan->side, cudaStreamNonBlocking, hi));
    GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_fork, cudaEventDisableTiming));
    GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_join, cudaEventDisableTiming));
    return GS_OK;
}

gs_status_t configure_leaf(gs_plan* plan)
{
    static bool done = false;
    if (done) return GS_OK;
    GS_CUDA(plan, cudaFuncSetAttribute(potrf_leaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeafSmemBytes));
    GS_CUDA(plan, cudaFuncSetAttribute(trtri_leaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeafSmemBytes));
    done = true;
    return GS_OK;
}

}  // namespace

extern "C" {

gs_status_t gs_plan_create(gs_plan_t** plan, int64_t N, gs_dtype_t dtype, int64_t nev)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    *plan = nullptr;
    if (N < 1 || N > (int64_t(1) << 20) || nev < 0 || nev > N) return GS_ERR_INVALID_ARG;
    if (dtype != GS_REAL64 && dtype != GS_COMPLEX128) return GS_ERR_INVALID_ARG;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return GS_ERR_UNSUPPORTED_DEVICE; }
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return GS_ERR_UNSUPPORTED_DEVICE; }
    if (major != 10) return GS_ERR_UNSUPPORTED_DEVICE;
    gs_plan* p = new (std::nothrow) gs_plan();
    if (p == nullptr) return GS_ERR_INVALID_ARG;
    p->N = N;
    p->nev = nev;
    p->dtype = dtype;
    p->nblk = int((N + LB - 1) / LB);
    if (const char* e = std::getenv("GS_POTRF_NB")) {
        const int v = std::atoi(e);
        if (v >= 1 && v <= 64) p->potrf_nb = v;
    }
    *plan = p;
    return GS_OK;
}

gs_status_t gs_plan_destroy(gs_plan_t* plan)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    clear_timed(plan);
    if (plan->ev_fork != nullptr) cudaEventDestroy(plan->ev_fork);
    if (plan->ev_join != nullptr) cudaEventDestroy(plan->ev_join);
    if (plan->side != nullptr) cudaStreamDestroy(plan->side);
    delete plan;
    return GS_OK;
}

gs_status_t gs_plan_workspace_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    *bytes = workspace_bytes(plan);
    return GS_OK;
}

gs_status_t gs_plan_set_workspace(gs_plan_t* plan, void* dev_workspace, size_t bytes)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    if (dev_workspace == nullptr || bytes < workspace_bytes(plan) || (reinterpret_cast<uintptr_t>(dev_workspace) & 255u) != 0)
        return GS_ERR_WORKSPACE;
    plan->ws = static_cast<unsigned char*>(dev_workspace);
    plan->ws_bytes = bytes;
    // the info flag must start cleared even if gs_cholesky is never called on this plan
    const cudaError_t e = cudaMemset(plan->ws, 0, kInfoBytes);
    if (e != cudaSuccess) return cuda_fail(plan, e);
    return GS_OK;
}

gs_status_t gs_cholesky(gs_plan_t* plan, void* S_inout, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (S_inout == nullptr || !aligned16(S_inout)) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    GS_CUDA(plan, cudaMemsetAsync(info_ptr(plan), 0, sizeof(int), stream));
    double* S = static_cast<double*>(S_inout);
    Potrf f;
    f.st = Stage{plan, stream, plan->N % 2 == 0};
    f.S = S;
    f.vS = MatView{S, plan->N, plan->N, plan->N};
    f.vW = MatView{winv_ptr(plan), LB, (long long)LB * plan->nblk, LB};
    if (plan->nblk > plan->potrf_nb) GS_TRY(ensure_side_stream(plan));
    GS_TRY(zero_lower(f.st, S));   // off-diagonal lower blocks: never touched by the factorisation
    return f.factor(plan->nblk, plan->potrf_nb, stream, plan->side, plan->ev_fork, plan->ev_join);
}

// Block-recursive inversion by doubling: with U = [A B; 0 D],  U^-1 = [A^-1, -A^-1 B D^-1; 0, D^-1].
// Level s (in 128-blocks): all pairs (A = blocks [2is, 2is+s), D = the next s blocks) at once:
//   W = B * D^-1   (k <= J: D^-1 upper)      -> workspace, at the position of the target block
//   X = -A^-1 * W  (k >= I: A^-1 upper)      -> V
gs_status_t gs_invert_triangular(gs_plan_t* plan, const void* U_, void* Uinv_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (U_ == nullptr || Uinv_ == nullptr || U_ == Uinv_ || !aligned16(U_) || !aligned16(Uinv_)) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    const double* U = static_cast<const double*>(U_);
    double* V = static_cast<double*>(Uinv_);
    double* W = big_ptr(plan);
    const int N = int(plan->N), nblk = plan->nblk;
    Stage st{plan, stream, plan->N % 2 == 0};

    {
        LaunchTimer timer(plan, L_TRTRI_LEAF, stream);
        trtri_leaf_kernel<<<nblk, kLeafThreads, kLeafSmemBytes, stream>>>(U, V, plan->N, N, info_ptr(plan));
    }
    GS_CUDA(plan, cudaGetLastError());
    plan->launches += 1;
    GS_TRY(zero_lower(st, V));

    const MatView vU{U, N, N, N}, vV{V, N, N, N}, vWs{W, N, N, N};
    for (int s = 1; s < nblk; s *= 2) {
        const int npairs = (nblk - s + 2 * s - 1) / (2 * s);
        const int stride = 2 * s * LB;   // elements between consecutive pairs
        {   // W = B * Dinv
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vU, true) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
            p.C = W; p.ldc = N;
            p.tiles_m = s; p.tiles_n = s; p.batch = npairs; p.order = ORDER_COL_REV;
            p.c_row0 = 0; p.c_col0 = s * LB; p.c_brow = stride; p.c_bcol = stride; p.c_rows = N; p.c_cols = N;
            p.khi_c = LB / BK; p.khi_j = LB / BK; p.kmax = s * (LB / BK);
            p.a.x0 = 0; p.a.bx = stride; p.a.k0 = s * LB; p.a.bk = stride;
            p.b.k0 = s * LB; p.b.bk = stride; p.b.x0 = s * LB; p.b.bx = stride;
            GS_TRY(launch(st, p, true, L_TRTRI_W));
        }
        {   // X = -Ainv * W
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vV, true) || !set_operand(st, p, 1, vWs, false)) return GS_ERR_CUDA;
            p.C = V; p.ldc = N;
            p.tiles_m = s; p.tiles_n = s; p.batch = npairs; p.order = ORDER_ROW;
            p.c_row0 = 0; p.c_col0 = s * LB; p.c_brow = stride; p.c_bcol = stride; p.c_rows = N; p.c_cols = N;
            p.klo_i = LB / BK; p.khi_c = s * (LB / BK); p.kmax = s * (LB / BK);
            p.a.x0 = 0; p.a.bx = stride; p.a.k0 = 0; p.a.bk = stride;
            p.b.k0 = 0; p.b.bk = stride; p.b.x0 = s * LB; p.b.bx = stride;
            p.alpha = -1.0;
            GS_TRY(launch(st, p, true, L_TRTRI_X));
        }
    }
    return GS_OK;
}

// H~ = V^T H V with H = T + T^T, T = triu(H,1) + diag(H)/2:
//   G  = T V                (upper x upper = upper; N^3/3 flop)   -> workspace
//   H~ = V^T G + G^T V      (upper triangle only; SYR2K-shaped, operands triangular; 2N^3/3 flop)
// N^3 flop in total instead of the 4N^3/3 of forming W = H V in full.
gs_status_t gs_to_standard(gs_plan_t* plan, const void* H_, const void* Uinv_, void* Htilde_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (H_ == nullptr || Uinv_ == nullptr || Htilde_ == nullptr || Htilde_ == H_ || Htilde_ == Uinv_ ||
        !aligned16(H_) || !aligned16(Uinv_) || !aligned16(Htilde_))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int N = int(plan->N), nblk = plan->nblk;
    Stage st{plan, stream, plan->N % 2 == 0};
    double* G = big_ptr(plan);
    const MatView vH{static_cast<const double*>(H_), N, N, N}, vV{static_cast<const double*>(Uinv_), N, N, N}, vG{G, N, N, N};
    const int kt = LB / BK;
    {
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, vH, true) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
        p.C = G; p.ldc = N;
        p.tiles_m = nblk; p.tiles_n = nblk; p.order = ORDER_TRI_DIAG_DESC;
        p.c_rows = N; p.c_cols = N;
        p.klo_i = kt; p.khi_c = kt; p.khi_j = kt; p.kmax = (N + BK - 1) / BK;
        p.flags = F_MASK_A | F_HALF_DIAG_A | F_MASK_B;
        GS_TRY(launch(st, p, true, L_TOSTD_G));
    }
    {
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, vV, false) || !set_operand(st, p, 1, vG, false) || !set_operand(st, p, 2, vG, false) ||
            !set_operand(st, p, 3, vV, false))
            return GS_ERR_CUDA;
        p.C = static_cast<double*>(Htilde_); p.ldc = N;
        p.tiles_m = nblk; p.tiles_n = nblk; p.order = ORDER_TRI_ROW_DESC;
        p.c_rows = N; p.c_cols = N;
        p.khi_c = kt; p.khi_i = kt; p.kmax = (N + BK - 1) / BK;
        p.flags = F_DUAL | F_MASK_A | F_MASK_B2 | F_STORE_UPPER;
        GS_TRY(launch(st, p, false, L_TOSTD_SYR2K));
    }
    return GS_OK;
}

gs_status_t gs_backtransform(gs_plan_t* plan, const void* Uinv_, const void* Ctilde_, void* C_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (plan->nev == 0) return GS_OK;
    if (Uinv_ == nullptr || Ctilde_ == nullptr || C_ == nullptr || C_ == Ctilde_ || C_ == Uinv_ || !aligned16(Uinv_) ||
        !aligned16(Ctilde_) || !aligned16(C_))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int N = int(plan->N), nev = int(plan->nev);
    Stage st{plan, stream, plan->N % 2 == 0};
    const MatView vV{static_cast<const double*>(Uinv_), N, N, N}, vC{static_cast<const double*>(Ctilde_), N, nev, N};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vV, true) || !set_operand(st, p, 1, vC, false)) return GS_ERR_CUDA;
    p.C = static_cast<double*>(C_); p.ldc = N;
    p.tiles_m = plan->nblk; p.tiles_n = (nev + BN - 1) / BN; p.order = ORDER_ROW;
    p.c_rows = N; p.c_cols = nev;
    p.klo_i = LB / BK; p.khi_c = (N + BK - 1) / BK; p.kmax = p.khi_c;
    p.flags = F_MASK_A;
    return launch(st, p, true, L_BACK_TRMM);
}

gs_status_t gs_last_info(gs_plan_t* plan, void* cuda_stream, int64_t* info)
{
    if (plan == nullptr || info == nullptr) return GS_ERR_INVALID_ARG;
    *info = 0;
    if (plan->ws == nullptr) return GS_ERR_WORKSPACE;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int h = 0;
    GS_CUDA(plan, cudaMemcpyAsync(&h, info_ptr(plan), sizeof(int), cudaMemcpyDeviceToHost, stream));
    GS_CUDA(plan, cudaStreamSynchronize(stream));
    if (h > 0) { *info = h; return GS_ERR_NOT_POSDEF; }
    if (h < 0) { *info = -int64_t(h); return GS_ERR_SINGULAR; }
    return GS_OK;
}

gs_status_t gs_reduce_host_scratch_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    const size_t mat = ((size_t(plan->N) * size_t(plan->N) * sizeof(double) + 255) / 256) * 256;
    *bytes = 4 * mat;   // S->U, H (later C~ and C), Uinv, Htilde
    return GS_OK;
}

gs_status_t gs_reduce_host(gs_plan_t* plan, const void* host_H, const void* host_S, void* host_U, void* host_Uinv,
                           void* host_Htilde, void* dev_scratch, size_t scratch_bytes, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    size_t need = 0;
    gs_reduce_host_scratch_bytes(plan, &need);
    if (host_H == nullptr || host_S == nullptr || host_Htilde == nullptr || dev_scratch == nullptr || scratch_bytes < need ||
        (reinterpret_cast<uintptr_t>(dev_scratch) & 255u) != 0)
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t bytes = size_t(plan->N) * size_t(plan->N) * sizeof(double);
    const size_t mat = need / 4;
    unsigned char* base = static_cast<unsigned char*>(dev_scratch);
    void *dS = base, *dH = base + mat, *dV = base + 2 * mat, *dHt = base + 3 * mat;
    GS_CUDA(plan, cudaMemcpyAsync(dS, host_S, bytes, cudaMemcpyHostToDevice, stream));
    GS_CUDA(plan, cudaMemcpyAsync(dH, host_H, bytes, cudaMemcpyHostToDevice, stream));
    GS_CUDA(plan, cudaMemsetAsync(dHt, 0, bytes, stream));
    GS_TRY(gs_cholesky(plan, dS, stream));
    GS_TRY(gs_invert_triangular(plan, dS, dV, stream));
    GS_TRY(gs_to_standard(plan, dH, dV, dHt, stream));
    if (host_U) GS_CUDA(plan, cudaMemcpyAsync(host_U, dS, bytes, cudaMemcpyDeviceToHost, stream));
    if (host_Uinv) GS_CUDA(plan, cudaMemcpyAsync(host_Uinv, dV, bytes, cudaMemcpyDeviceToHost, stream));
    GS_CUDA(plan, cudaMemcpyAsync(host_Htilde, dHt, bytes, cudaMemcpyDeviceToHost, stream));
    int64_t info = 0;
    return gs_last_info(plan, stream, &info);
}

gs_status_t gs_backtransform_host(gs_plan_t* plan, const void* host_Ctilde, void* host_C, void* dev_scratch,
                                  size_t scratch_bytes, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    size_t need = 0;
    gs_reduce_host_scratch_bytes(plan, &need);
    if (dev_scratch == nullptr || scratch_bytes < need || (reinterpret_cast<uintptr_t>(dev_scratch) & 255u) != 0)
        return GS_ERR_INVALID_ARG;
    if (plan->nev == 0) return GS_OK;
    if (host_Ctilde == nullptr || host_C == nullptr) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t mat = need / 4;
    const size_t cbytes = size_t(plan->N) * size_t(plan->nev) * sizeof(double);
    unsigned char* base = static_cast<unsigned char*>(dev_scratch);
    // U^-1 was left at base + 2*mat by gs_reduce_host; C~ and C reuse the S and H slots
    void *dV = base + 2 * mat, *dCt = base, *dC = base + mat;
    GS_CUDA(plan, cudaMemcpyAsync(dCt, host_Ctilde, cbytes, cudaMemcpyHostToDevice, stream));
    GS_TRY(gs_backtransform(plan, dV, dCt, dC, stream));
    GS_CUDA(plan, cudaMemcpyAsync(host_C, dC, cbytes, cudaMemcpyDeviceToHost, stream));
    int64_t info = 0;
    return gs_last_info(plan, stream, &info);
}

gs_status_t gs_plan_set_timing(gs_plan_t* plan, int mode)
{
    if (plan == nullptr || mode < 0 || mode > 2) return GS_ERR_INVALID_ARG;
    clear_timed(plan);
    plan->timing_mode = mode;
    return GS_OK;
}

gs_status_t gs_plan_launch_times(gs_plan_t* plan, gs_launch_time_t* out, int cap, int* count)
{
    if (plan == nullptr || count == nullptr || (out == nullptr && cap > 0)) return GS_ERR_INVALID_ARG;
    double ms[L_COUNT] = {0};
    int64_t n[L_COUNT] = {0};
    for (const TimedLaunch& t : plan->timed) {
        float f = 0.f;
        const cudaError_t e = cudaEventElapsedTime(&f, t.e0, t.e1);
        if (e != cudaSuccess) return cuda_fail(plan, e);
        ms[t.label] += f;
        n[t.label] += 1;
    }
    clear_timed(plan);
    int k = 0;
    for (int l = 0; l < L_COUNT; ++l) {
        if (n[l] == 0) continue;
        if (k < cap) {
            std::snprintf(out[k].label, sizeof(out[k].label), "%s", kLabelNames[l]);
            out[k].launches = n[l];
            out[k].ms = ms[l];
        }
        ++k;
    }
    *count = k;
    return GS_OK;
}

gs_status_t gs_plan_launch_count(const gs_plan_t* plan, int64_t* launches)
{
    if (plan == nullptr || launches == nullptr) return GS_ERR_INVALID_ARG;
    *launches = plan->launches;
    return GS_OK;
}

const char* gs_status_string(gs_status_t status)
{
    switch (status) {
        case GS_OK: return "GS_OK";
        case GS_ERR_INVALID_ARG: return "GS_ERR_INVALID_ARG";
        case GS_ERR_NOT_POSDEF: return "GS_ERR_NOT_POSDEF";
        case GS_ERR_SINGULAR: return "GS_ERR_SINGULAR";
        case GS_ERR_CUDA: return "GS_ERR_CUDA";
        case GS_ERR_WORKSPACE: return "GS_ERR_WORKSPACE";
        case GS_ERR_UNSUPPORTED_DEVICE: return "GS_ERR_UNSUPPORTED_DEVICE";
    }
    return "GS_ERR_UNKNOWN";
}

const char* gs_plan_last_cuda_error(const gs_plan_t* plan) { return plan != nullptr ? plan->cuda_error : ""; }

}  // extern "C"
