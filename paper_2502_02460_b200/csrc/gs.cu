// gs.cu -- the C ABI of include/gs.h: plan management, the four stage drivers, the density matrix and
// the host-buffer entry points.
//
// Every stage is a short host-side schedule of launches of (a) the FP64 tile engines -- TMA-staged DMMA
// tiles with triangular k-ranges: tile64_engine.cuh (real, 64 x 64 CTA tiles, the default),
// tile_engine.cuh (real, 128 x 128: in-place one-tile solves and odd N), ctile_half_engine.cuh /
// ctile_engine.cuh (complex128) -- and (b) the diagonal-block kernels (leaf_kernels.cuh, cleaf_kernels.cuh).
// Nothing here calls cuBLAS/cuSOLVER, and there is no CPU fallback.
//
//   gs_cholesky           blocked POTRF with look-ahead on a side stream  S = U^H U
//   gs_invert_triangular  block-recursive TRTRI by doubling               V = U^-1
//   gs_to_standard        G = T V (T = triu(H,1) + diag(H)/2), H~ = V^H G + G^H V
//   gs_backtransform      C = V C~
//   gs_density_matrix     P = sum_l f_l c*_l c_l (weighted SYRK / HERK)
#include "../../include/gs.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>   // header-only NVTX v3: no-ops unless a profiler injects itself

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <functional>
#include <new>
#include <vector>

#include "engine_host.cuh"
#include "leaf_kernels.cuh"
#include "leaf32_kernel.cuh"
#include "cleaf_kernels.cuh"

using namespace gs;

// launch labels for the optional per-launch timing (gs_plan_set_timing)
enum LaunchLabel : int {
    L_POTRF_LEAF = 0, L_POTRF_TRSM, L_POTRF_GEMM, L_POTRF_SYRK, L_ZERO_LOWER,
    L_TRTRI_LEAF, L_TRTRI_W, L_TRTRI_X, L_TOSTD_G, L_TOSTD_SYR2K, L_BACK_TRMM, L_DENS_T, L_DENS_SYRK, L_PUSH_BAND,
    L_EVP_SYMV, L_EVP_STEP, L_EVP_HER2K, L_EVP_DC, L_EVP_DC_GEMM, L_EVP_BACK, L_COUNT
};
static const char* const kLabelNames[L_COUNT] = {
    "potrf.leaf", "potrf.trsm_leaf", "potrf.gemm", "potrf.syrk", "zero_lower",
    "trtri.leaf", "trtri.w", "trtri.x", "to_standard.g", "to_standard.syr2k", "backtransform.trmm",
    "density.transpose", "density.syrk", "shard.push_band",
    "evp.tridiag.symv", "evp.tridiag.step", "evp.tridiag.her2k", "evp.solve.dc", "evp.solve.gemm", "evp.back"};

struct TimedLaunch {
    int label;
    int side;           // 1 = launched on the plan's side stream
    cudaEvent_t e0, e1;
};

struct gs_plan {
    int64_t N = 0;
    int64_t nev = 0;
    gs_dtype_t dtype = GS_REAL64;
    bool z = false;                  // GS_COMPLEX128
    int lb = LB;                     // leaf / tile block order in elements: 128 (real) or 64 (complex)
    int bk = BK;                     // k-slab of one pipeline stage in elements: 16 (real) or 8 (complex)
    size_t es = sizeof(double);      // bytes per element
    int nblk = 0;                    // ceil(N / lb)
    unsigned char* ws = nullptr;     // caller-owned device workspace
    size_t ws_bytes = 0;
    unsigned char* evp_ws = nullptr; // caller-owned device workspace of the standard eigensolver (gs_evp_set_workspace)
    size_t evp_ws_bytes = 0;
    int64_t launches = 0;
    int timing_mode = 0;
    std::vector<TimedLaunch> timed;
    // look-ahead of the blocked factorisation: a high-priority side stream owned by the plan, forked
    // from and joined back into the caller's stream with events inside every call that uses it
    cudaStream_t side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_rows = nullptr, ev_join = nullptr;
    cudaStream_t copy = nullptr;     // host-buffer entry points: H2D copies beside compute
    cudaStream_t copy_out = nullptr; // host-buffer entry points: D2H copies beside compute
    cudaEvent_t ev_copy = nullptr;
    // host path (gs_reduce_host): the rows of S below the first two panels arrive in slabs while step 1 is
    // already running; slab q = block rows [gates[q].first, gates[q+1].first or nblk) is on the device once
    // gates[q].second fires.  Empty: everything is there.
    std::vector<std::pair<int, cudaEvent_t>> gates;
    std::vector<cudaEvent_t> ev_pool;   // per-chunk events of the host-buffer entry points
    int potrf_nb = 8;                // panel width of the look-ahead schedule, in 128-blocks
    int potrf_nb_tail = 4;           // panel width once at most potrf_tail blocks remain
    int potrf_tail = 64;
    int potrf_nb_end = 1;            // panel width once at most potrf_end blocks remain
    int potrf_end = 32;
    int ctile_half = 1;              // complex: two 64 x 32 CTAs per logical tile (3 CTAs/SM) instead of one 64 x 64
    int tile64_mode = 2, tile64_below = 74;   // 64 x 64-tile engine for launches below this many logical tiles
    std::vector<void*> push[4];      // fused exchange: push targets per gs_push_kind_t (gs_plan_set_push_targets)
    int leaf_blocked = 0;            // real POTRF diagonal blocks: blocked sweep (potrf_leaf4_kernel) instead of the rank-1 sweep
    int leaf_mode = 2;               // 2: 32 x 32 sub-blocks, warp-level sweeps + in-CTA DMMA (leaf32_kernel.cuh, default); 1: 4-row panels; 0: rank-1 sweep over 256 threads
    int shard_panel = 8;             // column-range inversion: panel of the back substitution in blocks (power of two)
    int super_tile = 12;             // super-tile edge of triangular launches (about one wave of CTAs per super-tile)
    int super_syr2k = 4;             // the same for the SYR2K-shaped launch of gs_to_standard (four operand panels per tile)
    int potrf_flat = 1;              // diagonal panel blocks factored right-looking block by block (default) instead of recursively
    char cuda_error[256] = {0};
};

namespace {

constexpr size_t kInfoBytes = 256;
constexpr int KPB = 8;   // pipeline k-steps per block: 128 / 16 (real) = 64 / 8 (complex)
static_assert(LB / BK == KPB && CLB / CBK == KPB && CT == CLB, "block / k-slab ratio");

// Workspace layout: [info flag | 2 panel-inverse buffers Wp (ldw x ldw each) | one N x N matrix]
int wp_ld(const gs_plan* p) { return p->lb * (p->nblk < p->potrf_nb ? p->nblk : p->potrf_nb); }
size_t wp_bytes(const gs_plan* p) { return size_t(wp_ld(p)) * size_t(wp_ld(p)) * p->es; }
size_t big_offset(const gs_plan* p) { return kInfoBytes + ((2 * wp_bytes(p) + 255) / 256) * 256; }
// (+ 2 columns: gs_density_matrix pads the pitch of the transposed eigenvector block to an even value)
size_t workspace_bytes(const gs_plan* p) { return big_offset(p) + size_t(p->N) * size_t(p->N + 2) * p->es; }

int* info_ptr(const gs_plan* p) { return reinterpret_cast<int*>(p->ws); }
void* wp_ptr(const gs_plan* p, int which) { return p->ws + kInfoBytes + size_t(which & 1) * wp_bytes(p); }
void* big_ptr(const gs_plan* p) { return p->ws + big_offset(p); }

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
    bool nvtx;
    // GS_NVTX=1: every launch sits in an NVTX range named after its label ("to_standard.syr2k", ...), so that
    // `ncu --nvtx --print-nvtx-rename kernel` lists launches by label (profiles/r02_perkernel.md)
    static bool nvtx_on()
    {
        static const bool v = std::getenv("GS_NVTX") != nullptr && std::atoi(std::getenv("GS_NVTX")) != 0;
        return v;
    }
    LaunchTimer(gs_plan* p, int label, cudaStream_t s) : plan(p), stream(s), on(false), nvtx(nvtx_on())
    {
        if (nvtx) nvtxRangePushA(kLabelNames[label]);
        if (p->timing_mode == 1 || (p->timing_mode == 2 && label == L_TOSTD_SYR2K)) {
            t.label = label;
            t.side = (p->side != nullptr && s == p->side) ? 1 : 0;
            if (cudaEventCreate(&t.e0) == cudaSuccess && cudaEventCreate(&t.e1) == cudaSuccess) {
                on = true;
                cudaEventRecord(t.e0, stream);
            }
        }
    }
    ~LaunchTimer()
    {
        if (nvtx) nvtxRangePop();
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

// byte ranges [a, a + na) and [b, b + nb) intersect (the aliasing rule of include/gs.h is about ranges:
// an output that starts inside an input is as wrong as one that equals it)
bool overlaps(const void* a, size_t na, const void* b, size_t nb)
{
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
    return a0 < b0 + nb && b0 < a0 + na;
}
size_t mat_bytes(const gs_plan* p) { return size_t(p->N) * size_t(p->N) * p->es; }
size_t vec_bytes(const gs_plan* p) { return size_t(p->N) * size_t(p->nev) * p->es; }

// Device-side ordering of the fused exchange: stream memory operations (see include/gs.h).
typedef CUresult (*StreamValue32Fn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
StreamValue32Fn stream_value_fn(const char* name)
{
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) return nullptr;
    return reinterpret_cast<StreamValue32Fn>(fn);
}
gs_status_t stream_values(gs_plan* plan, bool wait, int count, void* const* flags, uint32_t value, void* cuda_stream)
{
    if (plan == nullptr || count < 0 || count > 64 || (count > 0 && flags == nullptr)) return GS_ERR_INVALID_ARG;
    for (int d = 0; d < count; ++d)
        if (flags[d] == nullptr || (reinterpret_cast<uintptr_t>(flags[d]) & 3u) != 0) return GS_ERR_INVALID_ARG;
    static StreamValue32Fn wr = stream_value_fn("cuStreamWriteValue32"), wt = stream_value_fn("cuStreamWaitValue32");
    StreamValue32Fn fn = wait ? wt : wr;
    if (fn == nullptr) return GS_ERR_CUDA;
    for (int d = 0; d < count; ++d) {
        const CUresult r = fn(static_cast<CUstream>(cuda_stream), reinterpret_cast<CUdeviceptr>(flags[d]), value,
                              wait ? unsigned(CU_STREAM_WAIT_VALUE_GEQ) : unsigned(CU_STREAM_WRITE_VALUE_DEFAULT));
        if (r != CUDA_SUCCESS) {
            std::snprintf(plan->cuda_error, sizeof(plan->cuda_error), "%s failed (CUresult %d)", wait ? "cuStreamWaitValue32" : "cuStreamWriteValue32", int(r));
            return GS_ERR_CUDA;
        }
    }
    return GS_OK;
}

// A stage under construction: knows whether every operand can go through TMA.
struct Stage {
    gs_plan* plan;
    cudaStream_t stream;
    bool tma;
    bool z;       // complex128
    int lb, bk;   // block order and k-slab in elements (plan->lb, plan->bk)
    // operands of the launch under construction (tensor maps are encoded in launch(), once the tile
    // size of the kernel is known)
    MatView opv[4];
    bool opm[4];
    bool opset[4];
};

Stage make_stage(gs_plan* plan, cudaStream_t stream)
{
    // a real matrix with odd N has a row pitch that is not a multiple of 16 bytes: no tensor map
    Stage st{};
    st.plan = plan; st.stream = stream; st.tma = plan->z || plan->N % 2 == 0; st.z = plan->z; st.lb = plan->lb; st.bk = plan->bk;
    return st;
}

EngineParams blank_params(const gs_plan* plan)
{
    EngineParams p;
    std::memset(&p, 0, sizeof(p));
    p.batch = 1;
    p.alpha = 1.0;
    p.beta = 0.0;
    p.info = info_ptr(plan);
    p.super = plan->super_tile;
    return p;
}

// fused exchange: the launch also stores its tiles into the plan's push targets of `kind` (include/gs.h)
void set_peers(const gs_plan* plan, EngineParams& p, int kind, size_t byte_offset = 0)
{
    const std::vector<void*>& t = plan->push[kind];
    p.npeer = int(t.size());
    p.peer_col0 = 0;
    for (int d = 0; d < p.npeer; ++d) p.peer[d] = reinterpret_cast<double*>(static_cast<unsigned char*>(t[d]) + byte_offset);
}

// which: 0 = A, 1 = B, 2 = A2, 3 = B2.  mcontig selects the m-contiguous box of the A operand.
bool set_operand(Stage& st, EngineParams& p, int which, const MatView& m, bool mcontig)
{
    RawOperand r{static_cast<const double*>(m.ptr), m.ld, int(m.rows), int(m.cols)};
    (which == 0 ? p.rawA : which == 1 ? p.rawB : which == 2 ? p.rawA2 : p.rawB2) = r;
    st.opv[which] = m; st.opm[which] = mcontig; st.opset[which] = true;
    return true;
}

// Real launches with few logical tiles go to the 64 x 64-tile engine (four CTAs per tile: a quarter of
// the latency on the panel chain); GS_TILE64 = 0 never, 1 below plan->tile64_below tiles, 2 always.
bool use_tile64(const Stage& st, const EngineParams& p)
{
    if (st.z || !st.tma || st.plan->tile64_mode == 0 || (p.flags & F_NO_SPLIT) != 0) return false;
    return st.plan->tile64_mode == 2 || num_tiles(p) < st.plan->tile64_below;
}

gs_status_t launch(Stage& st, EngineParams& p, bool a_nn, int label)
{
    const bool t64 = use_tile64(st, p);
    for (int w = 0; w < 4; ++w) {
        if (!st.opset[w]) continue;
        st.opset[w] = false;
        if (!st.tma) continue;
        CUtensorMap* map = w == 0 ? &p.mapA : w == 1 ? &p.mapB : w == 2 ? &p.mapA2 : &p.mapB2;
        const bool zhalf = st.z && st.plan->ctile_half != 0;
        const int box = st.z ? (st.opm[w] ? 8 : ((zhalf && (w & 1)) ? 32 : CT)) : (st.opm[w] ? 16 : (t64 ? T64 : BN));
        if (!make_tensor_map(map, st.opv[w], box, st.z)) return GS_ERR_CUDA;
    }
    LaunchTimer timer(st.plan, label, st.stream);
    const cudaError_t e = st.z ? cengine_launch(p, a_nn, st.plan->ctile_half != 0, st.stream)
                               : t64 ? engine64_launch(p, a_nn, st.stream) : engine_launch(p, a_nn, st.tma, st.stream);
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
    if (plan->ws == nullptr || plan->ws_bytes < workspace_bytes(plan)) return GS_ERR_WORKSPACE;
    return GS_OK;
}

gs_status_t zero_lower(Stage& st, void* X)
{
    const gs_plan* plan = st.plan;
    const int N = int(plan->N);
    if (N <= st.lb) return GS_OK;
    dim3 grid(N, N > 2048 ? 8 : (N + 255) / 256);   // columns on grid.x: gridDim.y stops at 65535
    LaunchTimer timer(st.plan, L_ZERO_LOWER, st.stream);
    if (st.z) zero_lower_blocks_kernel<double2, CLB><<<grid, 256, 0, st.stream>>>(static_cast<double2*>(X), plan->N, N, info_ptr(plan));
    else zero_lower_blocks_kernel<double, LB><<<grid, 256, 0, st.stream>>>(static_cast<double*>(X), plan->N, N, info_ptr(plan));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(st.plan, e);
    st.plan->launches += 1;
    return GS_OK;
}

// ------------------------------------------------------------------------------------------------
// Block-recursive inversion by doubling of an nb-block upper triangular matrix whose diagonal
// 128-blocks are already inverted in the destination.  With U = [A B; 0 D],
// U^-1 = [A^-1, -A^-1 B D^-1; 0, D^-1].  Level s (in 128-blocks): all pairs (A = blocks
// [2is, 2is+s), D = the next s blocks) at once:
//   W = B * D^-1   (k <= J: D^-1 upper)      -> temp T, at the position of the target block
//   X = -A^-1 * W  (k >= I: A^-1 upper)      -> V
// The triangular matrix is the diagonal sub-block of vU starting at element offset uo; likewise vo
// (destination V) and to (temp T).
// ------------------------------------------------------------------------------------------------
gs_status_t invert_levels(Stage& st, const MatView& vU, int uo, const MatView& vV, int vo, const MatView& vT, int to,
                          int nb, int label_w, int label_x, int s_end = 1 << 30)
{
    gs_plan* plan = st.plan;
    double* V = static_cast<double*>(const_cast<void*>(vV.ptr));
    double* T = static_cast<double*>(const_cast<void*>(vT.ptr));
    for (int s = 1; s < nb && s < s_end; s *= 2) {   // s_end: stop once the diagonal s_end-blocks are inverted
        const int npairs = (nb - s + 2 * s - 1) / (2 * s);
        const int stride = 2 * s * st.lb;   // elements between consecutive pairs
        {   // W = B * Dinv
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vU, true) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
            p.C = T; p.ldc = vT.ld;
            p.tiles_m = s; p.tiles_n = s; p.batch = npairs; p.order = ORDER_COL_REV;
            p.c_row0 = to; p.c_col0 = to + s * st.lb; p.c_brow = stride; p.c_bcol = stride;
            p.c_rows = int(vT.rows); p.c_cols = int(vT.cols);
            p.khi_c = KPB; p.khi_j = KPB; p.kmax = s * (KPB);
            p.a.x0 = uo; p.a.bx = stride; p.a.k0 = uo + s * st.lb; p.a.bk = stride;
            p.b.k0 = vo + s * st.lb; p.b.bk = stride; p.b.x0 = vo + s * st.lb; p.b.bx = stride;
            GS_TRY(launch(st, p, true, label_w));
        }
        {   // X = -Ainv * W
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vV, true) || !set_operand(st, p, 1, vT, false)) return GS_ERR_CUDA;
            p.C = V; p.ldc = vV.ld;
            p.tiles_m = s; p.tiles_n = s; p.batch = npairs; p.order = ORDER_ROW;
            p.c_row0 = vo; p.c_col0 = vo + s * st.lb; p.c_brow = stride; p.c_bcol = stride;
            p.c_rows = int(vV.rows); p.c_cols = int(vV.cols);
            p.klo_i = KPB; p.khi_c = s * (KPB); p.kmax = s * (KPB);
            p.a.x0 = vo; p.a.bx = stride; p.a.k0 = vo; p.a.bk = stride;
            p.b.k0 = to; p.b.bk = stride; p.b.x0 = to + s * st.lb; p.b.bx = stride;
            p.alpha = -1.0;
            GS_TRY(launch(st, p, true, label_x));
        }
    }
    return GS_OK;
}

// ------------------------------------------------------------------------------------------------
// gs_cholesky: right-looking over panels of NB 128-blocks with one panel of look-ahead.
//
//   panel p = block rows [b1, b2).  Given the finished row panel p-1 = U[b0:b1, b1:n]:
//     side stream : A  S[b1:b2, b1:b2] -= U[b0:b1, b1:b2]^T U[b0:b1, b1:b2]     (diagonal block, upper tiles)
//                   B  recursive POTRF of the diagonal block (leaf kernels emit the inverted 128-blocks)
//                   C  Wp = U_pp^-1 by doubling
//     main stream : D  S[b1:b2, b2:n] -= U[b0:b1, b1:b2]^T U[b0:b1, b2:n]       (rest of the panel's rows)
//                   E  S[b2:n, b2:n] -= U[b0:b1, b2:n]^T U[b0:b1, b2:n]         (trailing matrix, upper tiles)
//     side stream : F  U[b1:b2, b2:n] = Wp^T S[b1:b2, b2:n]  (after D; one launch; out of place + copy back)
//   so the latency-bound chain A-B-C runs beside the large updates D, E, and the panel solve is a
//   single tensor-core launch instead of a chain of 128-row solves.
//   potrf(b0,b1): potrf(b0,mid); S12 = U11^-T S12 (trsm); S22 -= S12^T S12 (syrk); potrf(mid,b1)
//   trsm(r0,r1 | c0,c1): recursive on the triangular block; leaves multiply by the inverted
//   diagonal block W = U_kk^-1 produced by the leaf factorisation.
// ------------------------------------------------------------------------------------------------
struct Potrf {
    Stage st;
    void* S;
    MatView vS;
    MatView vT;   // the N x N workspace matrix
    MatView vW;   // inverse of the current panel's diagonal block (ldw x ldw), diagonal 128-blocks first
    int pb;       // first block of the current panel

    gs_status_t leaf(int b)
    {
        gs_plan* plan = st.plan;
        LaunchTimer timer(plan, L_POTRF_LEAF, st.stream);
        void* w = static_cast<unsigned char*>(const_cast<void*>(vW.ptr)) + size_t(b - pb) * st.lb * (vW.ld + 1) * plan->es;
        cudaError_t e;
        if (st.z)
            e = launch_pdl(potrf_cleaf_kernel, 1, kCLeafThreads, kCLeafSmemBytes, st.stream, static_cast<double2*>(S), plan->N, int(plan->N),
                           b * st.lb, static_cast<double2*>(w), vW.ld, info_ptr(plan));
        else if (plan->leaf_mode == 2)
            e = launch_pdl(potrf_leaf32_kernel, 1, kLeaf32Threads, kLeaf32SmemBytes, st.stream, static_cast<double*>(S), plan->N, int(plan->N),
                           b * st.lb, static_cast<double*>(w), vW.ld, info_ptr(plan));
        else
            e = launch_pdl(plan->leaf_mode == 1 ? potrf_leaf4_kernel : potrf_leaf_kernel, 1, kLeafThreads, kLeafSmemBytes, st.stream, static_cast<double*>(S), plan->N, int(plan->N),
                           b * st.lb, static_cast<double*>(w), vW.ld, info_ptr(plan));
        if (e != cudaSuccess) return cuda_fail(plan, e);
        plan->launches += 1;
        return GS_OK;
    }

    // X = W_r0^T * S[r0, c0:c1], in place (each CTA reads exactly the tile it overwrites)
    gs_status_t trsm_leaf(int r0, int c0, int c1)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vW, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(S); p.ldc = vS.ld;
        p.tiles_m = 1; p.tiles_n = c1 - c0; p.order = ORDER_COL;
        p.c_row0 = r0 * st.lb; p.c_col0 = c0 * st.lb; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = KPB; p.kmax = KPB;
        p.a.k0 = (r0 - pb) * st.lb; p.a.x0 = (r0 - pb) * st.lb;
        p.b.k0 = r0 * st.lb; p.b.x0 = c0 * st.lb;
        p.flags = F_NO_SPLIT;   // in place: a CTA may only read the tile it overwrites
        return launch(st, p, false, L_POTRF_TRSM);
    }

    // S[h:r1, c0:c1] -= U[r0:h, h:r1]^T * S[r0:h, c0:c1]
    gs_status_t gemm_update(int r0, int h, int r1, int c0, int c1)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vS, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(S); p.ldc = vS.ld;
        p.tiles_m = r1 - h; p.tiles_n = c1 - c0; p.order = ORDER_COL;
        p.c_row0 = h * st.lb; p.c_col0 = c0 * st.lb; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (h - r0) * (KPB); p.kmax = p.khi_c;
        p.a.k0 = r0 * st.lb; p.a.x0 = h * st.lb;
        p.b.k0 = r0 * st.lb; p.b.x0 = c0 * st.lb;
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
        p.C = static_cast<double*>(S); p.ldc = vS.ld;
        p.tiles_m = c1 - c0; p.tiles_n = c1 - c0; p.order = ORDER_TRI_ROW_DESC;
        p.c_row0 = c0 * st.lb; p.c_col0 = c0 * st.lb; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (k1 - k0) * (KPB); p.kmax = p.khi_c;
        p.a.k0 = k0 * st.lb; p.a.x0 = c0 * st.lb;
        p.b.k0 = k0 * st.lb; p.b.x0 = c0 * st.lb;
        p.alpha = -1.0; p.beta = 1.0;
        p.flags = F_STORE_UPPER | F_REAL_DIAG;   // HERK: the diagonal of U^H U is real
        return launch(st, p, false, L_POTRF_SYRK);
    }

    // rows [i0, i1) of the same update of S[.., i0:n]: S[i0:i1, i0:n] -= S[k0:k1, i0:i1]^T S[k0:k1, i0:n], upper tiles
    gs_status_t syrk_rows(int k0, int k1, int i0, int i1, int n)
    {
        EngineParams p = blank_params(st.plan);
        if (!set_operand(st, p, 0, vS, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(S); p.ldc = vS.ld;
        p.tiles_m = i1 - i0; p.tiles_n = n - i0; p.order = ORDER_TRAPEZOID;
        p.c_row0 = i0 * st.lb; p.c_col0 = i0 * st.lb; p.c_rows = int(vS.rows); p.c_cols = int(vS.cols);
        p.khi_c = (k1 - k0) * (KPB); p.kmax = p.khi_c;
        p.a.k0 = k0 * st.lb; p.a.x0 = i0 * st.lb;
        p.b.k0 = k0 * st.lb; p.b.x0 = i0 * st.lb;
        p.alpha = -1.0; p.beta = 1.0;
        p.flags = F_STORE_UPPER | F_REAL_DIAG;
        return launch(st, p, false, L_POTRF_SYRK);
    }

    // recursive factorisation of the diagonal block [b0, b1) (touches nothing outside it)
    gs_status_t potrf(int b0, int b1)
    {
        if (b1 - b0 == 1) return leaf(b0);
        if (st.plan->potrf_flat != 0) {
            // flat right-looking form: per block the leaf, ONE in-place solve of its row inside the panel, ONE update of the
            // rest of the panel block (3 launches per block instead of the recursion's 4: fewer, but K = 128 everywhere)
            for (int k = b0; k < b1; ++k) {
                GS_TRY(leaf(k));
                if (k + 1 < b1) {
                    GS_TRY(trsm_leaf(k, k + 1, b1));
                    GS_TRY(syrk(k, k + 1, k + 1, b1));
                }
            }
            return GS_OK;
        }
        const int mid = b0 + (b1 - b0 + 1) / 2;
        GS_TRY(potrf(b0, mid));
        GS_TRY(trsm(b0, mid, mid, b1));
        GS_TRY(syrk(b0, mid, mid, b1));
        return potrf(mid, b1);
    }

    // B + C: factor the diagonal block of panel [b1, b2) and, if a row panel follows, invert it
    gs_status_t panel_diag(int b1, int b2, int n)
    {
        pb = b1;
        GS_TRY(potrf(b1, b2));
        if (b2 < n) GS_TRY(invert_levels(st, vS, b1 * st.lb, vW, 0, vT, b1 * st.lb, b2 - b1, L_POTRF_GEMM, L_POTRF_GEMM));
        return GS_OK;
    }

    // F: U[b1:b2, c0:c1] = Wp^T S[b1:b2, c0:c1], through the workspace matrix (W = vW of that panel)
    gs_status_t panel_solve(const MatView& W, int b1, int b2, int c0, int c1)
    {
        if (c1 <= c0) return GS_OK;
        gs_plan* plan = st.plan;
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, W, false) || !set_operand(st, p, 1, vS, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(const_cast<void*>(vT.ptr)); p.ldc = vT.ld;
        p.tiles_m = b2 - b1; p.tiles_n = c1 - c0; p.order = ORDER_ROW_REV;
        p.c_row0 = b1 * st.lb; p.c_col0 = c0 * st.lb; p.c_rows = int(vT.rows); p.c_cols = int(vT.cols);
        p.khi_c = KPB; p.khi_i = KPB; p.kmax = (b2 - b1) * (KPB);
        p.a.k0 = 0; p.a.x0 = 0;
        p.b.k0 = b1 * st.lb; p.b.x0 = c0 * st.lb;
        GS_TRY(launch(st, p, false, L_POTRF_TRSM));
        const int N = int(plan->N);
        const int rows = (b2 * st.lb < N ? b2 * st.lb : N) - b1 * st.lb;
        const int cols = (c1 * st.lb < N ? c1 * st.lb : N) - c0 * st.lb;
        dim3 grid(cols, (rows + 255) / 256);
        LaunchTimer timer(plan, L_POTRF_TRSM, st.stream);
        cudaError_t e;
        if (st.z)
            e = launch_pdl(copy_block_kernel<double2>, grid, 256, 0, st.stream, static_cast<const double2*>(vT.ptr), static_cast<double2*>(S),
                           plan->N, b1 * st.lb, rows, c0 * st.lb, static_cast<const int*>(info_ptr(plan)));
        else
            e = launch_pdl(copy_block_kernel<double>, grid, 256, 0, st.stream, static_cast<const double*>(vT.ptr), static_cast<double*>(S),
                           plan->N, b1 * st.lb, rows, c0 * st.lb, static_cast<const int*>(info_ptr(plan)));
        if (e != cudaSuccess) return cuda_fail(plan, e);
        plan->launches += 1;
        return GS_OK;
    }

    // D: S[b1:b2, b2:n] -= U[b0:b1, b1:b2]^T U[b0:b1, b2:n]
    gs_status_t update_rows(int b0, int b1, int b2, int n) { return gemm_update(b0, b1, b2, b2, n); }

    // Panel boundaries: wide panels while the trailing matrix is large (the trailing update hides the
    // panel chain), narrower ones in the tail (the chain is exposed there, and it is shorter per row),
    // single blocks at the very end (the leaf's inverse IS the panel inverse: no doubling, no recursion).
    static std::vector<int> panel_starts(int n, const gs_plan* plan)
    {
        std::vector<int> s;
        int b = 0;
        while (b < n) {
            s.push_back(b);
            const int left = n - b;
            b += left > plan->potrf_tail ? plan->potrf_nb : left > plan->potrf_end ? plan->potrf_nb_tail : plan->potrf_nb_end;
        }
        s.push_back(n);
        return s;
    }

    // Iteration i applies row panel i-1 = U[s0:s1, s1:n] and factors panel i = [s1, s2); s3 = end of panel i+1.
    //   side : A_i  S[s1:s2, s1:s2] -= U[s0:s1, s1:s2]^T U[s0:s1, s1:s2]
    //          B_i, C_i  factor the diagonal block, invert it (Wp_i)
    //          F1_i U[s1:s2, s2:s3] = Wp_i^T S[s1:s2, s2:s3]     (after D_i; the columns panel i+1 needs first)
    //   main : F2_{i-1}  the remaining columns [s2, n) of row panel i-1
    //          D_i  S[s1:s2, s2:n] -= U[s0:s1, s1:s2]^T U[s0:s1, s2:n]
    //          E_i  S[s2:n, s2:n] -= U[s0:s1, s2:n]^T U[s0:s1, s2:n]
    gs_status_t factor(int n, cudaStream_t main_stream)
    {
        gs_plan* plan = st.plan;
        cudaStream_t side = plan->side;
        const std::vector<int> ps = panel_starts(n, plan);
        const int np = int(ps.size()) - 1;
        const int ldw = wp_ld(plan);
        auto W = [&](int i) { return MatView{wp_ptr(plan, i), ldw, ldw, ldw}; };
        st.stream = main_stream;
        vW = W(0);
        GS_TRY(panel_diag(ps[0], ps[1], n));
        if (np == 1) return GS_OK;
        GS_TRY(panel_solve(W(0), ps[0], ps[1], ps[1], ps[2]));            // F1_0
        gs_status_t rc = GS_OK;
        cudaError_t ce = cudaSuccess;
        auto cu = [&](cudaError_t e) { if (ce == cudaSuccess) ce = e; };
        for (int i = 1; i < np && rc == GS_OK && ce == cudaSuccess; ++i) {
            const int s0 = ps[i - 1], s1 = ps[i], s2 = ps[i + 1], s3 = (i + 1 < np) ? ps[i + 2] : n;
            cu(cudaEventRecord(plan->ev_fork, main_stream));
            cu(cudaStreamWaitEvent(side, plan->ev_fork, 0));
            st.stream = side;
            vW = W(i);
            rc = syrk(s0, s1, s1, s2);                                           // A_i
            if (rc == GS_OK) rc = panel_diag(s1, s2, n);                          // B_i, C_i
            st.stream = main_stream;
            if (rc == GS_OK) rc = panel_solve(W(i - 1), s0, s1, s2, n);           // F2_{i-1}
            if (s2 < n) {
                if (rc == GS_OK) rc = update_rows(s0, s1, s2, n);                 // D_i
                cu(cudaEventRecord(plan->ev_rows, main_stream));
                if (i == 1 && !plan->gates.empty()) {
                    // E_1 is the first launch that touches rows of S below the second panel: slab by slab
                    // as the rows arrive (gs_reduce_host); the slabs start at s2
                    for (size_t q = 0; q < plan->gates.size() && rc == GS_OK; ++q) {
                        const int r0 = plan->gates[q].first, r1 = q + 1 < plan->gates.size() ? plan->gates[q + 1].first : n;
                        cu(cudaStreamWaitEvent(main_stream, plan->gates[q].second, 0));
                        rc = syrk_rows(s0, s1, r0, r1, n);
                    }
                } else if (rc == GS_OK) {
                    rc = syrk(s0, s1, s2, n);                                     // E_i
                }
                cu(cudaStreamWaitEvent(side, plan->ev_rows, 0));
                st.stream = side;
                if (rc == GS_OK) rc = panel_solve(W(i), s1, s2, s2, s3);          // F1_i
                st.stream = main_stream;
            }
            // main continues only when the side chain of this iteration is done (also on failure)
            cu(cudaEventRecord(plan->ev_join, side));
            cu(cudaStreamWaitEvent(main_stream, plan->ev_join, 0));
        }
        GS_TRY(rc);
        GS_CUDA(plan, ce);
        return GS_OK;
    }
};

// ------------------------------------------------------------------------------------------------
// gs_cholesky_sharded: step 1 over the R GPUs of one NVSwitch domain.  Panels of potrf_nb blocks are dealt
// round-robin (panel p belongs to rank p mod R); a rank keeps the block columns of its own panels up to date
// and nothing else.  Per panel p = block rows [s1, s2), owner o:
//   o     : factor the diagonal block and invert it (the single-GPU chain: leaf kernels, one-tile solves, doubling),
//           copy U_pp and W_p = U_pp^-1 into every rank (copy_block_push_kernel), signal a_p
//   all   : wait a_p; for each own panel q > p:  U[p, q] = W_p^T S[p, q]  (one engine launch into the workspace),
//           copied into the own S AND into every peer's S -- the all-gather of the row panel, rank by rank, piece
//           by piece; signal b_p; wait for b_p of every rank
//   all   : for each own panel q > p:  S[(p, q], q] -= U[p, (p, q]]^T U[p, q]   (rectangle + upper diagonal block)
// (before the first panel every rank signals that its S is in place and waits for the others: nothing is stored into a
// buffer its owner is still filling)
// Look-ahead: the owner of panel p + 1 updates that panel first and factors its diagonal block before its other updates,
// so a_{p+1} is usually there when the other ranks have finished their updates of panel p.
// Ordering is on the device (gs_exchange_signal / gs_exchange_wait on flags[rank][source]); one stream per rank.
// On return (stream order) every rank holds the complete U.
// ------------------------------------------------------------------------------------------------
struct ShardedChol {
    int rank, nranks;
    void* const* peer_S;       // nranks entries (own entry = the rank's S)
    void* const* peer_ws;      // nranks entries: workspace base of every rank's plan (same geometry)
    void* const* flags;        // nranks entries: flag array (nranks x uint32) of every rank, own entry local
    uint32_t epoch0;
};

gs_status_t sharded_copy(Potrf& f, const void* src, long long lds, int srow0, int scol0, const PushTargets& dst, long long ldd,
                         int drow0, int dcol0, int rows, int cols, bool upper_only)
{
    gs_plan* plan = f.st.plan;
    if (rows <= 0 || cols <= 0 || dst.n == 0) return GS_OK;
    dim3 grid(cols, (rows + 255) / 256);
    LaunchTimer timer(plan, L_POTRF_TRSM, f.st.stream);
    cudaError_t e;
    if (f.st.z)
        e = launch_pdl(copy_block_push_kernel<double2>, grid, 256, 0, f.st.stream, static_cast<const double2*>(src), lds, srow0, scol0, dst, ldd,
                       drow0, dcol0, rows, upper_only ? 1 : 0, static_cast<const int*>(info_ptr(plan)));
    else
        e = launch_pdl(copy_block_push_kernel<double>, grid, 256, 0, f.st.stream, static_cast<const double*>(src), lds, srow0, scol0, dst, ldd,
                       drow0, dcol0, rows, upper_only ? 1 : 0, static_cast<const int*>(info_ptr(plan)));
    if (e != cudaSuccess) return cuda_fail(plan, e);
    plan->launches += 1;
    return GS_OK;
}

gs_status_t factor_sharded(Potrf& f, const ShardedChol& sh, cudaStream_t stream)
{
    gs_plan* plan = f.st.plan;
    const int N = int(plan->N), n = plan->nblk, lb = f.st.lb, R = sh.nranks, me = sh.rank;
    const int nbp = plan->potrf_nb < n ? plan->potrf_nb : n;
    const int np = (n + nbp - 1) / nbp;
    const int ldw = wp_ld(plan);
    auto start = [&](int p) { return p * nbp < n ? p * nbp : n; };
    auto el = [&](int b) { return b * lb < N ? b * lb : N; };      // first element of block b, clipped
    // flags: slot `me` of every other rank's array; own slots of every other rank
    std::vector<void*> sig, wt_all;
    for (int s = 0; s < R; ++s) {
        if (s == me) continue;
        sig.push_back(static_cast<unsigned char*>(sh.flags[s]) + 4 * size_t(me));
        wt_all.push_back(static_cast<unsigned char*>(sh.flags[me]) + 4 * size_t(s));
    }
    f.st.stream = stream;
    GS_TRY(zero_lower(f.st, f.S));
    // every rank's S is in place (whatever the caller enqueued before this call) before anything is stored into it
    if (!sig.empty()) {
        GS_TRY(stream_values(plan, false, int(sig.size()), sig.data(), sh.epoch0 + 1u, stream));
        GS_TRY(stream_values(plan, true, int(wt_all.size()), wt_all.data(), sh.epoch0 + 1u, stream));
    }
    auto a_of = [&](int p) { return sh.epoch0 + 2u * uint32_t(p) + 2u; };
    auto Wof = [&](int p) { return MatView{wp_ptr(plan, p), ldw, ldw, ldw}; };
    // owner: factor and invert the diagonal block of panel p, copy U_pp and (if a row panel follows) W_p into every other
    // rank, signal a_p
    auto diag_block = [&](int p) -> gs_status_t {
        const int s1 = start(p), s2 = start(p + 1);
        f.vW = Wof(p);
        GS_TRY(f.panel_diag(s1, s2, n));
        PushTargets ts{}, tw{};
        for (int s = 0; s < R; ++s) {
            if (s == me) continue;
            ts.ptr[ts.n++] = sh.peer_S[s];
            tw.ptr[tw.n++] = static_cast<unsigned char*>(sh.peer_ws[s]) + (static_cast<unsigned char*>(wp_ptr(plan, p)) - plan->ws);
        }
        const int rows = el(s2) - el(s1);
        GS_TRY(sharded_copy(f, f.S, plan->N, el(s1), el(s1), ts, plan->N, el(s1), el(s1), rows, rows, false));   // (with the zeros below its diagonal)
        if (s2 < n) GS_TRY(sharded_copy(f, Wof(p).ptr, ldw, 0, 0, tw, ldw, 0, 0, rows, rows, false));
        if (!sig.empty()) GS_TRY(stream_values(plan, false, int(sig.size()), sig.data(), a_of(p), stream));
        return GS_OK;
    };
    auto update_panel = [&](int p, int q) -> gs_status_t {     // S[(p, q], q] -= U[p, (p, q]]^H U[p, q]
        const int s1 = start(p), s2 = start(p + 1), c0 = start(q), c1 = start(q + 1);
        if (c0 > s2) GS_TRY(f.gemm_update(s1, s2, c0, c0, c1));        // rows (p, q) of the block columns of q
        return f.syrk(s1, s2, c0, c1);                                  // the diagonal block of q, upper tiles
    };
    bool have_diag = false;     // this rank factored the diagonal block of the current panel one iteration early
    for (int p = 0; p < np; ++p) {
        const int s1 = start(p), s2 = start(p + 1), o = p % R;
        const uint32_t b_p = a_of(p) + 1u;
        const MatView W = Wof(p);
        if (me == o) {
            if (!have_diag) GS_TRY(diag_block(p));
        } else {
            void* w = static_cast<unsigned char*>(sh.flags[me]) + 4 * size_t(o);
            GS_TRY(stream_values(plan, true, 1, &w, a_of(p), stream));
        }
        have_diag = false;
        if (s2 >= n) break;
        // own pieces of row panel p: into the workspace, then into the own S and every peer's S
        PushTargets all{};
        for (int s = 0; s < R; ++s) all.ptr[all.n++] = sh.peer_S[s];
        for (int q = p + 1; q < np; ++q) {
            if (q % R != me) continue;
            const int c0 = start(q), c1 = start(q + 1);
            EngineParams ep = blank_params(plan);
            if (!set_operand(f.st, ep, 0, W, false) || !set_operand(f.st, ep, 1, f.vS, false)) return GS_ERR_CUDA;
            ep.C = static_cast<double*>(const_cast<void*>(f.vT.ptr)); ep.ldc = f.vT.ld;
            ep.tiles_m = s2 - s1; ep.tiles_n = c1 - c0; ep.order = ORDER_ROW_REV;
            ep.c_row0 = s1 * lb; ep.c_col0 = c0 * lb; ep.c_rows = int(f.vT.rows); ep.c_cols = int(f.vT.cols);
            ep.khi_c = KPB; ep.khi_i = KPB; ep.kmax = (s2 - s1) * (KPB);
            ep.a.k0 = 0; ep.a.x0 = 0;
            ep.b.k0 = s1 * lb; ep.b.x0 = c0 * lb;
            GS_TRY(launch(f.st, ep, false, L_POTRF_TRSM));
            GS_TRY(sharded_copy(f, f.vT.ptr, f.vT.ld, el(s1), el(c0), all, plan->N, el(s1), el(c0), el(s2) - el(s1), el(c1) - el(c0), false));
        }
        if (!sig.empty()) {
            GS_TRY(stream_values(plan, false, int(sig.size()), sig.data(), b_p, stream));
            GS_TRY(stream_values(plan, true, int(wt_all.size()), wt_all.data(), b_p, stream));
        }
        // look-ahead: the owner of the NEXT panel updates that panel first and factors its diagonal block at once, so that
        // its chain runs beside the other ranks' (and its own remaining) trailing updates
        const int pn = p + 1;
        if (pn < np && pn % R == me) {
            GS_TRY(update_panel(p, pn));
            GS_TRY(diag_block(pn));
            have_diag = true;
        }
        for (int q = p + 1; q < np; ++q) {
            if (q % R != me || (q == pn && have_diag)) continue;
            GS_TRY(update_panel(p, q));
        }
    }
    return GS_OK;
}

gs_status_t ensure_side_stream(gs_plan* plan)
{
    if (plan->side != nullptr) return GS_OK;
    int lo = 0, hi = 0;
    GS_CUDA(plan, cudaDeviceGetStreamPriorityRange(&lo, &hi));
    GS_CUDA(plan, cudaStreamCreateWithPriority(&plan->side, cudaStreamNonBlocking, hi));
    GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_fork, cudaEventDisableTiming));
    GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_rows, cudaEventDisableTiming));
    GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_join, cudaEventDisableTiming));
    return GS_OK;
}

// the opt-in to > 48 KB of dynamic shared memory is a per-device attribute (engine_host.cuh: PerDeviceOnce)
gs_status_t configure_leaf(gs_plan* plan)
{
    static PerDeviceOnce once;
    const cudaError_t e = once.run([]() -> cudaError_t {
        cudaError_t r = cudaFuncSetAttribute(potrf_leaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeafSmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(potrf_leaf4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeafSmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(potrf_leaf32_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeaf32SmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(trtri_leaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kLeafSmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(potrf_cleaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCLeafSmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(trtri_cleaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCLeafSmemBytes);
        return r;
    });
    if (e != cudaSuccess) return cuda_fail(plan, e);
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
    p->z = dtype == GS_COMPLEX128;
    p->lb = p->z ? CLB : LB;
    p->bk = p->z ? CBK : BK;
    p->es = p->z ? 2 * sizeof(double) : sizeof(double);
    p->nblk = int((N + p->lb - 1) / p->lb);
    // tuning knobs of the POTRF schedule
    auto knob = [](const char* name, int lo, int hi, int* out) {
        if (const char* e = std::getenv(name)) {
            const int v = std::atoi(e);
            if (v >= lo && v <= hi) *out = v;
        }
    };
    knob("GS_POTRF_NB", 1, 256, &p->potrf_nb);
    knob("GS_POTRF_NB_TAIL", 1, 32, &p->potrf_nb_tail);
    knob("GS_POTRF_TAIL", 0, 1 << 20, &p->potrf_tail);
    knob("GS_POTRF_NB_END", 1, 32, &p->potrf_nb_end);
    knob("GS_POTRF_END", 0, 1 << 20, &p->potrf_end);
    if (p->potrf_nb_end > p->potrf_nb_tail) p->potrf_nb_end = p->potrf_nb_tail;
    if (p->potrf_nb_tail > p->potrf_nb) p->potrf_nb_tail = p->potrf_nb;
    p->super_tile = p->z ? 16 : 8;
    knob("GS_SUPER_TILE", 0, 64, &p->super_tile);
    p->super_syr2k = p->super_tile > 4 ? 4 : p->super_tile;
    knob("GS_SUPER_SYR2K", 0, 64, &p->super_syr2k);
    knob("GS_POTRF_FLAT", 0, 1, &p->potrf_flat);
    knob("GS_TILE64", 0, 2, &p->tile64_mode);
    knob("GS_CTILE_HALF", 0, 1, &p->ctile_half);
    knob("GS_TILE64_BELOW", 0, 1 << 30, &p->tile64_below);
    knob("GS_LEAF_BLOCKED", 0, 1, &p->leaf_blocked);
    if (p->leaf_blocked) p->leaf_mode = 1;
    knob("GS_LEAF", 0, 2, &p->leaf_mode);
    int shard_log2 = p->z ? 4 : 3;   // 1024 rows per panel of the column-range inversion
    knob("GS_SHARD_PANEL_LOG2", 0, 8, &shard_log2);
    p->shard_panel = 1 << shard_log2;
    *plan = p;
    return GS_OK;
}

gs_status_t gs_plan_destroy(gs_plan_t* plan)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    clear_timed(plan);
    if (plan->ev_fork != nullptr) cudaEventDestroy(plan->ev_fork);
    if (plan->ev_rows != nullptr) cudaEventDestroy(plan->ev_rows);
    if (plan->ev_join != nullptr) cudaEventDestroy(plan->ev_join);
    if (plan->side != nullptr) cudaStreamDestroy(plan->side);
    if (plan->ev_copy != nullptr) cudaEventDestroy(plan->ev_copy);
    if (plan->copy != nullptr) cudaStreamDestroy(plan->copy);
    if (plan->copy_out != nullptr) cudaStreamDestroy(plan->copy_out);
    for (cudaEvent_t e : plan->ev_pool) cudaEventDestroy(e);
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

// the leading nlead blocks (leading principal blocks of a Cholesky factor nest: chol(S[:k,:k]) = U[:k,:k])
static gs_status_t cholesky_blocks(gs_plan_t* plan, void* S_inout, int nlead, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (S_inout == nullptr || !aligned16(S_inout)) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    GS_CUDA(plan, cudaMemsetAsync(info_ptr(plan), 0, sizeof(int), stream));
    void* S = S_inout;
    Potrf f;
    f.st = make_stage(plan, stream);
    f.S = S;
    f.vS = MatView{S, plan->N, plan->N, plan->N};
    f.vT = MatView{big_ptr(plan), plan->N, plan->N, plan->N};
    f.pb = 0;
    if (plan->nblk <= 1) return f.factor(plan->nblk, stream);
    GS_TRY(ensure_side_stream(plan));
    // the off-diagonal lower blocks are never touched by the factorisation: zero them on the side
    // stream, beside the first panel (its own fork/join events; factor() forks after this work)
    GS_CUDA(plan, cudaEventRecord(plan->ev_fork, stream));
    GS_CUDA(plan, cudaStreamWaitEvent(plan->side, plan->ev_fork, 0));
    f.st.stream = plan->side;
    const gs_status_t zs = zero_lower(f.st, S);
    f.st.stream = stream;
    const gs_status_t fs = zs == GS_OK ? f.factor(nlead, stream) : zs;
    // factor() joins the side stream after every panel; a single-panel factorisation has no join of its own
    const cudaError_t e1 = cudaEventRecord(plan->ev_join, plan->side);
    const cudaError_t e2 = cudaStreamWaitEvent(stream, plan->ev_join, 0);
    GS_TRY(fs);
    GS_CUDA(plan, e1);
    GS_CUDA(plan, e2);
    return GS_OK;
}

gs_status_t gs_cholesky(gs_plan_t* plan, void* S_inout, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    return cholesky_blocks(plan, S_inout, plan->nblk, cuda_stream);
}

gs_status_t gs_cholesky_leading(gs_plan_t* plan, void* S_inout, int64_t ncols, void* cuda_stream)
{
    if (plan == nullptr || ncols < 0 || ncols > plan->N || (ncols % plan->lb != 0 && ncols != plan->N)) return GS_ERR_INVALID_ARG;
    if (ncols == 0) return check_ready(plan);
    return cholesky_blocks(plan, S_inout, int((ncols + plan->lb - 1) / plan->lb), cuda_stream);
}

// first exact zero among the first n diagonal entries of U -> info = -(index + 1), deterministically
static gs_status_t check_diagonal(gs_plan* plan, const void* U, int64_t n, cudaStream_t stream)
{
    LaunchTimer timer(plan, L_TRTRI_LEAF, stream);
    if (plan->z) check_diagonal_kernel<double2><<<1, 1024, 0, stream>>>(static_cast<const double2*>(U), plan->N, int(n), info_ptr(plan));
    else check_diagonal_kernel<double><<<1, 1024, 0, stream>>>(static_cast<const double*>(U), plan->N, int(n), info_ptr(plan));
    GS_CUDA(plan, cudaGetLastError());
    plan->launches += 1;
    return GS_OK;
}

// V = U^-1: every diagonal 128-block inverted by the leaf kernel, then block-recursive doubling.
gs_status_t gs_invert_triangular(gs_plan_t* plan, const void* U_, void* Uinv_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (U_ == nullptr || Uinv_ == nullptr || !aligned16(U_) || !aligned16(Uinv_) ||
        overlaps(U_, mat_bytes(plan), Uinv_, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    const void* U = U_;
    void* V = Uinv_;
    const int N = int(plan->N), nblk = plan->nblk;
    Stage st = make_stage(plan, stream);

    GS_TRY(check_diagonal(plan, U, N, stream));
    {
        LaunchTimer timer(plan, L_TRTRI_LEAF, stream);
        if (plan->z)
            trtri_cleaf_kernel<<<nblk, kCLeafThreads, kCLeafSmemBytes, stream>>>(static_cast<const double2*>(U), static_cast<double2*>(V),
                                                                                 plan->N, N, info_ptr(plan));
        else
            trtri_leaf_kernel<<<nblk, kLeafThreads, kLeafSmemBytes, stream>>>(static_cast<const double*>(U), static_cast<double*>(V),
                                                                              plan->N, N, info_ptr(plan));
    }
    GS_CUDA(plan, cudaGetLastError());
    plan->launches += 1;
    GS_TRY(zero_lower(st, V));

    const MatView vU{U, N, N, N}, vV{V, N, N, N}, vT{big_ptr(plan), N, N, N};
    return invert_levels(st, vU, 0, vV, 0, vT, 0, nblk, L_TRTRI_W, L_TRTRI_X);
}

// H~ = V^T H V with H = T + T^T, T = triu(H,1) + diag(H)/2:
//   G  = T V                (upper x upper = upper; N^3/3 flop)   -> workspace
//   H~ = V^T G + G^T V      (upper triangle only; SYR2K-shaped, operands triangular; 2N^3/3 flop)
// N^3 flop in total instead of the 4N^3/3 of forming W = H V in full.
// Row ranges of the SYR2K-shaped launch for the host-buffer path: splits (in blocks, ascending) and a hook
// that is called after range r = [splits[r], splits[r+1]) has been enqueued.
struct RowRanges {
    std::vector<int> splits;
    std::function<gs_status_t(int)> after;
};

// rows [I0, I1) (in blocks) of H~ = V^H G + G^H V, upper tiles; whole = the plain triangular launch
static gs_status_t to_standard_rows(gs_plan* plan, Stage& st, const MatView& vV, const MatView& vG, void* Htilde_, int I0, int I1, bool whole)
{
    const int N = int(plan->N), nblk = plan->nblk, kt = KPB;
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vV, false) || !set_operand(st, p, 1, vG, false) || !set_operand(st, p, 2, vG, false) ||
        !set_operand(st, p, 3, vV, false))
        return GS_ERR_CUDA;
    p.C = static_cast<double*>(Htilde_); p.ldc = N;
    p.c_rows = N; p.c_cols = N;
    p.kmax = (N + st.bk - 1) / st.bk;
    p.flags = F_DUAL | F_MASK_A | F_MASK_B2 | F_STORE_UPPER | F_REAL_DIAG;   // Hermitian: Im(diag) = 0 exactly
    if (whole) {
        p.tiles_m = nblk; p.tiles_n = nblk; p.order = ORDER_TRI_ROW_DESC;
        p.khi_c = kt; p.khi_i = kt;
        if (!plan->z) p.super = plan->super_syr2k;   // four operand panels per tile: its own super-tile edge (profiles/)
    } else {
        p.tiles_m = I1 - I0; p.tiles_n = nblk - I0; p.order = ORDER_TRAPEZOID;
        p.c_row0 = I0 * st.lb; p.c_col0 = I0 * st.lb;
        p.a.x0 = p.b.x0 = p.a2.x0 = p.b2.x0 = I0 * st.lb;
        p.khi_c = kt * (I0 + 1); p.khi_i = kt;
    }
    return launch(st, p, false, L_TOSTD_SYR2K);
}

static gs_status_t to_standard_impl(gs_plan* plan, const void* H_, const void* Uinv_, void* Htilde_, void* cuda_stream, RowRanges* ranges)
{
    GS_TRY(check_ready(plan));
    if (H_ == nullptr || Uinv_ == nullptr || Htilde_ == nullptr || !aligned16(H_) || !aligned16(Uinv_) || !aligned16(Htilde_) ||
        overlaps(Htilde_, mat_bytes(plan), H_, mat_bytes(plan)) || overlaps(Htilde_, mat_bytes(plan), Uinv_, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int N = int(plan->N), nblk = plan->nblk;
    Stage st = make_stage(plan, stream);
    void* G = big_ptr(plan);
    const MatView vH{H_, N, N, N}, vV{Uinv_, N, N, N}, vG{G, N, N, N};
    const int kt = KPB;
    {
        // G = T V computed as L^H V with L = tril(H,-1) + diag(H)/2 (L^H = T because H is Hermitian): the
        // k-contiguous ("TN") mainloop reads column I of H below the diagonal -- it runs ~4 % closer to
        // the pipe than the m-contiguous one (profiles/r01c_perkernel.md)
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, vH, false) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(G); p.ldc = N;
        p.tiles_m = nblk; p.tiles_n = nblk; p.order = ORDER_TRI_DIAG_DESC;
        p.c_rows = N; p.c_cols = N;
        p.klo_i = kt; p.khi_c = kt; p.khi_j = kt; p.kmax = (N + st.bk - 1) / st.bk;
        p.flags = F_MASK_A | F_LOWER_A | F_HALF_DIAG_A | F_MASK_B;
        GS_TRY(launch(st, p, false, L_TOSTD_G));
    }
    if (ranges == nullptr) return to_standard_rows(plan, st, vV, vG, Htilde_, 0, nblk, true);
    // host-buffer path: the triangle is formed in row ranges of about equal work so that the D2H copy of a
    // finished range runs beside the next one; top rows first -- they are the long ones, the copy that
    // is left exposed at the end is the short bottom trapezoid
    for (int r = 0; r + 1 < int(ranges->splits.size()); ++r) {
        GS_TRY(to_standard_rows(plan, st, vV, vG, Htilde_, ranges->splits[r], ranges->splits[r + 1], false));
        GS_TRY(ranges->after(r));
    }
    return GS_OK;
}

gs_status_t gs_to_standard(gs_plan_t* plan, const void* H_, const void* Uinv_, void* Htilde_, void* cuda_stream)
{
    return to_standard_impl(plan, H_, Uinv_, Htilde_, cuda_stream, nullptr);
}

// C[:, col0 : col0+ncols] = V * C~[:, col0 : col0+ncols]
static gs_status_t backtransform_cols(gs_plan* plan, const void* Uinv_, const void* Ctilde_, void* C_, int col0, int ncols, cudaStream_t stream,
                                      bool push = false)
{
    const int N = int(plan->N);
    Stage st = make_stage(plan, stream);
    const size_t off = size_t(col0) * size_t(N) * plan->es;
    const MatView vV{Uinv_, N, N, N}, vC{static_cast<const unsigned char*>(Ctilde_) + off, N, ncols, N};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vV, true) || !set_operand(st, p, 1, vC, false)) return GS_ERR_CUDA;
    p.C = reinterpret_cast<double*>(static_cast<unsigned char*>(C_) + off); p.ldc = N;
    p.tiles_m = plan->nblk; p.tiles_n = (ncols + st.lb - 1) / st.lb; p.order = ORDER_ROW;
    p.c_rows = N; p.c_cols = ncols;
    p.klo_i = KPB; p.khi_c = (N + st.bk - 1) / st.bk; p.kmax = p.khi_c;
    p.flags = F_MASK_A;
    if (push) set_peers(plan, p, GS_PUSH_C, off);
    return launch(st, p, true, L_BACK_TRMM);
}

gs_status_t gs_backtransform(gs_plan_t* plan, const void* Uinv_, const void* Ctilde_, void* C_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (plan->nev == 0) return GS_OK;
    if (Uinv_ == nullptr || Ctilde_ == nullptr || C_ == nullptr || !aligned16(Uinv_) || !aligned16(Ctilde_) || !aligned16(C_) ||
        overlaps(C_, vec_bytes(plan), Ctilde_, vec_bytes(plan)) || overlaps(C_, vec_bytes(plan), Uinv_, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    return backtransform_cols(plan, Uinv_, Ctilde_, C_, 0, int(plan->nev), static_cast<cudaStream_t>(cuda_stream));
}

// ------------------------------------------------------------------------------------------------
// Column-range entry points: every call forms the
// block columns J = [col0, col0 + ncols) of its result from inputs that do not depend on the other
// columns of the same result, so R GPUs form disjoint column ranges side by side and exchange the
// finished slabs once.
// ------------------------------------------------------------------------------------------------
static bool col_range_ok(const gs_plan* plan, int64_t col0, int64_t ncols, int64_t width)
{
    if (col0 < 0 || ncols < 0 || col0 + ncols > width) return false;
    if (ncols == 0) return true;                       // an empty range (more ranks than blocks) is a no-op
    if (col0 % plan->lb != 0) return false;
    return (col0 + ncols) % plan->lb == 0 || col0 + ncols == width;
}

// V[:, J] = (U^-1)[:, J] by blocked back substitution over panels of P blocks (U X = E_J):
//   diagonal P-blocks D_i^-1 by the doubling levels s < P (every rank forms them; N (P lb)^2 / 3 flop),
//   T[:, J] = 0, then right-looking from the last panel row that reaches into J up to panel 0:
//     X[i, cols right of panel i] = -D_i^-1 T[i, .]                      (T[i, .] is complete by now)
//     T[0 : i, cols] += U[0 : i, i] X[i, cols]      for all rows above, cols of J from panel i on
//   N^3/3 flop over all columns, as the doubling scheme, but no column needs another column range; the
//   updates are launches of (i P) x |J| tiles, so narrow ranges still fill the machine.
gs_status_t gs_invert_triangular_cols(gs_plan_t* plan, const void* U_, void* Uinv_, int64_t col0, int64_t ncols, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (U_ == nullptr || Uinv_ == nullptr || !aligned16(U_) || !aligned16(Uinv_) || overlaps(U_, mat_bytes(plan), Uinv_, mat_bytes(plan)) ||
        !col_range_ok(plan, col0, ncols, plan->N))
        return GS_ERR_INVALID_ARG;
    if (ncols == 0) return GS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    const int N = int(plan->N), lb = plan->lb;
    const int jb0 = int(col0 / lb), jb1 = int((col0 + ncols + lb - 1) / lb);
    const int P = plan->shard_panel;
    Stage st = make_stage(plan, stream);
    double* V = static_cast<double*>(Uinv_);
    GS_TRY(check_diagonal(plan, U_, std::min<int64_t>(int64_t(jb1) * lb, N), stream));
    {
        LaunchTimer timer(plan, L_TRTRI_LEAF, stream);
        if (plan->z)
            trtri_cleaf_kernel<<<jb1, kCLeafThreads, kCLeafSmemBytes, stream>>>(static_cast<const double2*>(U_), static_cast<double2*>(Uinv_),
                                                                                plan->N, N, info_ptr(plan));
        else
            trtri_leaf_kernel<<<jb1, kLeafThreads, kLeafSmemBytes, stream>>>(static_cast<const double*>(U_), V, plan->N, N, info_ptr(plan));
    }
    GS_CUDA(plan, cudaGetLastError());
    plan->launches += 1;
    GS_TRY(zero_lower(st, Uinv_));
    const MatView vU{U_, N, N, N}, vV{Uinv_, N, N, N}, vT{big_ptr(plan), N, N, N};
    GS_TRY(invert_levels(st, vU, 0, vV, 0, vT, 0, jb1, L_TRTRI_W, L_TRTRI_X, P));
    if (!plan->push[GS_PUSH_UINV].empty()) {   // the diagonal band of the slab goes out by a copy kernel, the rest from the engine
        PushTargets pt{};
        pt.n = int(plan->push[GS_PUSH_UINV].size());
        for (int d = 0; d < pt.n; ++d) pt.ptr[d] = plan->push[GS_PUSH_UINV][d];
        const int band = P * lb;
        dim3 grid(unsigned(ncols), (band + 255) / 256);
        LaunchTimer timer(plan, L_PUSH_BAND, stream);
        if (plan->z) push_band_kernel<double2><<<grid, 256, 0, stream>>>(static_cast<const double2*>(Uinv_), pt, plan->N, N, int(col0), band, info_ptr(plan));
        else push_band_kernel<double><<<grid, 256, 0, stream>>>(static_cast<const double*>(Uinv_), pt, plan->N, N, int(col0), band, info_ptr(plan));
        GS_CUDA(plan, cudaGetLastError());
        plan->launches += 1;
    }
    const int npan = (jb1 + P - 1) / P;
    if (npan < 2) return GS_OK;
    {
        LaunchTimer timer(plan, L_ZERO_LOWER, stream);
        GS_CUDA(plan, cudaMemsetAsync(static_cast<unsigned char*>(big_ptr(plan)) + size_t(col0) * size_t(N) * plan->es, 0,
                                      size_t(ncols) * size_t(N) * plan->es, stream));
    }
    for (int i = npan - 1; i >= 0; --i) {
        const int r0 = i * P, r1 = (r0 + P < jb1) ? r0 + P : jb1;   // panel rows [r0, r1) in blocks
        const int cb = jb0 > r0 + P ? jb0 : r0 + P;                 // first column block right of the panel
        if (cb < jb1) {   // X[r0:r1, cb:] = -D_i^-1 T[r0:r1, cb:]   (a panel left of other columns is a full one)
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vV, true) || !set_operand(st, p, 1, vT, false)) return GS_ERR_CUDA;
            p.C = V; p.ldc = N;
            p.tiles_m = P; p.tiles_n = jb1 - cb; p.order = ORDER_ROW;
            p.c_row0 = r0 * lb; p.c_col0 = cb * lb; p.c_rows = N; p.c_cols = N;
            p.klo_i = KPB; p.khi_c = P * KPB; p.kmax = P * KPB;
            p.a.x0 = r0 * lb; p.a.k0 = r0 * lb; p.b.k0 = r0 * lb; p.b.x0 = cb * lb;
            p.alpha = -1.0;
            set_peers(plan, p, GS_PUSH_UINV);
            GS_TRY(launch(st, p, true, L_TRTRI_X));
        }
        if (i == 0) break;
        const int cu = jb0 > r0 ? jb0 : r0;                         // columns of J from the panel's own block on
        {   // T[0:r0, cu:] += U[0:r0, r0:r1] X[r0:r1, cu:]; inside the panel X is upper triangular: k up to the column's block
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vU, true) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
            p.C = static_cast<double*>(big_ptr(plan)); p.ldc = N;
            p.tiles_m = r0; p.tiles_n = jb1 - cu; p.order = ORDER_COL_REV;
            p.c_col0 = cu * lb; p.c_rows = N; p.c_cols = N;
            p.khi_c = KPB * (cu - r0 + 1); p.khi_j = KPB; p.kmax = KPB * (r1 - r0);
            p.a.k0 = r0 * lb; p.b.k0 = r0 * lb; p.b.x0 = cu * lb;
            p.beta = 1.0;
            GS_TRY(launch(st, p, true, L_TRTRI_W));
        }
    }
    return GS_OK;
}

// G[:, J] = T Uinv[:, J], T = triu(H,1) + diag(H)/2, evaluated as L^H Uinv like the first launch of
// gs_to_standard; rows below the diagonal blocks of J are written as zeros.
gs_status_t gs_to_standard_g_cols(gs_plan_t* plan, const void* H_, const void* Uinv_, void* G_, int64_t col0, int64_t ncols,
                                  void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (H_ == nullptr || Uinv_ == nullptr || G_ == nullptr || !aligned16(H_) || !aligned16(Uinv_) || !aligned16(G_) ||
        overlaps(G_, mat_bytes(plan), H_, mat_bytes(plan)) || overlaps(G_, mat_bytes(plan), Uinv_, mat_bytes(plan)) ||
        !col_range_ok(plan, col0, ncols, plan->N))
        return GS_ERR_INVALID_ARG;
    if (ncols == 0) return GS_OK;
    const int N = int(plan->N), lb = plan->lb, kt = KPB;
    const int jb0 = int(col0 / lb), jb1 = int((col0 + ncols + lb - 1) / lb);
    Stage st = make_stage(plan, static_cast<cudaStream_t>(cuda_stream));
    const MatView vH{H_, N, N, N}, vV{Uinv_, N, N, N};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vH, false) || !set_operand(st, p, 1, vV, false)) return GS_ERR_CUDA;
    p.C = static_cast<double*>(G_); p.ldc = N;
    p.tiles_m = jb1; p.tiles_n = jb1 - jb0; p.order = ORDER_COL_REV;
    p.c_col0 = jb0 * lb; p.b.x0 = jb0 * lb;
    p.c_rows = N; p.c_cols = int(col0 + ncols);
    p.klo_i = kt; p.khi_c = kt * (jb0 + 1); p.khi_j = kt; p.kmax = (N + st.bk - 1) / st.bk;
    p.flags = F_MASK_A | F_LOWER_A | F_HALF_DIAG_A | F_MASK_B;
    set_peers(plan, p, GS_PUSH_G);
    return launch(st, p, false, L_TOSTD_G);
}

// Htilde[0 : col0+ncols, J] = Uinv^H G + G^H Uinv, upper part: needs the columns [0, col0 + ncols) of
// Uinv and of G (those of the lower-numbered ranges and its own), nothing to the right of J.
gs_status_t gs_to_standard_cols(gs_plan_t* plan, const void* Uinv_, const void* G_, void* Htilde_, int64_t col0, int64_t ncols,
                                void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (Uinv_ == nullptr || G_ == nullptr || Htilde_ == nullptr || !aligned16(Uinv_) || !aligned16(G_) || !aligned16(Htilde_) ||
        overlaps(Htilde_, mat_bytes(plan), G_, mat_bytes(plan)) || overlaps(Htilde_, mat_bytes(plan), Uinv_, mat_bytes(plan)) ||
        overlaps(G_, mat_bytes(plan), Uinv_, mat_bytes(plan)) || !col_range_ok(plan, col0, ncols, plan->N))
        return GS_ERR_INVALID_ARG;
    if (ncols == 0) return GS_OK;
    const int N = int(plan->N), lb = plan->lb, kt = KPB;
    const int jb0 = int(col0 / lb), jb1 = int((col0 + ncols + lb - 1) / lb);
    Stage st = make_stage(plan, static_cast<cudaStream_t>(cuda_stream));
    const MatView vV{Uinv_, N, N, N}, vG{G_, N, N, N};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vV, false) || !set_operand(st, p, 1, vG, false) || !set_operand(st, p, 2, vG, false) ||
        !set_operand(st, p, 3, vV, false))
        return GS_ERR_CUDA;
    p.C = static_cast<double*>(Htilde_); p.ldc = N;
    p.tiles_m = jb1; p.tiles_n = jb1 - jb0; p.order = ORDER_ROW_REV;      // rows descending: long tiles first
    p.c_col0 = jb0 * lb; p.b.x0 = p.b2.x0 = jb0 * lb;
    p.c_rows = N; p.c_cols = int(col0 + ncols);
    p.kmax = (N + st.bk - 1) / st.bk;
    p.khi_c = kt; p.khi_i = kt;
    // tiles below the diagonal (I > jb0 + J) get an empty k-range and store nothing: k_lo = kmax (I - jb0 - J)
    p.klo_c = -p.kmax * jb0; p.klo_i = p.kmax; p.klo_j = -p.kmax;
    p.flags = F_DUAL | F_MASK_A | F_MASK_B2 | F_STORE_UPPER | F_REAL_DIAG;
    set_peers(plan, p, GS_PUSH_HTILDE);
    return launch(st, p, false, L_TOSTD_SYR2K);
}

// C[:, K] = Uinv Ctilde[:, K] for the eigenvector columns K = [col0, col0 + ncols) of the plan's nev.
gs_status_t gs_backtransform_cols(gs_plan_t* plan, const void* Uinv_, const void* Ctilde_, void* C_, int64_t col0, int64_t ncols,
                                  void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (col0 < 0 || ncols < 0 || col0 + ncols > plan->nev) return GS_ERR_INVALID_ARG;
    if (ncols == 0) return GS_OK;
    if (Uinv_ == nullptr || Ctilde_ == nullptr || C_ == nullptr || !aligned16(Uinv_) || !aligned16(Ctilde_) || !aligned16(C_) ||
        overlaps(C_, vec_bytes(plan), Ctilde_, vec_bytes(plan)) || overlaps(C_, vec_bytes(plan), Uinv_, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    if (!plan->z && ((col0 * plan->N) % 2 != 0)) return GS_ERR_INVALID_ARG;   // 16-byte aligned column start
    return backtransform_cols(plan, Uinv_, Ctilde_, C_, int(col0), int(ncols), static_cast<cudaStream_t>(cuda_stream), true);
}

// Fused exchange: see include/gs.h.
gs_status_t gs_plan_set_push_targets(gs_plan_t* plan, gs_push_kind_t kind, int count, void* const* targets)
{
    if (plan == nullptr || int(kind) < 0 || int(kind) > 3 || count < 0 || count > kMaxPeers || (count > 0 && targets == nullptr))
        return GS_ERR_INVALID_ARG;
    for (int d = 0; d < count; ++d)
        if (targets[d] == nullptr || !aligned16(targets[d])) return GS_ERR_INVALID_ARG;
    plan->push[kind].assign(targets, targets + count);
    return GS_OK;
}

gs_status_t gs_exchange_signal(gs_plan_t* plan, int count, void* const* flags, uint32_t value, void* cuda_stream)
{
    return stream_values(plan, false, count, flags, value, cuda_stream);
}

gs_status_t gs_exchange_wait(gs_plan_t* plan, int count, void* const* flags, uint32_t value, void* cuda_stream)
{
    return stream_values(plan, true, count, flags, value, cuda_stream);
}

// CUDA IPC plumbing for the push targets: a device allocation of another process (one process per GPU) mapped here.
gs_status_t gs_ipc_export(const void* dev_ptr, unsigned char* handle64, uint64_t* offset)
{
    if (dev_ptr == nullptr || handle64 == nullptr || offset == nullptr) return GS_ERR_INVALID_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "IPC handle size");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
        return GS_ERR_CUDA;
    CUdeviceptr base = 0;
    size_t size = 0;
    if (reinterpret_cast<CUresult (*)(CUdeviceptr*, size_t*, CUdeviceptr)>(fn)(&base, &size, reinterpret_cast<CUdeviceptr>(dev_ptr)) != CUDA_SUCCESS)
        return GS_ERR_CUDA;
    cudaIpcMemHandle_t h;
    if (cudaIpcGetMemHandle(&h, reinterpret_cast<void*>(base)) != cudaSuccess) { cudaGetLastError(); return GS_ERR_CUDA; }
    std::memcpy(handle64, &h, 64);
    *offset = uint64_t(reinterpret_cast<CUdeviceptr>(dev_ptr) - base);
    return GS_OK;
}

gs_status_t gs_ipc_open(const unsigned char* handle64, uint64_t offset, void** dev_ptr)
{
    if (handle64 == nullptr || dev_ptr == nullptr) return GS_ERR_INVALID_ARG;
    cudaIpcMemHandle_t h;
    std::memcpy(&h, handle64, 64);
    void* base = nullptr;
    if (cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess) != cudaSuccess) { cudaGetLastError(); return GS_ERR_CUDA; }
    *dev_ptr = static_cast<unsigned char*>(base) + offset;
    return GS_OK;
}

gs_status_t gs_ipc_close(void* dev_ptr, uint64_t offset)
{
    if (dev_ptr == nullptr) return GS_ERR_INVALID_ARG;
    if (cudaIpcCloseMemHandle(static_cast<unsigned char*>(dev_ptr) - offset) != cudaSuccess) { cudaGetLastError(); return GS_ERR_CUDA; }
    return GS_OK;
}

// P(i,j) = sum_l f_l conj(C(i,l)) C(j,l) = (X^H X)(i,j) with X(l,i) = sqrt(f_l) C(i,l): one transpose-and-scale
// pass into the workspace, then a SYRK / HERK of k-extent nev on the tile engine (upper tiles only).
gs_status_t gs_density_matrix(gs_plan_t* plan, const void* C_, const double* f, void* P_, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (P_ == nullptr || !aligned16(P_)) return GS_ERR_INVALID_ARG;
    const int N = int(plan->N), nev = int(plan->nev);
    if (nev > 0 && (C_ == nullptr || f == nullptr || !aligned16(C_) || overlaps(P_, mat_bytes(plan), C_, vec_bytes(plan))))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Stage st = make_stage(plan, stream);
    void* X = big_ptr(plan);
    const long long ldx = nev == 0 ? 2 : (plan->z ? nev : ((nev + 1) & ~1LL));   // real: even pitch so that TMA applies
    if (nev > 0) {
        dim3 grid((N + 31) / 32, (nev + 31) / 32), block(32, 8);
        LaunchTimer timer(plan, L_DENS_T, stream);
        if (plan->z)
            transpose_scale_kernel<double2><<<grid, block, 0, stream>>>(static_cast<const double2*>(C_), plan->N, f,
                                                                       static_cast<double2*>(X), ldx, N, nev, info_ptr(plan));
        else
            transpose_scale_kernel<double><<<grid, block, 0, stream>>>(static_cast<const double*>(C_), plan->N, f,
                                                                     static_cast<double*>(X), ldx, N, nev, info_ptr(plan));
        GS_CUDA(plan, cudaGetLastError());
        plan->launches += 1;
    }
    // nev == 0: an empty k-range stores zeros; the operand view only has to be a valid tensor
    const MatView vX{X, nev > 0 ? nev : 1, N, ldx};
    st.tma = true;   // X has a 16-byte-multiple pitch by construction, also for odd N
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vX, false) || !set_operand(st, p, 1, vX, false)) return GS_ERR_CUDA;
    p.C = static_cast<double*>(P_); p.ldc = N;
    p.tiles_m = plan->nblk; p.tiles_n = plan->nblk; p.order = ORDER_TRI_ROW_DESC;
    p.c_rows = N; p.c_cols = N;
    p.khi_c = (nev + st.bk - 1) / st.bk; p.kmax = p.khi_c;
    p.flags = F_STORE_UPPER | F_REAL_DIAG;
    return launch(st, p, false, L_DENS_SYRK);
}

gs_status_t gs_cholesky_sharded_epochs(const gs_plan_t* plan, uint32_t* count)
{
    if (plan == nullptr || count == nullptr) return GS_ERR_INVALID_ARG;
    const int nbp = plan->potrf_nb < plan->nblk ? plan->potrf_nb : plan->nblk;
    *count = 2u * uint32_t((plan->nblk + nbp - 1) / nbp) + 1u;
    return GS_OK;
}

gs_status_t gs_cholesky_sharded(gs_plan_t* plan, void* S_inout, int rank, int nranks, void* const* peer_S, void* const* peer_workspace,
                                void* const* flags, uint32_t epoch0, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (S_inout == nullptr || !aligned16(S_inout) || nranks < 1 || nranks > kMaxPeers || rank < 0 || rank >= nranks) return GS_ERR_INVALID_ARG;
    if (nranks > 1) {
        if (peer_S == nullptr || peer_workspace == nullptr || flags == nullptr) return GS_ERR_INVALID_ARG;
        for (int s = 0; s < nranks; ++s) {
            if (peer_S[s] == nullptr || !aligned16(peer_S[s]) || peer_workspace[s] == nullptr || (reinterpret_cast<uintptr_t>(peer_workspace[s]) & 255u) != 0 ||
                flags[s] == nullptr || (reinterpret_cast<uintptr_t>(flags[s]) & 3u) != 0)
                return GS_ERR_INVALID_ARG;
        }
        if (peer_S[rank] != S_inout || peer_workspace[rank] != plan->ws) return GS_ERR_INVALID_ARG;
    }
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(configure_leaf(plan));
    // Every kernel of the call is loaded BEFORE the first wait is enqueued: with lazy module loading the first launch of
    // a kernel may synchronise with the device, and a stream that sits in a wait for a rank whose work this very host
    // thread has yet to enqueue would never let it return.
    {
        static PerDeviceOnce once;
        const cudaError_t pe = once.run([]() -> cudaError_t {
            cudaError_t r = engine_configure();
            cudaFuncAttributes fa;
            if (r == cudaSuccess) r = cudaFuncGetAttributes(&fa, copy_block_push_kernel<double>);
            if (r == cudaSuccess) r = cudaFuncGetAttributes(&fa, copy_block_push_kernel<double2>);
            if (r == cudaSuccess) r = cudaFuncGetAttributes(&fa, zero_lower_blocks_kernel<double, LB>);
            if (r == cudaSuccess) r = cudaFuncGetAttributes(&fa, zero_lower_blocks_kernel<double2, CLB>);
            return r;
        });
        if (pe != cudaSuccess) return cuda_fail(plan, pe);
    }
    GS_CUDA(plan, cudaMemsetAsync(info_ptr(plan), 0, sizeof(int), stream));
    Potrf f;
    f.st = make_stage(plan, stream);
    f.S = S_inout;
    f.vS = MatView{S_inout, plan->N, plan->N, plan->N};
    f.vT = MatView{big_ptr(plan), plan->N, plan->N, plan->N};
    f.pb = 0;
    void* self_S[1] = {S_inout};
    void* self_ws[1] = {plan->ws};
    void* self_flags[1] = {plan->ws};     // (never used with one rank)
    ShardedChol sh{rank, nranks, nranks > 1 ? peer_S : self_S, nranks > 1 ? peer_workspace : self_ws, nranks > 1 ? flags : self_flags, epoch0};
    return factor_sharded(f, sh, stream);
}

// ------------------------------------------------------------------------------------------------
// gs_density_matrix_static: the same two launches with their scratch (the status flag and the scaled,
// transposed eigenvector block X) in a file-scope device array instead of the caller's workspace, for callers
// that cannot allocate device memory (CUDA graph capture, serving loops).  The array's name is a host-side
// stand-in in host code: its device address comes from cudaGetSymbolAddress, looked up once per device with
// that device current.  Every call shares the array: calls that overlap on the GPU race (include/gs.h).
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[GS_STATIC_SCRATCH_BYTES];

static cudaError_t static_scratch_address(unsigned char** out)
{
    static std::mutex mu;
    static unsigned char* addr[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (addr[dev] == nullptr) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr || (reinterpret_cast<uintptr_t>(p) & 255u) != 0) return cudaErrorInvalidSymbol;
        addr[dev] = static_cast<unsigned char*>(p);
    }
    *out = addr[dev];
    return cudaSuccess;
}

gs_status_t gs_density_matrix_static(gs_plan_t* plan, const void* C_, const double* f, void* P_, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;   // the plan's own workspace is not used: none has to be set
    if (P_ == nullptr || !aligned16(P_)) return GS_ERR_INVALID_ARG;
    const int N = int(plan->N), nev = int(plan->nev);
    if (nev > 0 && (C_ == nullptr || f == nullptr || !aligned16(C_) || overlaps(P_, mat_bytes(plan), C_, vec_bytes(plan))))
        return GS_ERR_INVALID_ARG;
    const long long ldx = nev == 0 ? 2 : (plan->z ? nev : ((nev + 1) & ~1LL));   // as in gs_density_matrix
    const size_t need = kInfoBytes + size_t(N) * size_t(ldx) * plan->es;
    if (need > size_t(GS_STATIC_SCRATCH_BYTES)) {
        std::snprintf(plan->cuda_error, sizeof(plan->cuda_error),
                      "gs_density_matrix_static: N = %d, nev = %d needs %zu bytes of scratch, the static array holds %zu "
                      "(GS_STATIC_SCRATCH_BYTES); use gs_density_matrix with a workspace", N, nev, need, size_t(GS_STATIC_SCRATCH_BYTES));
        return GS_ERR_WORKSPACE;
    }
    unsigned char* scratch = nullptr;
    GS_CUDA(plan, static_scratch_address(&scratch));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    // the array keeps the previous call's contents: the status flag the kernels test must start at zero
    // (X is overwritten in full before it is read: rows l < nev by the transpose, TMA zero-fills the ragged k tail)
    int* info = reinterpret_cast<int*>(scratch);
    GS_CUDA(plan, cudaMemsetAsync(info, 0, kInfoBytes, stream));
    void* X = scratch + kInfoBytes;
    Stage st = make_stage(plan, stream);
    if (nev > 0) {
        dim3 grid((N + 31) / 32, (nev + 31) / 32), block(32, 8);
        LaunchTimer timer(plan, L_DENS_T, stream);
        if (plan->z)
            transpose_scale_kernel<double2><<<grid, block, 0, stream>>>(static_cast<const double2*>(C_), plan->N, f,
                                                                       static_cast<double2*>(X), ldx, N, nev, info);
        else
            transpose_scale_kernel<double><<<grid, block, 0, stream>>>(static_cast<const double*>(C_), plan->N, f,
                                                                     static_cast<double*>(X), ldx, N, nev, info);
        GS_CUDA(plan, cudaGetLastError());
        plan->launches += 1;
    }
    const MatView vX{X, nev > 0 ? nev : 1, N, ldx};
    st.tma = true;
    EngineParams p = blank_params(plan);
    p.info = info;
    if (!set_operand(st, p, 0, vX, false) || !set_operand(st, p, 1, vX, false)) return GS_ERR_CUDA;
    p.C = static_cast<double*>(P_); p.ldc = N;
    p.tiles_m = plan->nblk; p.tiles_n = plan->nblk; p.order = ORDER_TRI_ROW_DESC;
    p.c_rows = N; p.c_cols = N;
    p.khi_c = (nev + st.bk - 1) / st.bk; p.kmax = p.khi_c;
    p.flags = F_STORE_UPPER | F_REAL_DIAG;
    return launch(st, p, false, L_DENS_SYRK);
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
    if (h <= -(1 << 30)) { *info = 0; return GS_ERR_NO_CONVERGENCE; }   // the tridiagonal eigensolver gave up (evp_dc.cuh)
    if (h < 0) { *info = -int64_t(h); return GS_ERR_SINGULAR; }
    return GS_OK;
}

gs_status_t gs_plan_clear_info(gs_plan_t* plan, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    if (plan->ws == nullptr) return GS_ERR_WORKSPACE;
    GS_CUDA(plan, cudaMemsetAsync(info_ptr(plan), 0, sizeof(int), static_cast<cudaStream_t>(cuda_stream)));
    return GS_OK;
}

gs_status_t gs_reduce_host_scratch_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    const size_t mat = ((size_t(plan->N) * size_t(plan->N) * plan->es + 255) / 256) * 256;
    *bytes = 4 * mat;   // S->U, H (later C~ and C), Uinv, Htilde
    return GS_OK;
}

// Row ranges (in blocks) of about equal work for the split SYR2K launch of the host path: row I of the
// triangle costs (I + 1)(n - I) tile-steps.
static std::vector<int> host_row_splits(const gs_plan* plan)
{
    const int n = plan->nblk, parts = n >= 16 ? 4 : 1;
    std::vector<int> s{0};
    double total = 0.0;
    for (int I = 0; I < n; ++I) total += double(I + 1) * double(n - I);
    double acc = 0.0;
    for (int I = 0; I < n; ++I) {
        acc += double(I + 1) * double(n - I);
        if (int(s.size()) < parts && acc >= total * double(s.size()) / parts) s.push_back(I + 1);
    }
    if (s.back() != n) s.push_back(n);
    // the copy of the last range is the one left exposed: keep halving that range until it is a few block
    // rows (its trapezoid is then a few MB)
    if (parts > 1) {
        s.pop_back();
        while (n - s.back() > 8) s.push_back(s.back() + (n - s.back() + 1) / 2);
        s.push_back(n);
    }
    return s;
}

gs_status_t gs_reduce_host_d2h_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    const std::vector<int> sp = host_row_splits(plan);
    size_t b = 0;
    for (size_t r = 0; r + 1 < sp.size(); ++r) {
        const int64_t r0 = int64_t(sp[r]) * plan->lb, r1 = std::min<int64_t>(int64_t(sp[r + 1]) * plan->lb, plan->N);
        b += size_t(r1 - r0) * size_t(plan->N - r0) * plan->es;
    }
    *bytes = b;
    return GS_OK;
}

// Host -> device copy of one triangle (diagonal included) of an N x N column-major matrix in column
// chunks: chunk [c0, c1) moves rows [0, c1) (upper) or [c0, N) (lower) of its columns.
constexpr int64_t kTriangleChunkCols = 512;

static size_t triangle_h2d_bytes(const gs_plan* plan)
{
    size_t b = 0;
    for (int64_t c0 = 0; c0 < plan->N; c0 += kTriangleChunkCols) {
        const int64_t c1 = std::min<int64_t>(c0 + kTriangleChunkCols, plan->N);
        b += size_t(c1) * size_t(c1 - c0) * plan->es;   // the lower trapezoids have the same sizes, mirrored
    }
    return b;
}

// Upload of S's upper triangle in the order step 1 consumes it.  Nothing strictly below a diagonal block is
// written, so the copies may run beside gs_cholesky's zeroing of the strictly-lower blocks.
//   top part: rows [0, top) of every block column (chunk [c0, c1) moves rows [0, min(top, c1)));
//   slab [R0, R1) (block rows, below the top part): for each of its block columns b the rows from the slab
//   start to the end of the diagonal block, then the rectangle right of the slab's diagonal square.
static gs_status_t copy_2d_h2d(gs_plan* plan, void* dev, const void* host, int64_t r0, int64_t r1, int64_t c0, int64_t c1, cudaStream_t stream)
{
    if (r1 <= r0 || c1 <= c0) return GS_OK;
    const size_t pitch = size_t(plan->N) * plan->es;
    const size_t off = size_t(r0) * plan->es + size_t(c0) * pitch;
    GS_CUDA(plan, cudaMemcpy2DAsync(static_cast<unsigned char*>(dev) + off, pitch, static_cast<const unsigned char*>(host) + off, pitch,
                                    size_t(r1 - r0) * plan->es, size_t(c1 - c0), cudaMemcpyHostToDevice, stream));
    return GS_OK;
}

static gs_status_t copy_upper_top_h2d(gs_plan* plan, void* dev, const void* host, int64_t top, cudaStream_t stream)
{
    for (int64_t c0 = 0; c0 < plan->N; c0 += plan->lb) {
        const int64_t c1 = std::min<int64_t>(c0 + plan->lb, plan->N);
        GS_TRY(copy_2d_h2d(plan, dev, host, 0, std::min<int64_t>(top, c1), c0, c1, stream));
        if (c1 >= top) {   // from here on every block column has the same rows: one copy for the rest
            GS_TRY(copy_2d_h2d(plan, dev, host, 0, top, c1, plan->N, stream));
            break;
        }
    }
    return GS_OK;
}

static gs_status_t copy_upper_slab_h2d(gs_plan* plan, void* dev, const void* host, int R0, int R1, cudaStream_t stream)
{
    const int64_t lb = plan->lb, N = plan->N;
    const int64_t r0 = R0 * lb, r1 = std::min<int64_t>(R1 * lb, N);
    for (int b = R0; b < R1; ++b)
        GS_TRY(copy_2d_h2d(plan, dev, host, r0, std::min<int64_t>((b + 1) * lb, N), b * lb, std::min<int64_t>((b + 1) * lb, N), stream));
    return copy_2d_h2d(plan, dev, host, r0, r1, r1, N, stream);
}

static size_t upper_h2d_bytes(const gs_plan* plan)
{
    size_t b = 0;
    for (int64_t c0 = 0; c0 < plan->N; c0 += plan->lb) {
        const int64_t c1 = std::min<int64_t>(c0 + plan->lb, plan->N);
        b += size_t(c1) * size_t(c1 - c0) * plan->es;
    }
    return b;
}

static gs_status_t copy_triangle_h2d(gs_plan* plan, void* dev, const void* host, bool upper, cudaStream_t stream)
{
    const size_t pitch = size_t(plan->N) * plan->es;
    for (int64_t c0 = 0; c0 < plan->N; c0 += kTriangleChunkCols) {
        const int64_t c1 = std::min<int64_t>(c0 + kTriangleChunkCols, plan->N);
        const int64_t r0 = upper ? 0 : c0, r1 = upper ? c1 : plan->N;
        const size_t off = size_t(r0) * plan->es + size_t(c0) * pitch;
        GS_CUDA(plan, cudaMemcpy2DAsync(static_cast<unsigned char*>(dev) + off, pitch, static_cast<const unsigned char*>(host) + off, pitch,
                                        size_t(r1 - r0) * plan->es, size_t(c1 - c0), cudaMemcpyHostToDevice, stream));
    }
    return GS_OK;
}

gs_status_t gs_reduce_host_h2d_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    *bytes = upper_h2d_bytes(plan) + triangle_h2d_bytes(plan);   // S upper (block columns) + H lower (512-column chunks)
    return GS_OK;
}

static gs_status_t ensure_copy_streams(gs_plan* plan, size_t events)
{
    if (plan->copy == nullptr) {
        GS_CUDA(plan, cudaStreamCreateWithFlags(&plan->copy, cudaStreamNonBlocking));
        GS_CUDA(plan, cudaStreamCreateWithFlags(&plan->copy_out, cudaStreamNonBlocking));
        GS_CUDA(plan, cudaEventCreateWithFlags(&plan->ev_copy, cudaEventDisableTiming));
    }
    while (plan->ev_pool.size() < events) {
        cudaEvent_t e;
        GS_CUDA(plan, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        plan->ev_pool.push_back(e);
    }
    return GS_OK;
}

gs_status_t gs_reduce_host(gs_plan_t* plan, const void* host_H, const void* host_S, void* host_U, void* host_Uinv,
                           void* host_Htilde, void* dev_scratch, size_t scratch_bytes, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    size_t need = 0;
    gs_reduce_host_scratch_bytes(plan, &need);
    if (dev_scratch == nullptr || scratch_bytes < need || (reinterpret_cast<uintptr_t>(dev_scratch) & 255u) != 0) return GS_ERR_WORKSPACE;
    if (host_H == nullptr || host_S == nullptr || host_Htilde == nullptr) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t bytes = size_t(plan->N) * size_t(plan->N) * plan->es;
    const size_t mat = need / 4;
    unsigned char* base = static_cast<unsigned char*>(dev_scratch);
    void *dS = base, *dH = base + mat, *dV = base + 2 * mat, *dHt = base + 3 * mat;
    RowRanges rr;
    rr.splits = host_row_splits(plan);
    const size_t nr = rr.splits.size();
    // Only the triangles the steps reference cross the link: the upper one of S (step 1) and the lower one
    // of H (step 3) -- about half of each matrix; what stays unwritten in the scratch is never read.  All
    // uploads go, one after the other, on the plan's copy stream (forked from / joined into `stream`):
    //   1. the rows of S's triangle that the first two panels cover -- step 1 starts when they are in;
    //   2. the rest of S in slabs of eight block rows -- needed from the first trailing update on, which is
    //      applied slab by slab as they arrive (plan->gates), behind the first panel's factorisation, solve
    //      and row update;
    //   3. H, not needed before step 3, beside steps 1-2.
    const std::vector<int> ps = Potrf::panel_starts(plan->nblk, plan);
    const int top_blk = ps.size() > 2 ? ps[2] : plan->nblk;
    const int64_t top = std::min<int64_t>(int64_t(top_blk) * plan->lb, plan->N);
    const int slab = 8;
    const size_t nslabs = size_t((plan->nblk - top_blk + slab - 1) / slab);
    GS_TRY(ensure_copy_streams(plan, nr + 1 + nslabs));
    cudaEvent_t ev_top = plan->ev_pool[nr];
    GS_CUDA(plan, cudaEventRecord(plan->ev_copy, stream));
    GS_CUDA(plan, cudaStreamWaitEvent(plan->copy, plan->ev_copy, 0));
    GS_CUDA(plan, cudaStreamWaitEvent(plan->copy_out, plan->ev_copy, 0));
    GS_TRY(copy_upper_top_h2d(plan, dS, host_S, top, plan->copy));
    GS_CUDA(plan, cudaEventRecord(ev_top, plan->copy));
    GS_CUDA(plan, cudaStreamWaitEvent(stream, ev_top, 0));
    plan->gates.clear();
    for (size_t q = 0; q < nslabs; ++q) {
        const int R0 = top_blk + int(q) * slab, R1 = std::min(R0 + slab, plan->nblk);
        const gs_status_t cs = copy_upper_slab_h2d(plan, dS, host_S, R0, R1, plan->copy);
        if (cs != GS_OK) { plan->gates.clear(); return cs; }
        const cudaError_t ce = cudaEventRecord(plan->ev_pool[nr + 1 + q], plan->copy);
        if (ce != cudaSuccess) { plan->gates.clear(); return cuda_fail(plan, ce); }
        plan->gates.emplace_back(R0, plan->ev_pool[nr + 1 + q]);
    }
    gs_status_t rc = copy_triangle_h2d(plan, dH, host_H, false, plan->copy);
    if (rc == GS_OK && cudaEventRecord(plan->ev_copy, plan->copy) != cudaSuccess) rc = GS_ERR_CUDA;
    if (rc == GS_OK) rc = gs_cholesky(plan, dS, stream);
    plan->gates.clear();
    if (rc == GS_OK) rc = gs_invert_triangular(plan, dS, dV, stream);
    GS_CUDA(plan, cudaStreamWaitEvent(stream, plan->ev_copy, 0));   // join, also on failure
    GS_TRY(rc);
    if (host_U || host_Uinv) {   // U, U^-1 are final once steps 1-2 are done: they go back beside step 3
        GS_CUDA(plan, cudaEventRecord(plan->ev_pool[nr - 1], stream));
        GS_CUDA(plan, cudaStreamWaitEvent(plan->copy_out, plan->ev_pool[nr - 1], 0));
        if (host_U) GS_CUDA(plan, cudaMemcpyAsync(host_U, dS, bytes, cudaMemcpyDeviceToHost, plan->copy_out));
        if (host_Uinv) GS_CUDA(plan, cudaMemcpyAsync(host_Uinv, dV, bytes, cudaMemcpyDeviceToHost, plan->copy_out));
    }
    // step 3 in row ranges; the finished rows of H~ (upper trapezoid of each range) go back on the D2H stream
    rr.after = [&](int r) -> gs_status_t {
        const int64_t r0 = int64_t(rr.splits[r]) * plan->lb, r1 = std::min<int64_t>(int64_t(rr.splits[r + 1]) * plan->lb, plan->N);
        const size_t off = (size_t(r0) + size_t(r0) * size_t(plan->N)) * plan->es, pitch = size_t(plan->N) * plan->es;
        GS_CUDA(plan, cudaEventRecord(plan->ev_pool[r], stream));
        GS_CUDA(plan, cudaStreamWaitEvent(plan->copy_out, plan->ev_pool[r], 0));
        GS_CUDA(plan, cudaMemcpy2DAsync(static_cast<unsigned char*>(host_Htilde) + off, pitch, static_cast<unsigned char*>(dHt) + off,
                                        pitch, size_t(r1 - r0) * plan->es, size_t(plan->N - r0), cudaMemcpyDeviceToHost, plan->copy_out));
        return GS_OK;
    };
    rc = to_standard_impl(plan, dH, dV, dHt, stream, &rr);
    GS_CUDA(plan, cudaEventRecord(plan->ev_copy, plan->copy_out));
    GS_CUDA(plan, cudaStreamWaitEvent(stream, plan->ev_copy, 0));   // join the D2H stream
    GS_TRY(rc);
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
        return GS_ERR_WORKSPACE;
    if (plan->nev == 0) return GS_OK;
    if (host_Ctilde == nullptr || host_C == nullptr) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const size_t mat = need / 4;
    unsigned char* base = static_cast<unsigned char*>(dev_scratch);
    // U^-1 was left at base + 2*mat by gs_reduce_host; C~ and C reuse the S and H slots
    unsigned char *dV = base + 2 * mat, *dCt = base, *dC = base + mat;
    // column chunks: H2D of chunk c+1, the product of chunk c and the D2H of chunk c-1 run side by side
    // the first H2D and the last D2H are the exposed ones: those two chunks are narrow (two block columns)
    const int nev = int(plan->nev), lb = plan->lb;
    const int chunk = ((nev + 3) / 4 + lb - 1) / lb * lb;
    std::vector<int> cuts{0};
    if (nev >= 16 * lb) {
        cuts.push_back(2 * lb);
        while (nev - 2 * lb - cuts.back() > chunk) cuts.push_back(cuts.back() + chunk);
        if (cuts.back() < nev - 2 * lb) cuts.push_back(nev - 2 * lb);
    }
    cuts.push_back(nev);
    const int nchunks = int(cuts.size()) - 1;
    GS_TRY(ensure_copy_streams(plan, size_t(2 * nchunks)));
    GS_CUDA(plan, cudaEventRecord(plan->ev_copy, stream));
    GS_CUDA(plan, cudaStreamWaitEvent(plan->copy, plan->ev_copy, 0));
    GS_CUDA(plan, cudaStreamWaitEvent(plan->copy_out, plan->ev_copy, 0));
    gs_status_t rc = GS_OK;
    for (int c = 0; c < nchunks && rc == GS_OK; ++c) {
        const int col0 = cuts[c], ncols = cuts[c + 1] - cuts[c];
        const size_t off = size_t(col0) * size_t(plan->N) * plan->es, cb = size_t(ncols) * size_t(plan->N) * plan->es;
        GS_CUDA(plan, cudaMemcpyAsync(dCt + off, static_cast<const unsigned char*>(host_Ctilde) + off, cb, cudaMemcpyHostToDevice, plan->copy));
        GS_CUDA(plan, cudaEventRecord(plan->ev_pool[2 * c], plan->copy));
        GS_CUDA(plan, cudaStreamWaitEvent(stream, plan->ev_pool[2 * c], 0));
        rc = backtransform_cols(plan, dV, dCt, dC, col0, ncols, stream);
        GS_CUDA(plan, cudaEventRecord(plan->ev_pool[2 * c + 1], stream));
        GS_CUDA(plan, cudaStreamWaitEvent(plan->copy_out, plan->ev_pool[2 * c + 1], 0));
        GS_CUDA(plan, cudaMemcpyAsync(static_cast<unsigned char*>(host_C) + off, dC + off, cb, cudaMemcpyDeviceToHost, plan->copy_out));
    }
    GS_CUDA(plan, cudaEventRecord(plan->ev_copy, plan->copy_out));
    GS_CUDA(plan, cudaStreamWaitEvent(stream, plan->ev_copy, 0));   // join (the H2D stream was joined chunk by chunk)
    GS_TRY(rc);
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

gs_status_t gs_plan_launch_trace(gs_plan_t* plan, gs_launch_trace_t* out, int cap, int* count)
{
    if (plan == nullptr || count == nullptr || (out == nullptr && cap > 0)) return GS_ERR_INVALID_ARG;
    const int n = int(plan->timed.size());
    for (int i = 0; i < n && i < cap; ++i) {
        const TimedLaunch& t = plan->timed[i];
        float a = 0.f, b = 0.f;
        cudaError_t e = cudaEventElapsedTime(&a, plan->timed[0].e0, t.e0);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&b, plan->timed[0].e0, t.e1);
        if (e != cudaSuccess) return cuda_fail(plan, e);
        std::snprintf(out[i].label, sizeof(out[i].label), "%s", kLabelNames[t.label]);
        out[i].side_stream = t.side;
        out[i].t0_ms = a;
        out[i].t1_ms = b;
    }
    *count = n;
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
        case GS_ERR_NO_CONVERGENCE: return "GS_ERR_NO_CONVERGENCE";
    }
    return "GS_ERR_UNKNOWN";
}

const char* gs_plan_last_cuda_error(const gs_plan_t* plan) { return plan != nullptr ? plan->cuda_error : ""; }

}  // extern "C"

#include "evp_host.cuh"
