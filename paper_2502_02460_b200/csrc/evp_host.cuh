// evp_host.cuh -- host drivers of NEXT-4, the standard eigenproblem  H~ C~ = C~ eps  between step 3 and the
// back-transformation, in the three stages of the paper's Table 1:
//   gs_evp_tridiagonalize  "Tridiag."  one-stage Householder reduction H~ = Q T Q^H     (evp_tridiag.cuh)
//   gs_evp_tridiag_solve   "Solve"     divide and conquer on T, lowest nev pairs        (evp_dc.cuh)
//   gs_evp_backtransform   "Back"      C~ = Q Z, blocked reflectors on the tile engine
// Included by gs.cu (same translation unit: it uses the plan, Stage and launch() defined there).
#pragma once

#include "evp_dc.cuh"
#include "evp_tridiag.cuh"

namespace {

using namespace gs::evp;

// ---- workspace carving (the same walk computes the size and the pointers) ----
struct EvpLayout {
    size_t total = 0;
    unsigned char* base = nullptr;
    template <typename T>
    T* take(size_t count)
    {
        const size_t off = total;
        total += ((count * sizeof(T) + 255) / 256) * 256;
        return base != nullptr ? reinterpret_cast<T*>(base + off) : nullptr;
    }
};

constexpr int kBackSplit = 3;   // the back-transformation forms Y = Vp^H C~ (one tile row, long k) in this many k-ranges

struct EvpBuffers {
    // tridiagonalisation
    unsigned int* tickets; void* sc;
    void *u, *wp, *corr2, *tfin, *Pd, *Vt, *Wt, *Pt, *P1, *P2, *R, *Rinv, *Y, *Y2, *Ypart;
    long long ldp, ldj;
    int nb, npanels;
    // results kept for gs_standard_eigh
    double *d, *e, *dwork; void* tau; double* Z;
    // divide and conquer
    DcArrays dc;
    double* val;
    long long ldq;
};

// nev_cap: number of eigenvectors the carved buffers must hold (the plan's nev; N for the truncated-basis route,
// which needs ALL eigenvectors of S).  Everything that depends on it lies behind the R blocks, so the triangular
// factors a tridiagonalisation leaves are found again whatever nev_cap the next call carves with.
EvpBuffers evp_carve(const gs_plan* p, unsigned char* base, size_t* bytes, int64_t nev_cap)
{
    EvpLayout L;
    L.base = base;
    EvpBuffers b{};
    const size_t N = size_t(p->N), es = p->es, nev = size_t(nev_cap);
    const int nb = p->lb;
    const size_t th = p->z ? 64 : 128;
    const size_t nJ = (N + 127) / 128, nI = (N + th - 1) / th;
    b.nb = nb;
    b.npanels = int((N + nb - 1) / nb) + 1;
    b.ldp = (long long)((N + 1) & ~size_t(1));
    b.ldq = (long long)((N + 1) & ~size_t(1));
    auto takeb = [&](size_t elems) { return static_cast<void*>(L.take<unsigned char>(elems * es)); };
    b.tickets = L.take<unsigned int>(16);
    b.sc = L.take<unsigned char>(256);
    b.d = L.take<double>(N); b.e = L.take<double>(N + 1); b.dwork = L.take<double>(N); b.tau = takeb(N);
    b.u = takeb(N + 1); b.wp = takeb(N + 1); b.corr2 = takeb(N + 1); b.tfin = takeb(2 * size_t(nb)); b.Pd = takeb(N + 64);
    b.Vt = takeb(size_t(nb) * N); b.Wt = takeb(size_t(nb) * N);
    b.Pt = takeb(nJ * 2 * size_t(nb));
    b.ldj = (long long)(((nJ + 15) / 16) * 16);
    b.P1 = takeb(N * size_t(b.ldj)); b.P2 = takeb(nI * size_t(b.ldp));
    b.R = takeb(size_t(b.npanels) * nb * (nb + 1)); b.Rinv = takeb(size_t(b.npanels) * nb * (nb + 1));
    b.Y = takeb(size_t(nb) * (nev + 2)); b.Y2 = takeb(size_t(nb) * (nev + 2));
    b.Ypart = takeb(size_t(kBackSplit) * nb * (((nev + size_t(nb) - 1) / nb) * nb + 2));   // split-k partials of Y, padded to whole tiles
    b.Z = L.take<double>(N * (nev > 0 ? nev : 1));
    DcArrays& a = b.dc;
    a.ldq = b.ldq;
    a.Qcur = L.take<double>(size_t(b.ldq) * N); a.Qnew = L.take<double>(size_t(b.ldq) * N); a.G = L.take<double>(size_t(b.ldq) * N);
    a.dcur = L.take<double>(N); a.dnew = L.take<double>(N); a.dm = L.take<double>(N); a.zs = L.take<double>(N);
    a.dlam = L.take<double>(N); a.wz = L.take<double>(N); a.dval = L.take<double>(N); a.mu = L.take<double>(N); a.zhat = L.take<double>(N);
    a.rotc = L.take<double>(N); a.rots = L.take<double>(N); b.val = L.take<double>(N);
    a.idx = L.take<int>(N); a.idxnew = L.take<int>(N); a.srcm = L.take<int>(N); a.typ = L.take<int>(N); a.gsrc = L.take<int>(N);
    a.gpos = L.take<int>(N); a.gtyp = L.take<int>(N); a.dsrc = L.take<int>(N); a.dtyp = L.take<int>(N); a.org = L.take<int>(N);
    a.rota = L.take<int>(N); a.rotb = L.take<int>(N); a.rotta = L.take<int>(N); a.rottb = L.take<int>(N);
    a.desc = L.take<MergeDesc>((N + kDcLeaf - 1) / kDcLeaf + 1);
    a.info = base != nullptr ? info_ptr(p) : nullptr;
    if (bytes != nullptr) *bytes = L.total;
    return b;
}

gs_status_t evp_ready(const gs_plan* plan, EvpBuffers* b, int64_t nev_cap = -1)
{
    GS_TRY(check_ready(plan));
    if (nev_cap < 0) nev_cap = plan->nev;
    size_t need = 0;
    evp_carve(plan, nullptr, &need, nev_cap);
    if (plan->evp_ws == nullptr || plan->evp_ws_bytes < need) return GS_ERR_WORKSPACE;
    *b = evp_carve(plan, plan->evp_ws, nullptr, nev_cap);
    return GS_OK;
}

template <typename T>
StepParams<T> step_params(const gs_plan* plan, const EvpBuffers& b, void* A, double* d, double* e, void* tau)
{
    StepParams<T> p{};
    p.A = static_cast<T*>(A); p.ld = plan->N; p.N = int(plan->N); p.nb = b.nb; p.lb = b.nb;
    p.u = static_cast<T*>(b.u); p.wp = static_cast<T*>(b.wp); p.corr2 = static_cast<T*>(b.corr2);
    p.Vt = static_cast<T*>(b.Vt); p.Wt = static_cast<T*>(b.Wt);
    p.P1 = static_cast<T*>(b.P1); p.P2 = static_cast<T*>(b.P2); p.ldp = b.ldp; p.ldj = b.ldj;
    p.Pt = static_cast<T*>(b.Pt); p.tfin = static_cast<T*>(b.tfin); p.Pd = static_cast<T*>(b.Pd);
    p.sc = static_cast<StepScalars<T>*>(b.sc); p.tickets = b.tickets;
    p.d = d; p.e = e; p.tau = static_cast<T*>(tau); p.R = static_cast<T*>(b.R);
    p.info = info_ptr(plan);
    return p;
}

// GS_EVP_TRACE=1: synchronise after every launch of the eigensolver and name it on stderr (debugging aid)
inline bool evp_trace_on()
{
    static const bool on = std::getenv("GS_EVP_TRACE") != nullptr;
    return on;
}
inline void evp_trace(cudaStream_t stream, const char* what, int a = 0, int b = 0)
{
    if (!evp_trace_on()) return;
    const cudaError_t e = cudaStreamSynchronize(stream);
    std::fprintf(stderr, "[evp] %s %d %d -> %s\n", what, a, b, cudaGetErrorString(e));
    std::fflush(stderr);
}

// step kernels: programmatic dependent launch unless GS_EVP_PDL=0
template <typename... KArgs, typename... Args>
inline cudaError_t evp_launch(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args)
{
    static const bool pdl = !(std::getenv("GS_EVP_PDL") != nullptr && std::atoi(std::getenv("GS_EVP_PDL")) == 0);
    if (pdl) return launch_pdl(kernel, grid, block, 0, stream, args...);
    kernel<<<grid, block, 0, stream>>>(KArgs(args)...);
    return cudaGetLastError();
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl_smem(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    static const bool pdl = !(std::getenv("GS_EVP_PDL") != nullptr && std::atoi(std::getenv("GS_EVP_PDL")) == 0);
    if (pdl) return launch_pdl(kernel, grid, block, smem, stream, args...);
    kernel<<<grid, block, smem, stream>>>(KArgs(args)...);
    return cudaGetLastError();
}

#define GS_LAUNCH_OK(plan)                                       \
    do {                                                         \
        const cudaError_t le__ = cudaGetLastError();             \
        if (le__ != cudaSuccess) return cuda_fail((plan), le__); \
        (plan)->launches += 1;                                   \
    } while (0)

// tensor map of symv_tma_kernel: A as an (N * w8) x N FP64 tensor, box = 128 doubles (TH rows) x 16 columns, no swizzle
inline bool make_symv_map(CUtensorMap* out, const void* A, long long N, int w8)
{
    PFN_cuTensorMapEncodeTiled enc = tensor_map_encoder();
    if (enc == nullptr) return false;
    cuuint64_t dims[2] = {static_cast<cuuint64_t>(N) * w8, static_cast<cuuint64_t>(N)};
    cuuint64_t strides[1] = {static_cast<cuuint64_t>(N) * 8 * w8};
    cuuint32_t box[2] = {128, 16};
    cuuint32_t estr[2] = {1, 1};
    return enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(A), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// per-device opt-in of symv_tma_kernel to its dynamic shared memory; *sms = SM count of the current device
inline cudaError_t configure_symv(int* sms)
{
    static PerDeviceOnce once;
    cudaError_t e = once.run([]() -> cudaError_t {
        cudaError_t r = cudaFuncSetAttribute(symv_tma_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, SvCfg<double>::kSmemBytes);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(symv_tma_kernel<double2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SvCfg<double2>::kSmemBytes);
        // two CTAs of the real kernel share an SM only if the whole shared-memory carve-out is granted
        if (r == cudaSuccess) r = cudaFuncSetAttribute(symv_tma_kernel<double>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        if (r == cudaSuccess) r = cudaFuncSetAttribute(symv_tma_kernel<double2>, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
        return r;
    });
    if (e != cudaSuccess) return e;
    int dev = 0;
    e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    return cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev);
}

// A[0:m, 0:m] -= V W^H + W V^H (upper tiles) from the panel's conjugate-transposed images Vt, Wt (cnt x m, ld nb)
gs_status_t evp_her2k(gs_plan* plan, const EvpBuffers& b, void* A, int m, int cnt, cudaStream_t stream)
{
    Stage st = make_stage(plan, stream);
    st.tma = true;                       // the operands are the panels (even pitch by construction), also for odd N
    const MatView vV{b.Vt, cnt, m, b.nb}, vW{b.Wt, cnt, m, b.nb};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vV, false) || !set_operand(st, p, 1, vW, false) || !set_operand(st, p, 2, vW, false) ||
        !set_operand(st, p, 3, vV, false))
        return GS_ERR_CUDA;
    p.C = static_cast<double*>(A); p.ldc = plan->N;
    p.tiles_m = (m + st.lb - 1) / st.lb; p.tiles_n = p.tiles_m; p.order = ORDER_TRI_ROW_DESC;
    p.c_rows = m; p.c_cols = m;
    p.khi_c = (cnt + st.bk - 1) / st.bk; p.kmax = p.khi_c;
    p.alpha = -1.0; p.beta = 1.0;
    p.flags = F_DUAL | F_STORE_UPPER | F_REAL_DIAG;
    return launch(st, p, false, L_EVP_HER2K);
}

template <typename T>
gs_status_t evp_tridiagonalize_t(gs_plan* plan, const EvpBuffers& b, void* A, double* d, double* e, void* tau, cudaStream_t stream)
{
    constexpr int TH = SymvGeom<T>::TH, TW = kSymvTW;
    const int N = int(plan->N), nb = b.nb;
    GS_CUDA(plan, cudaMemsetAsync(b.tickets, 0, 16 * sizeof(unsigned int), stream));
    GS_CUDA(plan, cudaMemsetAsync(b.sc, 0, 256, stream));
    init_r_kernel<T><<<64, 256, 0, stream>>>(static_cast<T*>(b.R), nb, b.npanels);
    GS_LAUNCH_OK(plan);
    StepParams<T> p = step_params<T>(plan, b, A, d, e, tau);
    const bool vec = (N % 2 == 0);
    // S through TMA (symv_tma_kernel) whenever A admits a tensor map; GS_EVP_SYMV=0 keeps the plain-load kernel,
    // GS_EVP_CHUNK fixes the strip length (128-row blocks per work item: 1, 2 or 4)
    static const bool tma_off = std::getenv("GS_EVP_SYMV") != nullptr && std::atoi(std::getenv("GS_EVP_SYMV")) == 0;
    static const int chunk_env = std::getenv("GS_EVP_CHUNK") != nullptr ? std::atoi(std::getenv("GS_EVP_CHUNK")) : 0;
    static const int chunk_t = std::getenv("GS_EVP_CHUNK_T") != nullptr ? std::atoi(std::getenv("GS_EVP_CHUNK_T")) : 4;
    static const int comb_env = std::getenv("GS_EVP_COMBINE_THREADS") != nullptr ? std::atoi(std::getenv("GS_EVP_COMBINE_THREADS")) : 0;
    int comb_threads = comb_env;
    if (comb_threads <= 0) {
        int dev = 0, sms = 0;
        GS_CUDA(plan, cudaGetDevice(&dev));
        GS_CUDA(plan, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        comb_threads = sms * (plan->z ? 2 : 3) * 256;      // one wave of C: three CTAs per SM at the real kernel's register count, two at the complex one's
    }
    // L2 policy of the streamed tiles: 0 plain, 1 evict-first always, 2 evict-first while the triangle exceeds evict_bytes
    static const int evict_mode = std::getenv("GS_EVP_EVICT") != nullptr ? std::atoi(std::getenv("GS_EVP_EVICT")) : 2;
    static const double evict_bytes = std::getenv("GS_EVP_EVICT_MB") != nullptr ? 1e6 * std::atof(std::getenv("GS_EVP_EVICT_MB")) : 100e6;
    // ... except the tiles of the leading column blocks (27 MB: the same tiles in every column of the reduction), which stay
    // in the L2 from column to column with the plain policy: real 20 blocks, complex 14
    static const int keep_env = std::getenv("GS_EVP_KEEP") != nullptr ? std::atoi(std::getenv("GS_EVP_KEEP")) : -1;
    const int keep_blocks = keep_env >= 0 ? keep_env : (sizeof(T) == 8 ? 20 : 14);
    static const bool fuse_off = std::getenv("GS_EVP_FUSE") != nullptr && std::atoi(std::getenv("GS_EVP_FUSE")) == 0;
    const bool use_tma = !tma_off && (sizeof(T) == 16 || vec) && aligned16(A);
    SymvTmaParams<T> q{};
    int sv_ctas = 0;
    if (use_tma) {
        int sms = 0;
        GS_CUDA(plan, configure_symv(&sms));
        static const int ctas_env = std::getenv("GS_EVP_CTAS") != nullptr ? std::atoi(std::getenv("GS_EVP_CTAS")) : 0;
        sv_ctas = sms * (ctas_env > 0 ? ctas_env : SvCfg<T>::kCtasPerSm);
        if (!make_symv_map(&q.mapA, A, N, int(sizeof(T) / 8))) return GS_ERR_CUDA;
    }
    const int fgrid = std::max(1, std::min(64, (N + 255) / 256));
    auto finish = [&](int i, int jp, int mode) -> gs_status_t {
        p.i = i; p.jp = jp; p.mode = mode;
        LaunchTimer timer(plan, L_EVP_STEP, stream);
        const cudaError_t le = evp_launch(finish_kernel<T>, fgrid, 256, stream, p);
        if (le != cudaSuccess) return cuda_fail(plan, le);
        plan->launches += 1;
        evp_trace(stream, "finish", i, mode);
        return GS_OK;
    };
    GS_TRY(finish(N, 0, 1));                      // fresh load of column N-1
    int i = N - 1, panel = 0;
    while (i >= 1) {
        const int itop = i;
        int jp = 0;
        p.itop = itop; p.panel = panel;
        while (i >= 1 && jp < nb) {
            // TMA form: the F of the previous column (w, the next u, its norm and scalars) is formed inside this S
            p.i = i; p.jp = jp; p.mode = 0; p.fuse = (use_tma && !fuse_off && jp > 0) ? 1 : 0;
            const int nJ = (i + TW - 1) / TW, nI = (i + TH - 1) / TH;
            if (use_tma) {
                const int K = chunk_env == 1 || chunk_env == 2 || chunk_env == 4 || chunk_env == 8 ? chunk_env : sv_chunk_blocks(nJ, chunk_t * sv_ctas);
                const int nitems = sv_items_before(nJ, K);
                p.p2_chunk_rows = K * TW;
                q.s = p; q.chunk_blocks = K; q.dot_ctas = jp > 0 ? nJ : 0;
                q.keep_blocks = keep_blocks;
                q.evict_first = evict_mode == 1 || (evict_mode == 2 && (double)i * i * 4.0 * (sizeof(T) / 8) > evict_bytes) ? 1 : 0;
                const int stream_ctas = std::min(nitems, sv_ctas);
                LaunchTimer timer(plan, L_EVP_SYMV, stream);
                const cudaError_t le = launch_pdl_smem(symv_tma_kernel<T>, dim3(q.dot_ctas + stream_ctas), dim3(kSvThreads),
                                                       SvCfg<T>::kSmemBytes, stream, q);
                if (le != cudaSuccess) return cuda_fail(plan, le);
                plan->launches += 1;
                evp_trace(stream, "symv.tma", i, jp);
            } else {
                p.p2_chunk_rows = TH;
                LaunchTimer timer(plan, L_EVP_SYMV, stream);
                const dim3 grid(nJ, nI + (jp > 0 ? 1 : 0));
                const cudaError_t le = vec ? evp_launch(symv_kernel<T, true>, grid, kSymvThreads, stream, p)
                                           : evp_launch(symv_kernel<T, false>, grid, kSymvThreads, stream, p);
                if (le != cudaSuccess) return cuda_fail(plan, le);
                plan->launches += 1;
                evp_trace(stream, "symv", i, jp);
            }
            {
                LaunchTimer timer(plan, L_EVP_STEP, stream);
                // 16 threads per row while that is one wave of CTAs (three per SM at its register count), 8 beyond
                const bool wide = (long long)i * 16 <= (long long)comb_threads;
                const int rows_per_cta = wide ? 16 : 32;
                const cudaError_t le = wide ? evp_launch(combine_kernel<T, 16>, (i + rows_per_cta - 1) / rows_per_cta, 256, stream, p)
                                            : evp_launch(combine_kernel<T, 8>, (i + rows_per_cta - 1) / rows_per_cta, 256, stream, p);
                if (le != cudaSuccess) return cuda_fail(plan, le);
                plan->launches += 1;
                evp_trace(stream, "combine", i, jp);
            }
            const bool last = (jp == nb - 1) || (i == 1);
            if (last) GS_TRY(finish(i, jp, 2));
            else if (!(use_tma && !fuse_off)) GS_TRY(finish(i, jp, 0));
            --i; ++jp;
        }
        // the panel's rank-2 jp update of the leading (i + 1) x (i + 1) block, then the next column from the updated matrix
        GS_TRY(evp_her2k(plan, b, A, i + 1, jp, stream));
        evp_trace(stream, "her2k", i + 1, jp);
        GS_TRY(finish(i + 1, 0, 1));
        ++panel;
    }
    // T' = (D + stril(V^H V))^-1 per panel, kept as R^-1 with R = (T'^-1)^H upper triangular (one leaf launch)
    GS_TRY(configure_leaf(plan));
    const int nblocks = panel > 0 ? panel : 1;
    {
        LaunchTimer timer(plan, L_EVP_STEP, stream);
        if (plan->z)
            trtri_cleaf_kernel<<<nblocks, kCLeafThreads, kCLeafSmemBytes, stream>>>(static_cast<const double2*>(b.R), static_cast<double2*>(b.Rinv),
                                                                                   (long long)nb, nblocks * nb, info_ptr(plan));
        else
            trtri_leaf_kernel<<<nblocks, kLeafThreads, kLeafSmemBytes, stream>>>(static_cast<const double*>(b.R), static_cast<double*>(b.Rinv),
                                                                                 (long long)nb, nblocks * nb, info_ptr(plan));
        GS_LAUNCH_OK(plan);
        evp_trace(stream, "trtri_blocks", nblocks, 0);
    }
    return GS_OK;
}

// C~ = Q Z:  Q = H(N-1) ... H(1) applied panel by panel, lowest reflectors first:
//   Y = Vp^H C~[0:m, :],  Y2 = T'p Y = (Rp^-1)^H Y,  C~[0:m, :] -= Vp Y2.
gs_status_t evp_backtransform_impl(gs_plan* plan, const EvpBuffers& b, const void* A, const double* Z, long long ldz, void* Ct, int nev, cudaStream_t stream)
{
    const int N = int(plan->N), nb = b.nb;
    if (nev == 0) return GS_OK;
    {
        LaunchTimer timer(plan, L_EVP_BACK, stream);
        const dim3 grid((N + 255) / 256, std::min(nev, 4096));
        if (plan->z) widen_kernel<double2><<<grid, 256, 0, stream>>>(Z, ldz, static_cast<double2*>(Ct), plan->N, N, nev);
        else widen_kernel<double><<<grid, 256, 0, stream>>>(Z, ldz, static_cast<double*>(Ct), plan->N, N, nev);
        GS_LAUNCH_OK(plan);
        evp_trace(stream, "back.widen", N, nev);
    }
    if (N < 2) return GS_OK;
    Stage st = make_stage(plan, stream);
    const int lb = st.lb, bk = st.bk;
    static const bool back_split_off = std::getenv("GS_EVP_BACK_SPLIT") != nullptr && std::atoi(std::getenv("GS_EVP_BACK_SPLIT")) == 0;
    const int npan = (N - 1 + nb - 1) / nb;           // reflectors i = 1 .. N-1 in panels counted from the top
    const int tn = (nev + lb - 1) / lb;
    for (int pnl = npan - 1; pnl >= 0; --pnl) {
        const int itop = N - 1 - pnl * nb;
        int cnt = std::min(nb, itop);                  // reflectors itop - cnt + 1 .. itop
        int i0 = itop - cnt + 1, first = nb - cnt;
        const int m = itop;
        // a TMA box of FP64 elements must start at an even row: an odd start takes in the reflector below it, which for
        // the (only) partial panel is column 0 of the reflector matrix -- a zero vector with T' = 1, i.e. no reflector
        if (first % 2 != 0) { first -= 1; i0 -= 1; cnt += 1; }
        const MatView vA{A, m, i0 + cnt, N}, vC{Ct, m, nev, N};
        const MatView vY{b.Y, cnt, nev, nb}, vY2{b.Y2, cnt, nev, nb};
        const MatView vR{static_cast<const unsigned char*>(b.Rinv) + size_t(pnl) * nb * (nb + 1) * plan->es, nb, nb, nb};
        {   // Y = Vp^H C~: ONE row of tiles with a k-extent of m -- too few CTAs for the device, so the k-range is split
            // into kBackSplit batches (partials side by side in Ypart, summed in a fixed order by sum_parts_kernel)
            const int ksteps = (m + bk - 1) / bk;
            const int split = (back_split_off || ksteps < 8 * kBackSplit) ? 1 : kBackSplit;
            const int kc = (ksteps + split - 1) / split;
            const int ldpart = tn * lb;               // columns of one partial (whole tiles)
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vA, false) || !set_operand(st, p, 1, vC, false)) return GS_ERR_CUDA;
            p.C = static_cast<double*>(split > 1 ? b.Ypart : b.Y); p.ldc = nb;
            p.tiles_m = 1; p.tiles_n = tn; p.order = ORDER_ROW;
            p.c_rows = cnt; p.c_cols = split > 1 ? split * ldpart : nev;
            p.khi_c = kc; p.kmax = kc;
            p.a.x0 = i0;
            if (split > 1) { p.batch = split; p.c_bcol = ldpart; p.a.bk = kc * bk; p.b.bk = kc * bk; }
            GS_TRY(launch(st, p, false, L_EVP_BACK));
            evp_trace(stream, "back.y", pnl, cnt);
            if (split > 1) {
                LaunchTimer timer(plan, L_EVP_BACK, stream);
                const long long total = (long long)nb * nev;
                const int grid = int(std::min<long long>((total + 255) / 256, 4096));
                cudaError_t le;
                if (plan->z) le = launch_pdl(sum_parts_kernel<double2>, dim3(grid), dim3(256), 0, stream, static_cast<const double2*>(b.Ypart), (long long)nb * ldpart, split,
                                             static_cast<double2*>(b.Y), total, static_cast<const int*>(info_ptr(plan)));
                else le = launch_pdl(sum_parts_kernel<double>, dim3(grid), dim3(256), 0, stream, static_cast<const double*>(b.Ypart), (long long)nb * ldpart, split,
                                     static_cast<double*>(b.Y), total, static_cast<const int*>(info_ptr(plan)));
                if (le != cudaSuccess) return cuda_fail(plan, le);
                plan->launches += 1;
                evp_trace(stream, "back.ysum", pnl, split);
            }
        }
        {   // Y2 = (Rp^-1)^H Y  (the panel's block of R^-1 is upper triangular with zeros below)
            Stage s2 = st;
            s2.tma = true;
            EngineParams p = blank_params(plan);
            if (!set_operand(s2, p, 0, vR, false) || !set_operand(s2, p, 1, vY, false)) return GS_ERR_CUDA;
            p.C = static_cast<double*>(b.Y2); p.ldc = nb;
            p.tiles_m = 1; p.tiles_n = tn; p.order = ORDER_ROW;
            p.c_rows = cnt; p.c_cols = nev;
            p.khi_c = (cnt + bk - 1) / bk; p.kmax = p.khi_c;
            p.a.k0 = first; p.a.x0 = first;
            GS_TRY(launch(s2, p, false, L_EVP_BACK));
            evp_trace(stream, "back.ty", pnl, first);
        }
        {   // C~[0:m, :] -= Vp Y2
            EngineParams p = blank_params(plan);
            if (!set_operand(st, p, 0, vA, true) || !set_operand(st, p, 1, vY2, false)) return GS_ERR_CUDA;
            p.C = static_cast<double*>(Ct); p.ldc = N;
            p.tiles_m = (m + lb - 1) / lb; p.tiles_n = tn; p.order = ORDER_ROW;
            p.c_rows = m; p.c_cols = nev;
            p.khi_c = (cnt + bk - 1) / bk; p.kmax = p.khi_c;
            p.a.k0 = i0;
            p.alpha = -1.0; p.beta = 1.0;
            GS_TRY(launch(st, p, true, L_EVP_BACK));
            evp_trace(stream, "back.update", pnl, m);
        }
    }
    return GS_OK;
}

// Divide and conquer on tridiag(e, d, e): lowest nev eigenvalues -> eps, their eigenvectors -> Z (N x nev, ld ldz).
// d is modified (cut points).  Synchronises the stream once per level: the deflation counts decide the shapes of
// the launches that follow.
gs_status_t evp_solve_impl(gs_plan* plan, EvpBuffers& b, double* d, const double* e, double* eps, double* Z, long long ldz, int nev, cudaStream_t stream)
{
    const int N = int(plan->N);
    DcArrays a = b.dc;
    const int nleaf = (N + kDcLeaf - 1) / kDcLeaf;
    {
        LaunchTimer timer(plan, L_EVP_DC, stream);
        if (nleaf > 1) { dc_cut_kernel<<<(nleaf + 255) / 256, 256, 0, stream>>>(d, e, N); GS_LAUNCH_OK(plan); }
        {
            static PerDeviceOnce once;
            GS_CUDA(plan, once.run([]() -> cudaError_t {
                return cudaFuncSetAttribute(dc_leaf_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDcLeafSmemBytes);
            }));
        }
        dc_leaf_kernel<<<nleaf, kDcLeaf, kDcLeafSmemBytes, stream>>>(d, e, N, a);
        GS_LAUNCH_OK(plan);
    }
    // real engine launches, also inside a complex plan
    Stage st = make_stage(plan, stream);
    st.z = false; st.lb = LB; st.bk = BK; st.tma = true;
    std::vector<MergeDesc> hd;
    for (int span = 1; span < nleaf; span *= 2) {           // blocks of `span` leaves are solved; merge neighbours
        hd.clear();
        std::vector<std::pair<int, int>> pass;             // (off, n) of blocks without a partner
        for (int g = 0; g * span < nleaf; g += 2) {
            const int off = g * span * kDcLeaf;
            const int end1 = std::min((g + 1) * span * kDcLeaf, N);
            const int end2 = std::min((g + 2) * span * kDcLeaf, N);
            if (end2 > end1) { MergeDesc m{}; m.off = off; m.n1 = end1 - off; m.n2 = end2 - end1; hd.push_back(m); }
            else pass.emplace_back(off, end1 - off);
        }
        const int nm = int(hd.size());
        const bool top = span * 2 >= nleaf;
        int nmax = 0;
        for (const MergeDesc& m : hd) nmax = std::max(nmax, m.n1 + m.n2);
        GS_CUDA(plan, cudaMemcpyAsync(a.desc, hd.data(), sizeof(MergeDesc) * nm, cudaMemcpyHostToDevice, stream));
        {
            LaunchTimer timer(plan, L_EVP_DC, stream);
            dc_setup_kernel<<<nm, 256, 0, stream>>>(e, a); GS_LAUNCH_OK(plan);
            dc_deflate_kernel<<<nm, 256, 0, stream>>>(a); GS_LAUNCH_OK(plan);
            dc_rotate_kernel<<<dim3((nmax + 255) / 256, nm), 256, 0, stream>>>(a); GS_LAUNCH_OK(plan);
            dc_gather_kernel<<<dim3(nmax, nm), 256, 0, stream>>>(a); GS_LAUNCH_OK(plan);
            dc_secular_kernel<<<dim3((nmax + 7) / 8, nm), 256, 0, stream>>>(a); GS_LAUNCH_OK(plan);
            dc_zhat_kernel<<<dim3((nmax + 7) / 8, nm), 256, 0, stream>>>(a); GS_LAUNCH_OK(plan);
        }
        GS_CUDA(plan, cudaMemcpyAsync(hd.data(), a.desc, sizeof(MergeDesc) * nm, cudaMemcpyDeviceToHost, stream));
        GS_CUDA(plan, cudaStreamSynchronize(stream));
        for (MergeDesc& m : hd) m.r = top ? std::min(m.k, nev) : m.k;
        GS_CUDA(plan, cudaMemcpyAsync(a.desc, hd.data(), sizeof(MergeDesc) * nm, cudaMemcpyHostToDevice, stream));
        double* X = a.Qcur;                                  // the old eigenvector blocks are dead once gathered
        {
            LaunchTimer timer(plan, L_EVP_DC, stream);
            dc_xcols_kernel<<<dim3((nmax + 7) / 8, nm), 256, 0, stream>>>(a, X); GS_LAUNCH_OK(plan);
        }
        const long long ldq = a.ldq;
        for (const MergeDesc& m : hd) {
            if (m.r == 0) continue;
            const int off = m.off, n = m.n1 + m.n2;
            for (int half = 0; half < 2; ++half) {
                const int row0 = half == 0 ? off : off + m.n1, rows = half == 0 ? m.n1 : m.n2;
                // (the bottom k-range starts at an even row of X: one column of the Q1-only group, zero in these rows, may be taken in)
                const int kc0 = half == 0 ? 0 : (m.c1 & ~1), kk = half == 0 ? m.c1 + m.c2 : m.k - (m.c1 & ~1);
                const MatView vG{a.G, row0 + rows, off + kc0 + kk, ldq}, vX{X, off + kc0 + kk, off + m.r, ldq};
                EngineParams p = blank_params(plan);
                if (!set_operand(st, p, 0, vG, true) || !set_operand(st, p, 1, vX, false)) return GS_ERR_CUDA;
                p.C = a.Qnew; p.ldc = ldq;
                p.tiles_m = (rows + LB - 1) / LB; p.tiles_n = (m.r + LB - 1) / LB; p.order = ORDER_COL;
                p.c_row0 = row0; p.c_col0 = off; p.c_rows = row0 + rows; p.c_cols = off + m.r;
                p.khi_c = (kk + BK - 1) / BK; p.kmax = p.khi_c;
                p.a.x0 = row0; p.a.k0 = off + kc0;
                p.b.k0 = off + kc0; p.b.x0 = off;
                GS_TRY(launch(st, p, true, L_EVP_DC_GEMM));
            }
            (void)n;
        }
        {
            LaunchTimer timer(plan, L_EVP_DC, stream);
            dc_values_kernel<<<dim3((nmax + 255) / 256, nm), 256, 0, stream>>>(a, b.val); GS_LAUNCH_OK(plan);
            dc_rank_kernel<<<dim3((nmax + 255) / 256, nm), 256, 0, stream>>>(a, b.val); GS_LAUNCH_OK(plan);
            for (const auto& pb : pass) {
                dc_copy_block_kernel<<<pb.second, 256, 0, stream>>>(a.Qcur, a.Qnew, ldq, pb.first, pb.second); GS_LAUNCH_OK(plan);
                GS_CUDA(plan, cudaMemcpyAsync(a.dnew + pb.first, a.dcur + pb.first, sizeof(double) * pb.second, cudaMemcpyDeviceToDevice, stream));
                GS_CUDA(plan, cudaMemcpyAsync(a.idxnew + pb.first, a.idx + pb.first, sizeof(int) * pb.second, cudaMemcpyDeviceToDevice, stream));
            }
        }
        std::swap(a.Qcur, a.Qnew);
        std::swap(a.dcur, a.dnew);
        std::swap(a.idx, a.idxnew);
    }
    if (nev > 0) {
        LaunchTimer timer(plan, L_EVP_DC, stream);
        dc_output_kernel<<<nev, 256, 0, stream>>>(a.Qcur, a.ldq, a.dcur, a.idx, N, nev, eps, Z, ldz, info_ptr(plan));
        GS_LAUNCH_OK(plan);
    }
    return GS_OK;
}

// tridiagonalise, solve, back-transform: the lowest nev pairs of the upper triangle of A (destroyed)
gs_status_t evp_eigh_impl(gs_plan* plan, EvpBuffers& b, void* A, double* eps, void* Ct, int nev, cudaStream_t stream)
{
    GS_TRY(plan->z ? evp_tridiagonalize_t<double2>(plan, b, A, b.d, b.e, b.tau, stream)
                   : evp_tridiagonalize_t<double>(plan, b, A, b.d, b.e, b.tau, stream));
    GS_TRY(evp_solve_impl(plan, b, b.d, b.e, eps, b.Z, plan->N, nev, stream));
    return evp_backtransform_impl(plan, b, A, b.Z, plan->N, Ct, nev, stream);
}

}  // namespace

extern "C" {

gs_status_t gs_evp_workspace_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    evp_carve(plan, nullptr, bytes, plan->nev);
    return GS_OK;
}

gs_status_t gs_evp_set_workspace(gs_plan_t* plan, void* dev_workspace, size_t bytes)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    size_t need = 0;
    evp_carve(plan, nullptr, &need, plan->nev);
    if (dev_workspace == nullptr || bytes < need || (reinterpret_cast<uintptr_t>(dev_workspace) & 255u) != 0) return GS_ERR_WORKSPACE;
    plan->evp_ws = static_cast<unsigned char*>(dev_workspace);
    plan->evp_ws_bytes = bytes;
    return GS_OK;
}

gs_status_t gs_evp_tridiagonalize(gs_plan_t* plan, void* A_inout, double* d, double* e, void* tau, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));
    if (A_inout == nullptr || d == nullptr || e == nullptr || tau == nullptr || !aligned16(A_inout) || !aligned16(tau)) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    return plan->z ? evp_tridiagonalize_t<double2>(plan, b, A_inout, d, e, tau, stream)
                   : evp_tridiagonalize_t<double>(plan, b, A_inout, d, e, tau, stream);
}

gs_status_t gs_evp_tridiag_solve(gs_plan_t* plan, const double* d, const double* e, double* eps, double* Z, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));
    if (d == nullptr || e == nullptr || (plan->nev > 0 && (eps == nullptr || Z == nullptr))) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_CUDA(plan, cudaMemcpyAsync(b.dwork, d, sizeof(double) * size_t(plan->N), cudaMemcpyDeviceToDevice, stream));
    return evp_solve_impl(plan, b, b.dwork, e, eps, Z, plan->N, int(plan->nev), stream);
}

gs_status_t gs_evp_backtransform(gs_plan_t* plan, const void* A_reflectors, const double* Z, void* Ctilde, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));
    if (plan->nev == 0) return GS_OK;
    if (A_reflectors == nullptr || Z == nullptr || Ctilde == nullptr || !aligned16(A_reflectors) || !aligned16(Ctilde) ||
        overlaps(Ctilde, vec_bytes(plan), A_reflectors, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    return evp_backtransform_impl(plan, b, A_reflectors, Z, plan->N, Ctilde, int(plan->nev), static_cast<cudaStream_t>(cuda_stream));
}

gs_status_t gs_standard_eigh(gs_plan_t* plan, void* Htilde_inout, double* eps, void* Ctilde, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));
    if (Htilde_inout == nullptr || (plan->nev > 0 && (eps == nullptr || Ctilde == nullptr)) || !aligned16(Htilde_inout) ||
        (Ctilde != nullptr && (!aligned16(Ctilde) || overlaps(Ctilde, vec_bytes(plan), Htilde_inout, mat_bytes(plan)))))
        return GS_ERR_INVALID_ARG;
    return evp_eigh_impl(plan, b, Htilde_inout, eps, Ctilde, int(plan->nev), static_cast<cudaStream_t>(cuda_stream));
}

// Eigenvalues only: bisection on the tridiagonal matrix (evp_dc.cuh: tridiag_bisect_kernel); no eigensolver workspace needed
gs_status_t gs_evp_tridiag_eigenvalues(gs_plan_t* plan, const double* d, const double* e, int64_t count, double* eps, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (count < 0 || count > plan->N || d == nullptr || (plan->N > 1 && e == nullptr) || (count > 0 && eps == nullptr)) return GS_ERR_INVALID_ARG;
    if (count == 0) return GS_OK;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    LaunchTimer timer(plan, L_EVP_DC, stream);
    tridiag_bisect_kernel<<<unsigned((count + kBisectThreads - 1) / kBisectThreads), kBisectThreads, 0, stream>>>(d, e, int(plan->N), int(count), eps, info_ptr(plan));
    GS_LAUNCH_OK(plan);
    return GS_OK;
}

// ... of a Hermitian matrix: tridiagonalise, then bisection (H~ is destroyed as by gs_evp_tridiagonalize)
gs_status_t gs_standard_eigenvalues(gs_plan_t* plan, void* Htilde_inout, int64_t count, double* eps, void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));
    if (Htilde_inout == nullptr || !aligned16(Htilde_inout) || count < 0 || count > plan->N || (count > 0 && eps == nullptr)) return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    GS_TRY(plan->z ? evp_tridiagonalize_t<double2>(plan, b, Htilde_inout, b.d, b.e, b.tau, stream)
                   : evp_tridiagonalize_t<double>(plan, b, Htilde_inout, b.d, b.e, b.tau, stream));
    return gs_evp_tridiag_eigenvalues(plan, b.d, b.e, count, eps, cuda_stream);
}

// The whole generalized solve of PAPER.md:61-67 on one stream: steps 1-3, the standard eigensolver, the back-transformation.
gs_status_t gs_generalized_eigh(gs_plan_t* plan, const void* H, void* S_inout, void* Uinv, void* Htilde, void* Ctilde, double* eps, void* C,
                                void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b));                       // both workspaces, before anything is enqueued
    if (plan->nev > 0 && (Ctilde == nullptr || C == nullptr || eps == nullptr || overlaps(Ctilde, vec_bytes(plan), C, vec_bytes(plan))))
        return GS_ERR_INVALID_ARG;
    GS_TRY(gs_cholesky(plan, S_inout, cuda_stream));
    GS_TRY(gs_invert_triangular(plan, S_inout, Uinv, cuda_stream));
    GS_TRY(gs_to_standard(plan, H, Uinv, Htilde, cuda_stream));
    GS_TRY(gs_standard_eigh(plan, Htilde, eps, Ctilde, cuda_stream));
    return gs_backtransform(plan, Uinv, Ctilde, C, cuda_stream);
}

// ------------------------------------------------------------------------------------------------------
// (5) Ill-conditioned overlap: "electronic structure calculations can then be carried out by
// transforming the eigenproblem (2) to the basis of eigenvectors D_i of the overlap matrix, but omitting any D_i
// for which sigma_i is smaller than a small positive number delta".
//   S = D Sigma D^H (the eigensolver above, ALL N pairs);  X = D_kept Sigma_kept^-1/2  (X^H S X = I on the kept
//   directions; the dropped ones -- the lowest sigma, i.e. the first columns -- become zero columns);
//   H_r = X^H H X (two products on the tile engine; zero rows / columns for the dropped directions, whose diagonal
//   entries are set to a shift above the spectrum of H_r so that they can never be among the lowest nev);
//   then H_r y = eps y by gs_standard_eigh and C = X y by gs_backtransform_dense.
// ------------------------------------------------------------------------------------------------------
gs_status_t gs_truncated_workspace_bytes(const gs_plan_t* plan, size_t* bytes)
{
    if (plan == nullptr || bytes == nullptr) return GS_ERR_INVALID_ARG;
    evp_carve(plan, nullptr, bytes, plan->N);
    return GS_OK;
}

gs_status_t gs_truncated_to_standard(gs_plan_t* plan, const void* H, void* S_inout, double delta, void* X, void* Hr, double* sigma,
                                     void* cuda_stream)
{
    if (plan == nullptr) return GS_ERR_INVALID_ARG;
    EvpBuffers b;
    GS_TRY(evp_ready(plan, &b, plan->N));
    if (H == nullptr || S_inout == nullptr || X == nullptr || Hr == nullptr || sigma == nullptr || !(delta >= 0.0) || !aligned16(H) ||
        !aligned16(S_inout) || !aligned16(X) || !aligned16(Hr) || overlaps(X, mat_bytes(plan), H, mat_bytes(plan)) ||
        overlaps(X, mat_bytes(plan), S_inout, mat_bytes(plan)) || overlaps(Hr, mat_bytes(plan), H, mat_bytes(plan)) ||
        overlaps(Hr, mat_bytes(plan), X, mat_bytes(plan)) || overlaps(Hr, mat_bytes(plan), S_inout, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int N = int(plan->N);
    GS_TRY(evp_eigh_impl(plan, b, S_inout, sigma, X, N, stream));          // X = D (all eigenvectors), sigma ascending
    int* kept = info_ptr(plan) + 16;                                       // (a slot of the plan's 256-byte flag area)
    {
        LaunchTimer timer(plan, L_EVP_BACK, stream);
        const dim3 grid((N + 255) / 256, std::min(N, 4096));
        if (plan->z) truncate_scale_kernel<double2><<<grid, 256, 0, stream>>>(static_cast<double2*>(X), plan->N, N, sigma, delta, kept, info_ptr(plan));
        else truncate_scale_kernel<double><<<grid, 256, 0, stream>>>(static_cast<double*>(X), plan->N, N, sigma, delta, kept, info_ptr(plan));
        GS_LAUNCH_OK(plan);
    }
    Stage st = make_stage(plan, stream);
    const MatView vH{H, N, N, N}, vX{X, N, N, N}, vW{big_ptr(plan), N, N, N};
    const int kt = (N + st.bk - 1) / st.bk, nt = plan->nblk;
    {   // W = H X  (as H^H X: H is Hermitian, and the k-contiguous operand is the fast one)
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, vH, false) || !set_operand(st, p, 1, vX, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(big_ptr(plan)); p.ldc = N;
        p.tiles_m = nt; p.tiles_n = nt; p.order = ORDER_COL;
        p.c_rows = N; p.c_cols = N;
        p.khi_c = kt; p.kmax = kt;
        GS_TRY(launch(st, p, false, L_EVP_DC_GEMM));
    }
    {   // H_r = X^H W, upper triangle
        EngineParams p = blank_params(plan);
        if (!set_operand(st, p, 0, vX, false) || !set_operand(st, p, 1, vW, false)) return GS_ERR_CUDA;
        p.C = static_cast<double*>(Hr); p.ldc = N;
        p.tiles_m = nt; p.tiles_n = nt; p.order = ORDER_TRI_ROW_DESC;
        p.c_rows = N; p.c_cols = N;
        p.khi_c = kt; p.kmax = kt;
        p.flags = F_STORE_UPPER | F_REAL_DIAG;
        GS_TRY(launch(st, p, false, L_EVP_DC_GEMM));
    }
    {   // shift = 2 ||triu(H_r)||_F sqrt2 + 1 > lambda_max(H_r) on the diagonal of the dropped directions
        LaunchTimer timer(plan, L_EVP_BACK, stream);
        const int nb = std::min(64, (N + 255) / 256);
        if (plan->z) shift_dropped_kernel<double2><<<nb, 256, 0, stream>>>(static_cast<double2*>(Hr), plan->N, N, sigma, delta, static_cast<double*>(b.Pd), b.tickets + 3, info_ptr(plan));
        else shift_dropped_kernel<double><<<nb, 256, 0, stream>>>(static_cast<double*>(Hr), plan->N, N, sigma, delta, static_cast<double*>(b.Pd), b.tickets + 3, info_ptr(plan));
        GS_LAUNCH_OK(plan);
    }
    return GS_OK;
}

gs_status_t gs_truncated_rank(gs_plan_t* plan, void* cuda_stream, int64_t* kept)
{
    if (plan == nullptr || kept == nullptr) return GS_ERR_INVALID_ARG;
    GS_TRY(check_ready(plan));
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    int h = 0;
    GS_CUDA(plan, cudaMemcpyAsync(&h, info_ptr(plan) + 16, sizeof(int), cudaMemcpyDeviceToHost, stream));
    GS_CUDA(plan, cudaStreamSynchronize(stream));
    *kept = h;
    return GS_OK;
}

// C = X C~ with a DENSE X (N x N): the back-transformation of the truncated-basis route
gs_status_t gs_backtransform_dense(gs_plan_t* plan, const void* X, const void* Ctilde, void* C, void* cuda_stream)
{
    GS_TRY(check_ready(plan));
    if (plan->nev == 0) return GS_OK;
    if (X == nullptr || Ctilde == nullptr || C == nullptr || !aligned16(X) || !aligned16(Ctilde) || !aligned16(C) ||
        overlaps(C, vec_bytes(plan), Ctilde, vec_bytes(plan)) || overlaps(C, vec_bytes(plan), X, mat_bytes(plan)))
        return GS_ERR_INVALID_ARG;
    const int N = int(plan->N), nev = int(plan->nev);
    Stage st = make_stage(plan, static_cast<cudaStream_t>(cuda_stream));
    const MatView vX{X, N, N, N}, vC{Ctilde, N, nev, N};
    EngineParams p = blank_params(plan);
    if (!set_operand(st, p, 0, vX, true) || !set_operand(st, p, 1, vC, false)) return GS_ERR_CUDA;
    p.C = static_cast<double*>(C); p.ldc = N;
    p.tiles_m = plan->nblk; p.tiles_n = (nev + st.lb - 1) / st.lb; p.order = ORDER_ROW;
    p.c_rows = N; p.c_cols = nev;
    p.khi_c = (N + st.bk - 1) / st.bk; p.kmax = p.khi_c;
    return launch(st, p, true, L_BACK_TRMM);
}

}  // extern "C"

#ifdef GS_SV_TRACE
// Trace build only (evp_tridiag.cuh, "Timeline of one column"): arm the stamps for the blocks of order m and m - 1; read them back.
extern "C" int gs_trace_tridiag_arm(int m)
{
    unsigned long long init[2][4] = {{~0ull, ~0ull, 0ull, 0ull}, {~0ull, ~0ull, 0ull, 0ull}};
    void* ptr = nullptr;
    if (cudaMemcpyToSymbol(g_c_trace, init, sizeof(init)) != cudaSuccess || cudaGetSymbolAddress(&ptr, g_sv_trace) != cudaSuccess) return GS_ERR_CUDA;
    if (cudaMemset(ptr, 0, sizeof(unsigned long long) * 2 * kTraceCtas * 8) != cudaSuccess) return GS_ERR_CUDA;
    return cudaMemcpyToSymbol(g_sv_trace_m, &m, sizeof(int)) == cudaSuccess ? GS_OK : GS_ERR_CUDA;
}
extern "C" int gs_trace_tridiag_read(unsigned long long* s_stamps /* [2][600][8] */, unsigned long long* c_stamps /* [2][4] */)
{
    if (cudaDeviceSynchronize() != cudaSuccess) return GS_ERR_CUDA;
    if (cudaMemcpyFromSymbol(s_stamps, g_sv_trace, sizeof(unsigned long long) * 2 * kTraceCtas * 8) != cudaSuccess) return GS_ERR_CUDA;
    return cudaMemcpyFromSymbol(c_stamps, g_c_trace, sizeof(unsigned long long) * 2 * 4) == cudaSuccess ? GS_OK : GS_ERR_CUDA;
}
#endif
