/*
 * gs.h -- C ABI of libgs: reduction of the dense generalized eigenproblem  H C = eps S C
 * (H symmetric / Hermitian, S positive definite; Eq. 2) to standard form and the
 * eigenvector back-transformation, on ONE NVIDIA B200 (sm_100a), FP64.
 *
 * The four compute calls are the four steps of PAPER.md:61-67 ("Solving the generalized
 * eigenproblem"), which ELPA also exposes one by one ("interfaces for each individual
 * transformation step are also provided"):
 *
 *   gs_cholesky           1. Cholesky decomposition S = U^T U, U upper triangular
 *   gs_invert_triangular  2. inversion of the upper triangular matrix U -> U^-1
 *   gs_to_standard        3. two matrix products H~ = (U^-1)^T H U^-1
 *   gs_backtransform         back-transformation C = U^-1 C~
 *
 * "A^T corresponds to the transpose or conjugate-transpose of a real- or complex-valued matrix"
 * (PAPER.md:67).  The standard eigensolve H~ C~ = eps C~ between steps 3 and 4 is off the hot path of
 * BASELINE.json; the library has its own (gs_standard_eigh and its three stages, further down), and any other
 * eigensolver may be used instead.
 *
 * Conventions common to all calls
 * -------------------------------
 * Layout     Column-major, leading dimension = N (LAPACK/ELPA convention; eigenvectors are "stored
 *            as matrix columns").  C~ and C are N x nev with leading dimension N.
 *            GS_COMPLEX128 = interleaved (re, im) doubles.
 * Pointers   Every matrix argument is a DEVICE pointer (cudaMalloc-class memory on the current
 *            device), 16-byte aligned, caller-owned.  The library never allocates device memory
 *            for matrices; scratch is the caller-provided workspace (gs_plan_set_workspace).
 *            Outputs must not OVERLAP inputs (byte ranges, not only equal pointers) except the
 *            documented in-place S_inout: GS_ERR_INVALID_ARG.  NULL or misaligned matrix pointers:
 *            GS_ERR_INVALID_ARG.  Workspace / scratch missing, too small or misaligned: GS_ERR_WORKSPACE.
 * Streams    `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *            Compute calls only enqueue work on it and return without synchronising.
 * Errors     Every call returns a gs_status_t and never throws or exits.  Argument errors are
 *            returned synchronously.  Numerical failure (a pivot that is not > 0, or NaN, in
 *            gs_cholesky; a zero diagonal entry in gs_invert_triangular) is recorded in a
 *            device-side flag as the 1-based index of the first bad pivot; all later compute
 *            calls on the same plan become no-ops while the flag is set; gs_last_info synchronises
 *            the stream and reports it.  gs_cholesky clears the flag when it starts; a plan used
 *            for the later steps only clears it with gs_plan_clear_info.
 * No CPU fallback exists: without a device of compute capability 10.x plan creation fails with
 *            GS_ERR_UNSUPPORTED_DEVICE.
 * Domain     1 <= N <= 2^20, 0 <= nev <= N.  Any such N is accepted (ragged edges are handled in the
 *            kernels; odd N takes a loader without tensor maps).
 */
#ifndef GS_H_
#define GS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gs_plan gs_plan_t; /* opaque host object */

typedef enum { GS_REAL64 = 0, GS_COMPLEX128 = 1 } gs_dtype_t;

typedef enum {
    GS_OK = 0,
    GS_ERR_INVALID_ARG = 1,
    GS_ERR_NOT_POSDEF = 2,         /* gs_last_info: pivot `info` of S is not positive          */
    GS_ERR_SINGULAR = 3,           /* gs_last_info: U(info,info) == 0                            */
    GS_ERR_CUDA = 4,               /* a CUDA runtime/driver call failed                          */
    GS_ERR_WORKSPACE = 5,          /* workspace missing, too small or misaligned                 */
    GS_ERR_UNSUPPORTED_DEVICE = 6, /* current device is not compute capability 10.x              */
    GS_ERR_NO_CONVERGENCE = 7      /* gs_last_info: the tridiagonal eigensolver did not converge */
} gs_status_t;

/* Create a plan for problems of order N, element type dtype, and nev wanted eigenvectors
 * (BASELINE.json north_star: gs_plan_create(N, dtype, nev)).  Host-only state (tile schedule,
 * TMA descriptors are built per call from the pointers).  *plan is set to NULL on failure. */
gs_status_t gs_plan_create(gs_plan_t** plan, int64_t N, gs_dtype_t dtype, int64_t nev);
gs_status_t gs_plan_destroy(gs_plan_t* plan);

/* Scratch the compute calls need: at most one N x N matrix plus O(N * 128) elements.  The caller
 * allocates `bytes` of device memory (256-byte aligned) and hands it over; it stays caller-owned
 * and must outlive every compute call enqueued on the plan.  Contents are undefined between calls. */
gs_status_t gs_plan_workspace_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_plan_set_workspace(gs_plan_t* plan, void* dev_workspace, size_t bytes);

/* Step 1.  In place: on entry the upper triangle (incl. diagonal) of S_inout holds S
 * (the strictly-lower part is never read); on exit the upper triangle holds U with real, strictly
 * positive diagonal, S = U^H U, and the strictly-lower part is zero.
 * Blocked right-looking POTRF: diagonal blocks factored in shared memory, panel solve and SYRK/HERK
 * trailing update on FP64 tensor-core (DMMA) tiles. */
gs_status_t gs_cholesky(gs_plan_t* plan, void* S_inout, void* cuda_stream);

/* Step 1 restricted to the leading ncols x ncols block of S_inout (ncols a multiple of the block
 * order -- 128 real, 64 complex -- or equal to N): the leading principal blocks of the factor nest,
 * chol(S[:k,:k]) = U[:k,:k], so a rank of the sharded path that owns columns up to k factors only
 * that block.  Upper triangle of the leading block: U; strictly-lower blocks of the whole buffer:
 * zero; everything else in columns >= ncols is left as it was (still S).  ncols == 0 is a no-op. */
gs_status_t gs_cholesky_leading(gs_plan_t* plan, void* S_inout, int64_t ncols, void* cuda_stream);

/* Step 2.  Reads the upper triangle of U (N x N); writes Uinv = U^-1 (upper
 * triangle) and zeros below the diagonal.  Uinv must not alias U.  Blocked TRTRI. */
gs_status_t gs_invert_triangular(gs_plan_t* plan, const void* U, void* Uinv, void* cuda_stream);

/* Step 3.  Htilde = Uinv^H * H * Uinv.  H must be symmetric / Hermitian with both
 * triangles filled consistently (the kernels reference its lower triangle and diagonal); only the
 * upper triangle of Uinv is read.  Writes the UPPER triangle (incl. diagonal) of Htilde; the
 * strictly-lower part of the Htilde buffer is left untouched.  For GS_COMPLEX128 the diagonal of
 * Htilde is exactly real.  Fused triangular product pair: exploits the triangularity of Uinv and
 * forms one triangle of the symmetric result only. */
gs_status_t gs_to_standard(gs_plan_t* plan, const void* H, const void* Uinv, void* Htilde,
                           void* cuda_stream);

/* Back-transformation.  C = Uinv * Ctilde over the nev columns of the plan (no
 * conjugation).  Reads the upper triangle of Uinv and all of Ctilde (N x nev); writes C (N x nev).
 * nev == 0 is a no-op. */
gs_status_t gs_backtransform(gs_plan_t* plan, const void* Uinv, const void* Ctilde, void* C,
                             void* cuda_stream);

/* Step 1 over the GPUs of one NVSwitch domain (and the paper's
 * multi-GPU direction PAPER.md:118): one process per GPU, every rank calls it with its own copy of S
 * (N x N, ld N, upper triangle referenced) and on return -- in stream order -- holds the COMPLETE factor U in it
 * (upper triangle; zeros below), the same bits on every rank.
 * Panels of the plan's panel width (8 blocks of 128, 64 for GS_COMPLEX128) are dealt round-robin: panel p belongs
 * to rank p mod nranks, which keeps the block columns of its panels up to date and nothing else.  Per panel the
 * owner factors and inverts the diagonal block and copies both into every rank; every rank then forms its own
 * pieces of the row panel U[p, q] = W_p^H S[p, q] and stores them into its own S AND into every peer's S (the
 * all-gather of the row panel, fused into the producing side), and applies the trailing update to its own panels.
 *   peer_S[s], peer_workspace[s]  rank s's S buffer and the workspace of its plan (same N, dtype: same layout) as
 *                                 mapped in this process (gs_ipc_open; entry `rank` = this rank's own S_inout and
 *                                 the plan's workspace);
 *   flags[s]                      rank s's array of nranks 32-bit flags (zero before the first call; entry `rank`
 *                                 local).  Rank r writes slot r of every peer's array and waits on its own array
 *                                 (gs_exchange_signal / gs_exchange_wait: stream memory operations, no host
 *                                 synchronisation, no spinning kernel);
 *   epoch0                        the call uses the flag values epoch0 + 1 (every rank's S is in place: nothing is stored
 *                                 into a buffer its owner is still filling) ... epoch0 + gs_cholesky_sharded_epochs();
 *                                 every rank passes the same value and raises it by that count from call to call.
 * nranks == 1 needs no peers (NULL).  nranks <= 8.  One stream per rank; the owner of the next panel updates that
 * panel first and factors its diagonal block before its other updates (one panel of look-ahead), so the chain of a
 * diagonal block runs beside the other ranks' trailing updates.  Every rank signals whatever its
 * numerical status (a failed rank's kernels are no-ops, its signals are not): agree on gs_last_info afterwards. */
gs_status_t gs_cholesky_sharded_epochs(const gs_plan_t* plan, uint32_t* count);
gs_status_t gs_cholesky_sharded(gs_plan_t* plan, void* S_inout, int rank, int nranks, void* const* peer_S,
                                void* const* peer_workspace, void* const* flags, uint32_t epoch0, void* cuda_stream);

/* Column-range forms of steps 2, 3 and of the back-transformation: the path sharded over the
 * GPUs of one NVSwitch domain (the paper's multi-GPU direction,
 * PAPER.md:118).  Every rank holds U (step 1 is replicated) and owns a contiguous
 * range of block columns J = [col0, col0 + ncols): col0 a multiple of the block order (128 real,
 * 64 complex), col0 + ncols a multiple of it or equal to the matrix width.  ncols == 0 is a no-op.
 * All matrices are N x N (C~, C: N x nev), column-major, ld = N, device pointers, caller-owned; a
 * column range is therefore one contiguous slab of the buffer, which is what the ranks exchange.
 *
 * gs_invert_triangular_cols: columns J of Uinv = U^-1, rows 0 .. col0+ncols-1, by
 *   blocked back substitution of U X = E_J.  Zeroes the strictly-lower blocks of the whole Uinv buffer
 *   and writes the inverted diagonal blocks left of J (which it needs and forms itself); the columns right
 *   of J are left untouched above the diagonal blocks.  Reads only the upper triangle of U.
 * gs_to_standard_g_cols: columns J of the intermediate G = T Uinv, T = triu(H,1) + diag(H)/2
 *   (H = T + T^H, so H~ = Uinv^H G + G^H Uinv).  Needs only the columns J of Uinv.
 *   G is a caller-owned N x N buffer (it is exchanged between ranks).
 * gs_to_standard_cols: columns J of the UPPER triangle of Htilde (rows 0 .. diagonal).  Reads the
 *   columns [0, col0 + ncols) of Uinv and of G: the slabs of the lower-numbered ranges and its own.
 * gs_backtransform_cols: C[:, K] = Uinv C~[:, K] for the eigenvector columns K = [col0, col0+ncols)
 *   of the plan's nev (any col0 with a 16-byte aligned column start); needs all of Uinv.
 * Errors and asynchrony as for the whole-matrix calls. */
gs_status_t gs_invert_triangular_cols(gs_plan_t* plan, const void* U, void* Uinv, int64_t col0, int64_t ncols,
                                      void* cuda_stream);
gs_status_t gs_to_standard_g_cols(gs_plan_t* plan, const void* H, const void* Uinv, void* G, int64_t col0,
                                  int64_t ncols, void* cuda_stream);
gs_status_t gs_to_standard_cols(gs_plan_t* plan, const void* Uinv, const void* G, void* Htilde, int64_t col0,
                                int64_t ncols, void* cuda_stream);
gs_status_t gs_backtransform_cols(gs_plan_t* plan, const void* Uinv, const void* Ctilde, void* C, int64_t col0,
                                  int64_t ncols, void* cuda_stream);

/* Fused exchange of the sharded path: the column-range calls can store what they produce not only
 * into their own output buffer but, from the same kernel epilogue, into up to 8 further buffers of
 * the same shape and layout -- the other ranks' copies, mapped over NVLink/NVSwitch peer memory --
 * so the slabs travel while the remaining tiles are still being computed and no separate
 * collective follows.  `kind` selects the result:
 *   GS_PUSH_UINV    gs_invert_triangular_cols: the columns J of U^-1 (rows above and inside the
 *                   diagonal blocks).  Here the Uinv ARGUMENT of the call is the rank's private work
 *                   buffer; the targets are the exchange buffers of ALL ranks including its own,
 *                   whose strictly-lower part the owner has zeroed once (nothing is pushed there).
 *   GS_PUSH_G       gs_to_standard_g_cols: the columns J of G      (targets: the other ranks' G)
 *   GS_PUSH_HTILDE  gs_to_standard_cols:   the columns J of triu(H~) (targets: the other ranks' H~)
 *   GS_PUSH_C       gs_backtransform_cols: the columns K of C      (targets: the other ranks' C)
 * Every element of a target has exactly one writer (the owner of its column).  Completion: once the
 * writer's stream has been synchronised the stores have landed; a barrier between the ranks must
 * separate them from the first read (and the reads from the next round of stores).  count == 0
 * clears the set.  Targets are device pointers valid in this process: local buffers, or other
 * processes' allocations opened with gs_ipc_open. */
typedef enum { GS_PUSH_UINV = 0, GS_PUSH_G = 1, GS_PUSH_HTILDE = 2, GS_PUSH_C = 3 } gs_push_kind_t;
gs_status_t gs_plan_set_push_targets(gs_plan_t* plan, gs_push_kind_t kind, int count, void* const* targets);

/* Device-side ordering of the fused exchange (instead of a host `stream synchronise + barrier` between producing a
 * slab and consuming the peers' slabs): every rank owns a small array of 32-bit flags in device memory, mapped into
 * its peers like the push targets.
 *   gs_exchange_signal  enqueues on `cuda_stream`, BEHIND everything already enqueued there (so behind the kernels whose
 *                       epilogues pushed the slabs; a memory barrier precedes the write), the write of `value` to each
 *                       of the `count` flag addresses (local, or a peer's opened with gs_ipc_open);
 *   gs_exchange_wait    enqueues a wait until every one of the `count` LOCAL flags is >= `value` (wrap-around aware
 *                       comparison of the driver); later work of the stream starts only then.
 * Both are stream memory operations of the driver (cuStreamWriteValue32 / cuStreamWaitValue32): no kernel spins, no SM
 * is held, the host is not synchronised.  Flags are 4-byte aligned device addresses; use increasing epochs as values.
 * A wait whose signal is never enqueued blocks its stream for good: every rank must signal, also after a numerical
 * failure (the compute calls are no-ops then, the signals are not).
 * With CUDA's lazy module loading the FIRST launch of a kernel may synchronise with the device: behind a pending wait it
 * returns only once the wait is satisfied.  Across processes that is a delay in the first round; ranks emulated in ONE
 * process by one host thread would deadlock (the thread never gets to enqueue the signalling rank).  gs_cholesky_sharded
 * therefore loads its kernels before it enqueues its first wait; callers that build their own sequences around
 * gs_exchange_wait should run each call once before the first wait, or set CUDA_MODULE_LOADING=EAGER. */
gs_status_t gs_exchange_signal(gs_plan_t* plan, int count, void* const* flags, uint32_t value, void* cuda_stream);
gs_status_t gs_exchange_wait(gs_plan_t* plan, int count, void* const* flags, uint32_t value, void* cuda_stream);

/* CUDA IPC plumbing for the targets (one process per GPU).  gs_ipc_export: the 64-byte handle of the
 * device allocation that contains dev_ptr and dev_ptr's byte offset inside it (send both to the
 * peer).  gs_ipc_open (in another process): maps that allocation, enabling peer access, and returns
 * the pointer that corresponds to dev_ptr.  gs_ipc_close: unmaps (pass the pointer gs_ipc_open
 * returned and the same offset).  GS_ERR_CUDA if the driver refuses (e.g. memory that was not
 * allocated with cudaMalloc). */
gs_status_t gs_ipc_export(const void* dev_ptr, unsigned char* handle64, uint64_t* offset);
gs_status_t gs_ipc_open(const unsigned char* handle64, uint64_t offset, void** dev_ptr);
gs_status_t gs_ipc_close(void* dev_ptr, uint64_t offset);

/* Density matrix (the step that follows the path; "single-particle density matrix
 * P_ij = sum_l f_l c*_li c_lj", with c_li = C(i,l), eigenvectors stored as columns):
 *     P(i,j) = sum_{l < nev} f[l] * conj(C(i,l)) * C(j,l).
 * C is N x nev (ld N); f is a DEVICE array of nev real occupation numbers, f[l] >= 0 (a negative
 * occupation gives NaN); P is N x N (ld N): the UPPER triangle (incl. the diagonal, exactly real for
 * GS_COMPLEX128) is written, the strictly-lower part is left untouched.  nev == 0 writes zeros.
 * One weighted SYRK / HERK on the tensor-core tile engine over sqrt(f)-scaled, transposed C (held
 * in the plan's workspace). */
gs_status_t gs_density_matrix(gs_plan_t* plan, const void* C, const double* f, void* P, void* cuda_stream);

/* The same operation for callers that cannot allocate device memory -- code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc: identical kernels and results, but the scratch
 * (the status flag and the sqrt(f)-scaled, transposed eigenvector block) lives in a static device array of
 * GS_STATIC_SCRATCH_BYTES inside libgs, which every GPU that loads the library holds until the process exits.
 * The plan needs NO workspace (gs_plan_set_workspace may never have been called); the call allocates nothing
 * (no cudaMalloc / cudaFree, no allocating library routine) and, like the other compute calls, only enqueues
 * work.  C, f, P are the caller's device buffers as above.
 * Limit: 256 + N * nev' * sizeof(element) <= GS_STATIC_SCRATCH_BYTES, nev' = nev rounded up to even for
 * GS_REAL64 (2 for nev == 0) -- e.g. N = nev = 1024 complex, or N = 2048 with nev = 1024 real / 512 complex.
 * Beyond it: GS_ERR_WORKSPACE, and gs_plan_last_cuda_error names the sizes; use gs_density_matrix.
 * ALL calls in the process on one device share the one array, whatever their plan or stream: two calls whose
 * GPU work may overlap (different streams without an edge between them, several host threads) RACE on it --
 * order them.  The array keeps the previous call's contents; the call clears what must start at zero.
 * There is no numerical status to report (a negative occupation gives NaN, as above); the plan's own status
 * flag (gs_last_info) is neither read nor written. */
#define GS_STATIC_SCRATCH_BYTES (16u * 1024u * 1024u + 256u)
gs_status_t gs_density_matrix_static(gs_plan_t* plan, const void* C, const double* f, void* P, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------------
 * NEXT-4: the standard eigenproblem  H~ C~ = C~ eps  that sits between step 3 and the
 * back-transformation ("This reduces the generalized eigenproblem to the standard one, H~ C~ = eps C~, which has
 * the same set of eigenvalues"), for the LOWEST nev eigenpairs of the plan (ascending), in the
 * three stages of the paper's Table 1 under "Standard EVP":
 *
 *   gs_evp_tridiagonalize  "Tridiag."  H~ = Q T Q^H by the one-stage Householder reduction ("ELPA1", the
 *                          conventional one-stage method, which the paper reports as the faster one on GPUs,
 *                          PAPER.md:120).  A_inout: N x N, ld N; on entry its UPPER triangle holds H~ (what
 *                          gs_to_standard writes; the strictly-lower part is never read); on exit column i holds
 *                          the Householder vector v_i (rows 0 .. i-1, v_i(i-1) = 1, zeros below) of
 *                          H(i) = I - tau(i) v_i v_i^H, Q = H(N-1) ... H(1): H~ is destroyed.  d (N) and e (N-1
 *                          used) receive the diagonal and off-diagonal of the real symmetric tridiagonal T; tau
 *                          (N elements of the plan's dtype) the reflector scalars.  All device pointers.
 *   gs_evp_tridiag_solve   "Solve"     the lowest nev eigenvalues of T -> eps (nev, ascending) and their
 *                          eigenvectors -> Z (N x nev REAL, ld N), by divide and conquer (secular equation
 *                          solved per root, Gu-Eisenstat vectors, the block products on the tile engine).
 *                          d, e are not modified.  SYNCHRONISES the stream once per level of the recursion
 *                          (the deflation counts decide the shapes of the launches that follow).
 *   gs_evp_backtransform   "Back"      C~ = Q Z (N x nev, the plan's dtype, ld N): blocked reflectors (compact
 *                          WY, one panel = one block) applied on the tile engine.  A_reflectors is the matrix
 *                          gs_evp_tridiagonalize left; the triangular factors of the blocks are kept in the
 *                          plan's EVP workspace, so the call belongs to the LAST gs_evp_tridiagonalize on the plan.
 *   gs_standard_eigh       the three in a row: eps (nev) and C~ (N x nev) from the upper triangle of Htilde_inout
 *                          (destroyed).  C~ is what gs_backtransform takes.
 *
 * Scratch: a second caller-owned device buffer (about 3 N^2 + N nev doubles), gs_evp_workspace_bytes /
 * gs_evp_set_workspace, 256-byte aligned; GS_ERR_WORKSPACE if missing or too small.  The plan's ordinary
 * workspace must be set as well.  C~ is unique only up to the phase of each column (and up to rotations inside
 * clusters of equal eigenvalues): compare residuals and orthonormality, not elements.
 * Numerical failure: GS_ERR_NO_CONVERGENCE from gs_last_info if the QL iteration of a leaf does not converge. */
gs_status_t gs_evp_workspace_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_evp_set_workspace(gs_plan_t* plan, void* dev_workspace, size_t bytes);
gs_status_t gs_evp_tridiagonalize(gs_plan_t* plan, void* A_inout, double* d, double* e, void* tau, void* cuda_stream);
gs_status_t gs_evp_tridiag_solve(gs_plan_t* plan, const double* d, const double* e, double* eps, double* Z, void* cuda_stream);
gs_status_t gs_evp_backtransform(gs_plan_t* plan, const void* A_reflectors, const double* Z, void* Ctilde, void* cuda_stream);
gs_status_t gs_standard_eigh(gs_plan_t* plan, void* Htilde_inout, double* eps, void* Ctilde, void* cuda_stream);

/* Eigenvalues only ("If the eigenvectors are needed, one has to perform the backtransformation", PAPER.md:67 -- if they
 * are not, the divide and conquer and both back-transformations are not needed either):
 *   gs_evp_tridiag_eigenvalues  the `count` smallest eigenvalues (ascending, 0 <= count <= N) of the real symmetric
 *                               tridiagonal matrix tridiag(e, d, e) of order N by bisection on the Sturm count
 *                               (Sylvester's inertia of T - x I), each to the last bit the interval can be halved to.
 *                               d (N), e (N - 1 used), eps (count): device pointers; d, e are not modified.  Needs the
 *                               plan's ordinary workspace only; does not synchronise.
 *   gs_standard_eigenvalues     the `count` smallest eigenvalues of the Hermitian matrix whose upper triangle is in
 *                               Htilde_inout: gs_evp_tridiagonalize (Htilde_inout is destroyed: it holds the Householder
 *                               vectors afterwards) + gs_evp_tridiag_eigenvalues.  Needs the eigensolver workspace. */
gs_status_t gs_evp_tridiag_eigenvalues(gs_plan_t* plan, const double* d, const double* e, int64_t count, double* eps, void* cuda_stream);
gs_status_t gs_standard_eigenvalues(gs_plan_t* plan, void* Htilde_inout, int64_t count, double* eps, void* cuda_stream);

/* The whole generalized solve  H C = eps S C  of PAPER.md:61-67 in ONE call, for the lowest nev eigenpairs of the plan
 * (ELPA's own interface offers the one call and the individual steps): gs_cholesky, gs_invert_triangular,
 * gs_to_standard, gs_standard_eigh and gs_backtransform enqueued one after the other on `cuda_stream`, with the
 * arguments, triangles, aliasing rules and failure behaviour of those calls.
 *   H        N x N, both triangles, not modified        S_inout  N x N: S (upper triangle) on entry, U on return
 *   Uinv     N x N out: U^-1                            Htilde   N x N scratch (H~, then the Householder vectors)
 *   Ctilde   N x nev scratch (the eigenvectors of H~)   eps      nev eigenvalues, ascending
 *   C        N x nev out: the eigenvectors, C^H S C = I
 * All device pointers, caller-owned; both workspaces (gs_plan_set_workspace, gs_evp_set_workspace) must be set.
 * SYNCHRONISES the stream inside (the divide and conquer of gs_evp_tridiag_solve, once per level). */
gs_status_t gs_generalized_eigh(gs_plan_t* plan, const void* H, void* S_inout, void* Uinv, void* Htilde, void* Ctilde,
                                double* eps, void* C, void* cuda_stream);

/* ------------------------------------------------------------------------------------------------------
 * (5) Ill-conditioned overlap matrix.  "In the latter case (high condition number of S),
 * electronic structure calculations can then be carried out by transforming the eigenproblem (2) to the basis of
 * eigenvectors D_i of the overlap matrix, but omitting any D_i for which sigma_i is smaller than a small positive
 * number delta (typically delta <= 1e-5)".  The route that replaces steps 1-3 when S is close to
 * singular (steps 1-3 need "S must not be numerically singular"):
 *
 *   gs_truncated_to_standard   S = D Sigma D^H by the eigensolver above (all N pairs);  X = D Sigma^-1/2 on the kept
 *                              directions (sigma_i >= delta), ZERO columns for the dropped ones (the lowest sigma:
 *                              the first columns);  Hr = X^H H X.  S_inout (upper triangle = S) is destroyed.
 *                              X, Hr: N x N outputs (Hr: upper triangle written; rows / columns of dropped directions
 *                              are zero except for a diagonal entry above the spectrum of Hr, so they never enter the
 *                              lowest eigenvalues).  sigma: N eigenvalues of S, ascending.  H: both triangles filled.
 *   gs_truncated_rank          synchronises; number of kept directions (must be >= nev for the lowest nev to be meaningful).
 *   then  gs_standard_eigh(plan, Hr, eps, Ctilde)  and
 *   gs_backtransform_dense     C = X Ctilde (X dense N x N, Ctilde N x nev).  C^H S C = I, X^H (H C - S C eps) = 0.
 *
 * EVP workspace: gs_truncated_workspace_bytes (larger than gs_evp_workspace_bytes when nev < N: all N eigenvectors
 * of S are formed), registered with gs_evp_set_workspace. */
gs_status_t gs_truncated_workspace_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_truncated_to_standard(gs_plan_t* plan, const void* H, void* S_inout, double delta, void* X, void* Hr, double* sigma,
                                     void* cuda_stream);
gs_status_t gs_truncated_rank(gs_plan_t* plan, void* cuda_stream, int64_t* kept);
gs_status_t gs_backtransform_dense(gs_plan_t* plan, const void* X, const void* Ctilde, void* C, void* cuda_stream);

/* Synchronises `cuda_stream`, then reports the plan's numerical status: GS_OK with *info = 0, or
 * GS_ERR_NOT_POSDEF / GS_ERR_SINGULAR with *info = 1-based index of the first bad pivot
 * (LAPACK-style).  GS_ERR_CUDA if the stream reports an asynchronous error. */
gs_status_t gs_last_info(gs_plan_t* plan, void* cuda_stream, int64_t* info);

/* Clears the plan's numerical-failure flag (enqueued on `cuda_stream`): the way back to a usable plan
 * after GS_ERR_SINGULAR / GS_ERR_NOT_POSDEF when the next call is not gs_cholesky (which clears it itself). */
gs_status_t gs_plan_clear_info(gs_plan_t* plan, void* cuda_stream);

/* Host-buffer entry points (the calls an application with H, S in host memory makes; used for the
 * end-to-end measurement).  gs_reduce_host copies S and H from HOST memory into device scratch
 * inside [dev_scratch, dev_scratch + scratch_bytes) -- only the triangles the steps reference: the
 * UPPER triangle of host_S and the LOWER triangle of host_H (both with the diagonal, in chunks;
 * the other triangle of either host buffer is never read; step 1 starts once the rows of S that its
 * first two panels cover are in, and applies its first trailing update slab by slab as the remaining
 * rows arrive) --, runs steps 1-3 there and copies the UPPER
 * triangle of H~ back to host_Htilde (N x N, ld N; the strictly-lower part of the host buffer is
 * unspecified -- callers read the upper triangle only).  Copies overlap compute on plan-owned copy
 * streams that are joined before return: H goes in beside steps 1-2, step 3 is formed in row ranges
 * whose finished rows go back beside the next range; gs_backtransform_host pipelines column chunks.  host_U / host_Uinv may be NULL (then they are not copied back).  U^-1 stays
 * in the scratch: gs_backtransform_host, called later with the SAME scratch, copies C~ (N x nev) in,
 * forms C = U^-1 C~ and copies C out.  Both synchronise the stream before returning and report
 * numerical failure like gs_last_info.  Scratch size: gs_reduce_host_scratch_bytes(); 256-byte
 * aligned (NULL, too small or misaligned: GS_ERR_WORKSPACE).  gs_reduce_host_h2d_bytes / gs_reduce_host_d2h_bytes report the bytes gs_reduce_host
 * copies in for S and H / back for H~. */
gs_status_t gs_reduce_host_scratch_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_reduce_host_h2d_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_reduce_host_d2h_bytes(const gs_plan_t* plan, size_t* bytes);
gs_status_t gs_reduce_host(gs_plan_t* plan, const void* host_H, const void* host_S,
                           void* host_U, void* host_Uinv, void* host_Htilde,
                           void* dev_scratch, size_t scratch_bytes, void* cuda_stream);
gs_status_t gs_backtransform_host(gs_plan_t* plan, const void* host_Ctilde, void* host_C,
                                  void* dev_scratch, size_t scratch_bytes, void* cuda_stream);

/* Optional per-launch device timing (CUDA events on the launching stream), for roofline reports.
 * mode 0 = off (default); 1 = every kernel launch; 2 = only the dominant kernel (the SYR2K-shaped
 * launch of gs_to_standard).  gs_plan_launch_times synchronises nothing: call it after the stream
 * has been synchronised.  It fills up to `cap` entries (label, launches, total milliseconds)
 * accumulated since the last gs_plan_set_timing call and returns the number of labels in *count. */
typedef struct {
    char label[32];
    int64_t launches;
    double ms;
} gs_launch_time_t;
gs_status_t gs_plan_set_timing(gs_plan_t* plan, int mode);
gs_status_t gs_plan_launch_times(gs_plan_t* plan, gs_launch_time_t* out, int cap, int* count);

/* The same events as a timeline (does not clear them; call before gs_plan_launch_times): entry i =
 * launch i since gs_plan_set_timing(…, 1), start / end in milliseconds after the start of launch 0,
 * side_stream = 1 if it ran on the plan's look-ahead stream.  *count = number of launches recorded
 * (may exceed cap; only cap entries are written).  Call after the stream has been synchronised. */
typedef struct {
    char label[32];
    int32_t side_stream;
    double t0_ms, t1_ms;
} gs_launch_trace_t;
gs_status_t gs_plan_launch_trace(gs_plan_t* plan, gs_launch_trace_t* out, int cap, int* count);

/* Number of kernels the library has launched on behalf of this plan since creation. */
gs_status_t gs_plan_launch_count(const gs_plan_t* plan, int64_t* launches);

const char* gs_status_string(gs_status_t status);
/* Text of the last CUDA error seen by this plan ("" if none). */
const char* gs_plan_last_cuda_error(const gs_plan_t* plan);

#ifdef __cplusplus
}
#endif
#endif /* GS_H_ */
