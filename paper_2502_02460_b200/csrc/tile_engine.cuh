// tile_engine.cuh -- the FP64 tile engine every stage of libgs is built from (real FP64).
//
// One launch computes a set of 128 x 128 output tiles
//     C[I,J] = alpha * sum_{kt = k_lo(I,J)}^{k_hi(I,J)-1} ( opA(kt,I) * B(kt,J)  [+ opA2(kt,I) * B2(kt,J)] ) + beta * C[I,J]
// where the k-range of each tile is an affine function of its tile indices.  That is enough to
// express every contraction of PAPER.md:61-67 with its triangular structure exploited (tiles of
// zeros are never loaded or multiplied):
//   SYRK trailing update of the blocked Cholesky, the panel solve with inverted diagonal blocks,
//   the block-recursive triangular inversion, G = T * Uinv (upper x upper), the SYR2K-shaped
//   H~ = Uinv^T G + G^T Uinv (one triangle), and the back-transform C = Uinv * C~.
//
// Hardware mapping (sm_100a):
//   * FP64 tensor pipe: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4); tcgen05 has no FP64 kind and
//     wgmma does not exist on sm_100a, so the legacy warp-level MMA is the FP64 tensor route.
//   * Operand tiles are staged by TMA (cp.async.bulk.tensor.2d, 128-byte swizzle) into a
//     kStages-deep shared-memory ring guarded by full/empty mbarriers; one producer warp issues
//     the copies, eight consumer warps (4 x 2, each a 32 x 64 warp tile = 64 FP64 accumulators per
//     thread) issue the DMMAs.
//   * Fragments are read with conflict-free 128-bit shared loads: one LDS.128 yields the operand
//     of two consecutive DMMA k-steps (k-contiguous operands) or of two adjacent row groups
//     (m-contiguous operand); the swizzle XOR is chosen so each quarter-warp covers all 32 banks.
//
// Matrices are column-major.  B(kt,J) tiles are always "k-contiguous" (B is K x N column-major).
// opA is either k-contiguous (A stored K x M, used as A^T: "TN") or m-contiguous (A stored M x K:
// "NN").  Complex and ragged-pitch (odd N) variants live in their own kernels.
#pragma once
#include "ptx.cuh"

namespace gs {

constexpr int BM = 128;       // C tile rows
constexpr int BN = 128;       // C tile cols
constexpr int BK = 16;        // k-slab per pipeline stage (16 doubles = one 128-byte swizzle row)
constexpr int kStages = 6;    // 6 x 32 KB = 192 KB of the 227 KB shared memory
constexpr int kConsumerWarps = 8;
constexpr int kThreads = (kConsumerWarps + 1) * 32;
constexpr int kTileBytes = BM * BK * 8;                    // 16 KB per operand tile
constexpr int kStageBytes = 2 * kTileBytes;                // A + B
constexpr int kSmemBytes = kStages * kStageBytes + 1024 /*align*/ + 256 /*barriers*/;

// flags
enum : uint32_t {
    F_DUAL = 1u << 0,          // second operand pair (A2,B2) accumulated into the same tile
    F_MASK_A = 1u << 1,        // zero A elements whose global (row > col)
    F_HALF_DIAG_A = 1u << 2,   // scale A elements with global row == col by 0.5
    F_MASK_B = 1u << 3,        // zero B elements whose global (row > col)
    F_MASK_A2 = 1u << 4,
    F_MASK_B2 = 1u << 5,
    F_STORE_UPPER = 1u << 6,   // store only C elements with global row <= col
    F_NO_SPLIT = 1u << 9,      // host only: C aliases the B operand tile by tile (in-place solve): one CTA per logical tile
    F_LOWER_A = 1u << 8,       // with F_MASK_A: A keeps its LOWER triangle instead (zero where row < col)
    F_REAL_DIAG = 1u << 7,     // complex engine: store Im = 0 on the global diagonal (Hermitian results)
};

// tile enumeration orders (heaviest tiles first so the tail of the grid is made of short tiles)
enum : int {
    ORDER_COL = 0,        // full grid, I fastest
    ORDER_ROW = 1,        // full grid, J fastest (rows I ascending)
    ORDER_ROW_REV = 2,    // full grid, J fastest, J descending first... (I ascending, J descending)
    ORDER_COL_REV = 3,    // full grid, I fastest, J descending
    ORDER_TRI_ROW_DESC = 4,   // upper triangle I <= J, rows I descending (cost ~ I+1)
    ORDER_TRI_DIAG_DESC = 5,  // upper triangle, diagonals d = J-I descending (cost ~ d+1)
    ORDER_TRAPEZOID = 6,      // tiles_m rows of a tiles_n-wide upper trapezoid: row I holds J = I .. tiles_n-1
};

struct OperandCoord {
    int k0, x0;     // element origin along k and along the free index (m for A, n for B)
    int bk, bx;     // per-batch increments
};

// Raw view of an operand matrix for the non-TMA loader (odd leading dimension: a row pitch that is
// not a multiple of 16 bytes cannot be described by a tensor map).
struct RawOperand {
    const double* ptr;
    long long ld;
    int rows, cols;
};

constexpr int kMaxPeers = 8;   // push targets of one launch: the GPUs of one NVSwitch domain

struct EngineParams {
    CUtensorMap mapA, mapB, mapA2, mapB2;
    RawOperand rawA, rawB, rawA2, rawB2;
    double* C;
    long long ldc;
    const int* info;              // device flag: non-zero => the whole launch is a no-op
    int tiles_m, tiles_n, batch, order;
    int super;                    // triangular orders: edge (in tiles) of the square super-tiles the grid is rasterised in (<= 1: off)
    int c_row0, c_col0, c_brow, c_bcol;   // C tile (b,I,J) starts at (c_row0 + b*c_brow + BM*I, c_col0 + b*c_bcol + BN*J)
    int c_rows, c_cols;                   // stores are predicated on row < c_rows && col < c_cols
    int klo_c, klo_i, klo_j;              // k_lo = klo_c + klo_i*I + klo_j*J   (units of BK), clamped to >= 0
    int khi_c, khi_i, khi_j;              // k_hi likewise, clamped to <= kmax
    int kmax;
    OperandCoord a, b, a2, b2;
    uint32_t flags;
    double alpha, beta;
    // Fused exchange (sharded path): every C element this launch stores whose global column is >= peer_col0
    // is ALSO stored, at the same (row, col, ldc), into each of the npeer matrices peer[d] -- buffers of the
    // other ranks mapped over NVLink (or further local buffers).  Posted remote stores: the transfer runs
    // beside the mainloops of the CTAs that follow, tile by tile; nothing is read back.
    double* peer[kMaxPeers];
    int npeer, peer_col0;
};

// Returns false for the padding CTAs of a super-tiled triangular grid (they exit at once).
__device__ __forceinline__ bool decode_tile(const EngineParams& p, int id, int& b, int& I, int& J)
{
    const int tm = p.tiles_m, tn = p.tiles_n;
    switch (p.order) {
        case ORDER_COL: {
            const int per = tm * tn;
            b = id / per; const int r = id - b * per;
            J = r / tm; I = r - J * tm;
        } break;
        case ORDER_COL_REV: {
            const int per = tm * tn;
            b = id / per; const int r = id - b * per;
            J = r / tm; I = r - J * tm; J = tn - 1 - J;
        } break;
        case ORDER_ROW: {
            const int per = tm * tn;
            b = id / per; const int r = id - b * per;
            I = r / tn; J = r - I * tn;
        } break;
        case ORDER_ROW_REV: {
            const int per = tm * tn;
            b = id / per; const int r = id - b * per;
            I = r / tn; J = r - I * tn; I = tm - 1 - I;
        } break;
        case ORDER_TRAPEZOID: {
            const int per = tm * tn - tm * (tm - 1) / 2;
            b = id / per; int r = id - b * per;
            I = 0;
            while (r >= tn - I) { r -= tn - I; ++I; }
            J = I + r;
        } break;
        default: {
            // triangular enumerations over an n x n tile grid (n = tiles_n = tiles_m): group u has u+1 members.
            // With super-tiles the members are G x G squares of tiles: the ~1 wave of CTAs resident at a
            // time then shares 2G operand panels instead of G*G + 1, which is what keeps the operand
            // traffic in L2 (profiles/: DRAM bytes per launch).  Heavy tiles still come first.
            const int G = p.super > 1 ? p.super : 1;
            const int n = tn;
            const int ns = (n + G - 1) / G;
            const int per = ns * (ns + 1) / 2 * G * G;
            b = id / per; const int r0 = id - b * per;
            const int r = r0 / (G * G), t = r0 - r * (G * G);
            int u = static_cast<int>((sqrtf(8.0f * r + 1.0f) - 1.0f) * 0.5f);
            while ((u + 1) * (u + 2) / 2 <= r) ++u;
            while (u * (u + 1) / 2 > r) --u;
            const int v = r - u * (u + 1) / 2;   // 0..u
            int SI, SJ;
            if (p.order == ORDER_TRI_ROW_DESC) { SI = ns - 1 - u; SJ = SI + v; }
            else { const int d = ns - 1 - u; SI = v; SJ = v + d; }
            const int ti = t / G, tj = t - ti * G;
            I = SI * G + (p.order == ORDER_TRI_ROW_DESC ? G - 1 - ti : ti);
            J = SJ * G + (p.order == ORDER_TRI_ROW_DESC ? tj : G - 1 - tj);
            if (I > J || J >= n || I >= n) return false;
        } break;
    }
    return true;
}

// Zero / halve the part of an operand tile that lies below / on the global diagonal.
// k-contiguous tile: smem[x][k] (x = free index, 128 rows of 16 doubles), element (row=k0+k, col=x0+x).
// m-contiguous tile: 8 boxes [mb][k][16 m], element (row = x0 + 16*mb + m_in, col = k0 + k).
// The 128-byte swizzle permutes 16-byte chunks within a 128-byte row; masking works on logical
// coordinates and maps them to the swizzled address.
template <bool kMContig>
__device__ __forceinline__ void mask_tile(unsigned char* tile, int k0, int x0, bool half_diag, int ctid, bool lower = false)
{
    // 2048 elements, 256 consumer threads -> 8 elements (4 chunks of 2) per thread
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int chunk_lin = ctid + it * 256;          // 0..1023 : 16-byte chunk index in the tile
        const int row128 = chunk_lin >> 3;              // 128-byte row
        const int ch = chunk_lin & 7;                   // logical chunk within the row
        const int phys = ch ^ (row128 & 7);
        double2* ptr = reinterpret_cast<double2*>(tile + row128 * 128 + phys * 16);
        int grow0, gcol0, drow, dcol;                   // global coords of element 0 and the step to element 1
        if (!kMContig) { gcol0 = x0 + row128; grow0 = k0 + ch * 2; drow = 1; dcol = 0; }
        else { const int mb = row128 >> 4, k = row128 & 15; grow0 = x0 + mb * 16 + ch * 2; gcol0 = k0 + k; drow = 1; dcol = 0; }
        (void)dcol;
        if (lower) { const int t0 = grow0; grow0 = gcol0; gcol0 = t0; drow = -1; }   // compare (col, row): zero where row < col
        double2 v = *ptr;
        bool touched = false;
        if (grow0 > gcol0) { v.x = 0.0; touched = true; }
        else if (half_diag && grow0 == gcol0) { v.x *= 0.5; touched = true; }
        if (grow0 + drow > gcol0) { v.y = 0.0; touched = true; }
        else if (half_diag && grow0 + drow == gcol0) { v.y *= 0.5; touched = true; }
        if (touched) *ptr = v;
    }
}

// Non-TMA tile loaders (one warp): bounds-checked 8-byte global loads written into the same swizzled
// shared-memory layout the TMA path produces; out-of-range elements are zero, as TMA's OOB fill.
__device__ __forceinline__ void load_tile_kcontig(unsigned char* tile, const RawOperand& m, int k0, int x0, int lane)
{
    // element (k, x): global (row = k0 + k, col = x0 + x); smem offset x*128 + ((k>>1) ^ (x&7))*16 + (k&1)*8
    for (int idx = lane; idx < BM * BK; idx += 32) {
        const int x = idx >> 4, k = idx & 15;
        const long long row = k0 + k, col = x0 + x;
        double v = 0.0;
        if (row >= 0 && col >= 0 && row < m.rows && col < m.cols) v = m.ptr[row + col * m.ld];
        *reinterpret_cast<double*>(tile + x * 128 + (((k >> 1) ^ (x & 7)) * 16) + (k & 1) * 8) = v;
    }
}

__device__ __forceinline__ void load_tile_mcontig(unsigned char* tile, const RawOperand& m, int k0, int x0, int lane)
{
    // element (mm, k): global (row = x0 + mm, col = k0 + k); box mb = mm>>4, mi = mm&15:
    // smem offset mb*2048 + k*128 + ((mi>>1) ^ (k&7))*16 + (mi&1)*8
    for (int idx = lane; idx < BM * BK; idx += 32) {
        const int k = idx >> 7, mm = idx & 127;
        const int mb = mm >> 4, mi = mm & 15;
        const long long row = x0 + mm, col = k0 + k;
        double v = 0.0;
        if (row >= 0 && col >= 0 && row < m.rows && col < m.cols) v = m.ptr[row + col * m.ld];
        *reinterpret_cast<double*>(tile + mb * 2048 + k * 128 + (((mi >> 1) ^ (k & 7)) * 16) + (mi & 1) * 8) = v;
    }
}

template <bool kANN, bool kTMA>
__global__ void __launch_bounds__(kThreads, 1) tile_engine_kernel(const __grid_constant__ EngineParams p)
{
    extern __shared__ unsigned char smem_raw[];
    // 1024-byte alignment (128-byte swizzle atom = 8 rows x 128 B) without losing the shared address space
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes);
    const uint32_t full0 = smem_u32(bars);
    const uint32_t empty0 = smem_u32(bars + kStages);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    int b, I, J;
    if (!decode_tile(p, blockIdx.x, b, I, J)) return;
    if (p.c_row0 + (long long)b * p.c_brow + (long long)BM * I >= p.c_rows || p.c_col0 + (long long)b * p.c_bcol + (long long)BN * J >= p.c_cols)
        return;   // entirely outside the C bounds: nothing to store
    int k_lo = p.klo_c + p.klo_i * I + p.klo_j * J;
    int k_hi = p.khi_c + p.khi_i * I + p.khi_j * J;
    if (k_lo < 0) k_lo = 0;
    if (k_hi > p.kmax) k_hi = p.kmax;
    const int nk = k_hi > k_lo ? k_hi - k_lo : 0;
    const bool dual = (p.flags & F_DUAL) != 0;
    const int nsteps = dual ? 2 * nk : nk;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, kConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();
    // everything above touched only parameters and shared memory (ptx.cuh: programmatic dependent launch)
    grid_dep_launch();
    grid_dep_wait();
    if (p.info != nullptr && *p.info != 0) return;

    // global element coordinates of the operand tiles at k-step 0
    const int a_x = p.a.x0 + b * p.a.bx + BM * I, a_k = p.a.k0 + b * p.a.bk;
    const int b_x = p.b.x0 + b * p.b.bx + BN * J, b_k = p.b.k0 + b * p.b.bk;
    const int a2_x = p.a2.x0 + b * p.a2.bx + BM * I, a2_k = p.a2.k0 + b * p.a2.bk;
    const int b2_x = p.b2.x0 + b * p.b2.bx + BN * J, b2_k = p.b2.k0 + b * p.b2.bk;

    if (warp == kConsumerWarps) {
        if (!kTMA) {
            // ===================== plain-load producer (whole warp) =====================
            for (int s = 0; s < nsteps; ++s) {
                const int stage = s % kStages;
                const uint32_t ph = (s / kStages) & 1;
                mbar_wait(empty0 + 8 * stage, ph ^ 1);
                unsigned char* st = smem + stage * kStageBytes;
                const bool second = dual && (s & 1);
                const int kt = k_lo + (dual ? (s >> 1) : s);
                const RawOperand& rA = second ? p.rawA2 : p.rawA;
                const RawOperand& rB = second ? p.rawB2 : p.rawB;
                const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * BK;
                const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * BK;
                if (kANN) load_tile_mcontig(st, rA, ak, ax, lane);
                else load_tile_kcontig(st, rA, ak, ax, lane);
                load_tile_kcontig(st + kTileBytes, rB, bk, bx, lane);
                __syncwarp();
                if (lane == 0) mbar_arrive(full0 + 8 * stage);
            }
            return;
        }
        // ===================== TMA producer (one elected lane) =====================
        if (lane == 0) {
            tma_prefetch_desc(&p.mapA);
            tma_prefetch_desc(&p.mapB);
            if (dual) { tma_prefetch_desc(&p.mapA2); tma_prefetch_desc(&p.mapB2); }
            for (int s = 0; s < nsteps; ++s) {
                const int stage = s % kStages;
                const uint32_t ph = (s / kStages) & 1;
                mbar_wait(empty0 + 8 * stage, ph ^ 1);
                const uint32_t full = full0 + 8 * stage;
                mbar_arrive_expect_tx(full, kStageBytes);
                const uint32_t dstA = smem_u32(smem + stage * kStageBytes);
                const uint32_t dstB = dstA + kTileBytes;
                const bool second = dual && (s & 1);
                const int kt = k_lo + (dual ? (s >> 1) : s);
                const CUtensorMap* mA = second ? &p.mapA2 : &p.mapA;
                const CUtensorMap* mB = second ? &p.mapB2 : &p.mapB;
                const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * BK;
                const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * BK;
                if (kANN) {
#pragma unroll
                    for (int mb = 0; mb < BM / 16; ++mb)
                        tma_load_2d(dstA + mb * 2048, mA, ax + mb * 16, ak, full);
                } else {
                    tma_load_2d(dstA, mA, ak, ax, full);
                }
                tma_load_2d(dstB, mB, bk, bx, full);
            }
        }
        return;
    }

    // ===================== consumers: 8 warps, 4 (m) x 2 (n), warp tile 32 x 64 =====================
    const int wm = warp & 3, wn = warp >> 2;
    const int g = lane >> 2, q = lane & 3;
    const int rho = (g >> 1) + 4 * (g & 1);   // logical row within an 8-row group for k-contiguous operands

    // C tile coordinates of this thread's accumulators (fragment row g of m-group mg, fragment
    // columns 2q+e of n-group ng; the column was supplied by the B-lane with g' = 2q+e -> n = rho(g'))
    const long long crow0 = p.c_row0 + (long long)b * p.c_brow + (long long)BM * I + wm * 32;
    const long long ccol0 = p.c_col0 + (long long)b * p.c_bcol + (long long)BN * J + wn * 64;
    const bool upper_only = (p.flags & F_STORE_UPPER) != 0;
    const double alpha = p.alpha, beta = p.beta;
    auto c_row = [&](int mg) -> long long {
        return crow0 + (kANN ? ((mg >> 1) * 16 + 2 * g + (mg & 1)) : (mg * 8 + rho));
    };
    auto c_col = [&](int ng, int e) -> long long {
        const int gp = 2 * q + e;
        return ccol0 + ng * 8 + ((gp >> 1) + 4 * (gp & 1));
    };

    // beta != 0: the accumulators start from (beta/alpha) * C, so the loads of the C tile overlap
    // the pipeline fill instead of forming a dependent load-FMA-store chain in the epilogue.
    double acc[4][8][2];
    if (beta != 0.0) {
        const double sc = beta / alpha;
#pragma unroll
        for (int mg = 0; mg < 4; ++mg) {
            const long long row = c_row(mg);
#pragma unroll
            for (int ng = 0; ng < 8; ++ng)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long long col = c_col(ng, e);
                    const bool ok = row < p.c_rows && col < p.c_cols && (!upper_only || row <= col);
                    acc[mg][ng][e] = ok ? sc * __ldg(p.C + row + col * p.ldc) : 0.0;
                }
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
    }

    // per-thread byte offsets inside a stage (k8-step h = 0); h = 1 is offset ^ 64 (k-contig) / + 1024 (m-contig)
    const uint32_t offB = kTileBytes + (wn * 64 + rho) * 128 + ((q ^ rho) * 16);
    uint32_t offA0, offA1;
    if (kANN) {
        // box mb = wm*2 + {0,1}; row k = 2q + a; chunk g ^ (2q + a)
        offA0 = (wm * 2) * 2048 + (2 * q) * 128 + ((g ^ (2 * q)) * 16);
        offA1 = (wm * 2) * 2048 + (2 * q + 1) * 128 + ((g ^ (2 * q + 1)) * 16);
    } else {
        offA0 = (wm * 32 + rho) * 128 + ((q ^ rho) * 16);
        offA1 = 0;
    }
    const uint32_t mask_any = p.flags & (F_MASK_A | F_MASK_B | F_MASK_A2 | F_MASK_B2);
    const int ctid = threadIdx.x;   // 0..255 for consumers

    for (int s = 0; s < nsteps; ++s) {
        const int stage = s % kStages;
        const uint32_t ph = (s / kStages) & 1;
        mbar_wait(full0 + 8 * stage, ph);
        release_previous_stage(s, kStages, empty0, lane);
        unsigned char* st = smem + stage * kStageBytes;

        if (mask_any) {
            const bool second = dual && (s & 1);
            const int kt = k_lo + (dual ? (s >> 1) : s);
            const bool mA = (p.flags & (second ? F_MASK_A2 : F_MASK_A)) != 0;
            const bool mB = (p.flags & (second ? F_MASK_B2 : F_MASK_B)) != 0;
            const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * BK;
            const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * BK;
            bool did = false;
            if (mA) {
                // A element global (row, col): NN: (ax + m, ak + k); TN: (ak + k, ax + m)
                const bool lowerA = !second && (p.flags & F_LOWER_A) != 0;
                const bool straddle = lowerA ? (kANN ? (ax <= ak + BK - 1) : (ak <= ax + BM - 1))
                                             : (kANN ? (ax + BM - 1 >= ak) : (ak + BK - 1 >= ax));
                if (straddle) {
                    mask_tile<kANN>(st, ak, ax, !second && (p.flags & F_HALF_DIAG_A), ctid, lowerA);
                    did = true;
                }
            }
            if (mB) {
                if (bk + BK - 1 >= bx) { mask_tile<false>(st + kTileBytes, bk, bx, false, ctid); did = true; }
            }
            if (did) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                named_bar_sync(1, kConsumerWarps * 32);
            }
        }

#pragma unroll
        for (int h = 0; h < 2; ++h) {
            double af[4][2];
            if (kANN) {
#pragma unroll
                for (int mb = 0; mb < 2; ++mb) {
                    const double2 v0 = *reinterpret_cast<const double2*>(st + offA0 + mb * 2048 + h * 1024);
                    const double2 v1 = *reinterpret_cast<const double2*>(st + offA1 + mb * 2048 + h * 1024);
                    af[mb * 2 + 0][0] = v0.x; af[mb * 2 + 1][0] = v0.y;
                    af[mb * 2 + 0][1] = v1.x; af[mb * 2 + 1][1] = v1.y;
                }
            } else {
#pragma unroll
                for (int mg = 0; mg < 4; ++mg) {
                    const double2 v = *reinterpret_cast<const double2*>(st + ((offA0 + mg * 1024) ^ (h * 64)));
                    af[mg][0] = v.x; af[mg][1] = v.y;
                }
            }
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                double bf[4][2];
#pragma unroll
                for (int ng = 0; ng < 4; ++ng) {
                    const double2 v = *reinterpret_cast<const double2*>(st + ((offB + (half * 4 + ng) * 1024) ^ (h * 64)));
                    bf[ng][0] = v.x; bf[ng][1] = v.y;
                }
#pragma unroll
                for (int kk = 0; kk < 2; ++kk)
#pragma unroll
                    for (int mg = 0; mg < 4; ++mg)
#pragma unroll
                        for (int ng = 0; ng < 4; ++ng)
                            dmma_8x8x4(acc[mg][half * 4 + ng][0], acc[mg][half * 4 + ng][1], af[mg][kk], bf[ng][kk]);
            }
        }
    }

    // ===================== epilogue: C = alpha * acc (predicated, direct to global) =====================
    // (+ fused exchange: the same element to every push target whose column filter it passes)
    const int npeer = p.npeer;
#pragma unroll
    for (int mg = 0; mg < 4; ++mg) {
        const long long row = c_row(mg);
#pragma unroll
        for (int ng = 0; ng < 8; ++ng) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const long long col = c_col(ng, e);
                if (row < p.c_rows && col < p.c_cols && (!upper_only || row <= col)) {
                    const long long off = row + col * p.ldc;
                    const double v = alpha * acc[mg][ng][e];
                    p.C[off] = v;
                    if (npeer > 0 && col >= p.peer_col0)
                        for (int d = 0; d < npeer; ++d) p.peer[d][off] = v;
                }
            }
        }
    }
}

}  // namespace gs
