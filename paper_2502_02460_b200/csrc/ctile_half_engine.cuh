// ctile_half_engine.cuh -- the complex128 tile engine with 64 x 32 CTA tiles: every 64 x 64 logical tile
// of ctile_engine.cuh (same EngineParams, flags, orders, k-ranges) is computed by TWO CTAs, one per
// 32-column half.  Same reasoning as tile64_engine.cuh for the real path: half the accumulators per
// thread (32 FP64 = warp tile 32 x 16 complex) bring the kernel to 128 registers and 5 x 12 KB stages,
// so THREE CTAs share an SM instead of two, and a one-tile launch of the POTRF chain finishes in half
// the time on two SMs.  A CTA reads all k-rows of its own column strip only, so the in-place one-tile
// solve (C aliases B) stays legal.
#pragma once
#include "ctile_engine.cuh"

namespace gs {

constexpr int kHStages = 5;
constexpr int kHBTileBytes = 32 * CBK * 16;                 // 4 KB: the B operand tile of one 32-column half
constexpr int kHStageBytes = kCTileBytes + kHBTileBytes;    // 12 KB
constexpr int kHSmemBytes = kHStages * kHStageBytes + 1024 /*align*/ + 256 /*barriers*/;

// upper-triangular mask of the 32-row k-contiguous B tile (256 complex elements, 128 consumer threads)
__device__ __forceinline__ void mask_ctile_half_b(unsigned char* tile, int k0, int x0, int ctid)
{
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const int chunk_lin = ctid + it * 128;          // 0..255
        const int row128 = chunk_lin >> 3;
        const int ch = chunk_lin & 7;
        const int phys = ch ^ (row128 & 7);
        if (k0 + ch > x0 + row128) *reinterpret_cast<double2*>(tile + row128 * 128 + phys * 16) = make_double2(0.0, 0.0);
    }
}

template <bool kANN>
__global__ void __launch_bounds__(kCThreads, 3) ctile_half_engine_kernel(const __grid_constant__ EngineParams p)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kHStages * kHStageBytes);
    const uint32_t full0 = smem_u32(bars);
    const uint32_t empty0 = smem_u32(bars + kHStages);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    int b, I, J;
    if (!decode_tile(p, blockIdx.x >> 1, b, I, J)) return;
    const int qj = blockIdx.x & 1;   // which 32-column half of the logical 64 x 64 tile
    if (p.c_row0 + (long long)b * p.c_brow + (long long)CT * I >= p.c_rows ||
        p.c_col0 + (long long)b * p.c_bcol + (long long)CT * J + 32 * qj >= p.c_cols)
        return;   // entirely outside the C bounds: nothing to store
    int k_lo = p.klo_c + p.klo_i * I + p.klo_j * J;
    int k_hi = p.khi_c + p.khi_i * I + p.khi_j * J;
    if (k_lo < 0) k_lo = 0;
    if (k_hi > p.kmax) k_hi = p.kmax;
    const int nk = k_hi > k_lo ? k_hi - k_lo : 0;
    const bool dual = (p.flags & F_DUAL) != 0;
    const int nsteps = dual ? 2 * nk : nk;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kHStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, kCConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();
    // everything above touched only parameters and shared memory (ptx.cuh: programmatic dependent launch)
    grid_dep_launch();
    grid_dep_wait();
    if (p.info != nullptr && *p.info != 0) return;

    // element coordinates (complex elements) of the operand tiles at k-step 0
    const int a_x = p.a.x0 + b * p.a.bx + CT * I, a_k = p.a.k0 + b * p.a.bk;
    const int b_x = p.b.x0 + b * p.b.bx + CT * J + 32 * qj, b_k = p.b.k0 + b * p.b.bk;
    const int a2_x = p.a2.x0 + b * p.a2.bx + CT * I, a2_k = p.a2.k0 + b * p.a2.bk;
    const int b2_x = p.b2.x0 + b * p.b2.bx + CT * J + 32 * qj, b2_k = p.b2.k0 + b * p.b2.bk;

    if (warp == kCConsumerWarps) {
        // ===================== TMA producer (one elected lane) =====================
        if (lane == 0) {
            tma_prefetch_desc(&p.mapA);
            tma_prefetch_desc(&p.mapB);
            if (dual) { tma_prefetch_desc(&p.mapA2); tma_prefetch_desc(&p.mapB2); }
            for (int s = 0; s < nsteps; ++s) {
                const int stage = s % kHStages;
                const uint32_t ph = (s / kHStages) & 1;
                mbar_wait(empty0 + 8 * stage, ph ^ 1);
                const uint32_t full = full0 + 8 * stage;
                mbar_arrive_expect_tx(full, kHStageBytes);
                const uint32_t dstA = smem_u32(smem + stage * kHStageBytes);
                const uint32_t dstB = dstA + kCTileBytes;
                const bool second = dual && (s & 1);
                const int kt = k_lo + (dual ? (s >> 1) : s);
                const CUtensorMap* mA = second ? &p.mapA2 : &p.mapA;
                const CUtensorMap* mB = second ? &p.mapB2 : &p.mapB;
                const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * CBK;
                const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * CBK;
                // the tensor maps see the matrix as doubles: contiguous coordinate = 2 x complex index
                if (kANN) {
#pragma unroll
                    for (int mb = 0; mb < CT / 8; ++mb)
                        tma_load_2d(dstA + mb * 1024, mA, 2 * (ax + mb * 8), ak, full);
                } else {
                    tma_load_2d(dstA, mA, 2 * ak, ax, full);
                }
                tma_load_2d(dstB, mB, 2 * bk, bx, full);
            }
        }
        return;
    }

    // ===================== consumers: 4 warps, 2 (m) x 2 (n), warp tile 32 x 16 complex =====================
    const int wm = warp & 1, wn = warp >> 1;
    const int g = lane >> 2, q = lane & 3;
    const int rho = (g >> 1) + 4 * (g & 1);   // logical row within an 8-row group (conflict-free LDS.128)

    const long long crow0 = p.c_row0 + (long long)b * p.c_brow + (long long)CT * I + wm * 32;
    const long long ccol0 = p.c_col0 + (long long)b * p.c_bcol + (long long)CT * J + 32 * qj + wn * 16;
    const bool upper_only = (p.flags & F_STORE_UPPER) != 0;
    const bool real_diag = (p.flags & F_REAL_DIAG) != 0;
    const double alpha = p.alpha, beta = p.beta;
    double2* Cz = reinterpret_cast<double2*>(p.C);
    auto c_row = [&](int mg) -> long long { return crow0 + mg * 8 + rho; };
    auto c_col = [&](int ng, int e) -> long long {
        const int gp = 2 * q + e;
        return ccol0 + ng * 8 + ((gp >> 1) + 4 * (gp & 1));
    };

    double acc[4][2][2][2];   // [mg][ng][fragment column e][re, im]
    if (beta != 0.0) {
        const double sc = beta / alpha;
#pragma unroll
        for (int mg = 0; mg < 4; ++mg) {
            const long long row = c_row(mg);
#pragma unroll
            for (int ng = 0; ng < 2; ++ng)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long long col = c_col(ng, e);
                    const bool ok = row < p.c_rows && col < p.c_cols && (!upper_only || row <= col);
                    double2 v = make_double2(0.0, 0.0);
                    if (ok) v = __ldcg(Cz + row + col * p.ldc);
                    acc[mg][ng][e][0] = sc * v.x;
                    acc[mg][ng][e][1] = sc * v.y;
                }
        }
    } else {
#pragma unroll
        for (int mg = 0; mg < 4; ++mg)
#pragma unroll
            for (int ng = 0; ng < 2; ++ng)
#pragma unroll
                for (int e = 0; e < 2; ++e) { acc[mg][ng][e][0] = 0.0; acc[mg][ng][e][1] = 0.0; }
    }

    // per-thread byte offsets inside a stage at k4-step h = 0
    const uint32_t offB = kCTileBytes + (wn * 16 + rho) * 128 + ((q ^ rho) * 16);
    uint32_t offA;
    if (kANN) offA = (wm * 4) * 1024 + q * 128 + ((rho ^ q) * 16);   // box wm*4+mg, row k = q (+4h), chunk rho ^ k
    else offA = (wm * 32 + rho) * 128 + ((q ^ rho) * 16);            // row x = wm*32 + mg*8 + rho, chunk k ^ rho
    const uint32_t mask_any = p.flags & (F_MASK_A | F_MASK_B | F_MASK_A2 | F_MASK_B2);
    const int ctid = threadIdx.x;   // 0..127 for consumers

    for (int s = 0; s < nsteps; ++s) {
        const int stage = s % kHStages;
        const uint32_t ph = (s / kHStages) & 1;
        mbar_wait(full0 + 8 * stage, ph);
        release_previous_stage(s, kHStages, empty0, lane);
        unsigned char* st = smem + stage * kHStageBytes;

        if (mask_any) {
            const bool second = dual && (s & 1);
            const int kt = k_lo + (dual ? (s >> 1) : s);
            const bool mA = (p.flags & (second ? F_MASK_A2 : F_MASK_A)) != 0;
            const bool mB = (p.flags & (second ? F_MASK_B2 : F_MASK_B)) != 0;
            const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * CBK;
            const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * CBK;
            bool did = false;
            if (mA) {
                const bool lowerA = !second && (p.flags & F_LOWER_A) != 0;
                const bool straddle = lowerA ? (kANN ? (ax <= ak + CBK - 1) : (ak <= ax + CT - 1))
                                             : (kANN ? (ax + CT - 1 >= ak) : (ak + CBK - 1 >= ax));
                if (straddle) {
                    mask_ctile<kANN>(st, ak, ax, !second && (p.flags & F_HALF_DIAG_A), ctid, lowerA);
                    did = true;
                }
            }
            if (mB) {
                if (bk + CBK - 1 >= bx) { mask_ctile_half_b(st + kCTileBytes, bk, bx, ctid); did = true; }
            }
            if (did) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                named_bar_sync(1, kCConsumerWarps * 32);
            }
        }

#pragma unroll
        for (int h = 0; h < 2; ++h) {
            double ar[4], a2[4], a3[4];
#pragma unroll
            for (int mg = 0; mg < 4; ++mg) {
                const uint32_t off = kANN ? ((offA + mg * 1024 + h * 512) ^ (h * 64)) : ((offA + mg * 1024) ^ (h * 64));
                const double2 v = *reinterpret_cast<const double2*>(st + off);
                ar[mg] = v.x;
                // TN = conjugate transpose: (ar - i ai)(br + i bi) = (ar br + ai bi) + i (ar bi - ai br)
                a2[mg] = kANN ? -v.y : v.y;    // multiplies bi into the real part
                a3[mg] = kANN ? v.y : -v.y;    // multiplies br into the imaginary part
            }
            double2 bf[2];
#pragma unroll
            for (int ng = 0; ng < 2; ++ng)
                bf[ng] = *reinterpret_cast<const double2*>(st + ((offB + ng * 1024) ^ (h * 64)));
#pragma unroll
            for (int mg = 0; mg < 4; ++mg)
#pragma unroll
                for (int ng = 0; ng < 2; ++ng) {
                    dmma_8x8x4(acc[mg][ng][0][0], acc[mg][ng][1][0], ar[mg], bf[ng].x);
                    dmma_8x8x4(acc[mg][ng][0][1], acc[mg][ng][1][1], ar[mg], bf[ng].y);
                    dmma_8x8x4(acc[mg][ng][0][0], acc[mg][ng][1][0], a2[mg], bf[ng].y);
                    dmma_8x8x4(acc[mg][ng][0][1], acc[mg][ng][1][1], a3[mg], bf[ng].x);
                }
        }
    }

    // ===================== epilogue: C = alpha * acc (predicated 16-byte stores) =====================
#pragma unroll
    for (int mg = 0; mg < 4; ++mg) {
        const long long row = c_row(mg);
#pragma unroll
        for (int ng = 0; ng < 2; ++ng)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const long long col = c_col(ng, e);
                if (row < p.c_rows && col < p.c_cols && (!upper_only || row <= col)) {
                    double2 v = make_double2(alpha * acc[mg][ng][e][0], alpha * acc[mg][ng][e][1]);
                    if (real_diag && row == col) v.y = 0.0;
                    Cz[row + col * p.ldc] = v;
                }
            }
    }
    for (int d = 0; d < p.npeer; ++d) {   // fused exchange (tile_engine.cuh: EngineParams::peer)
        double2* Cd = reinterpret_cast<double2*>(p.peer[d]);
#pragma unroll
        for (int mg = 0; mg < 4; ++mg) {
            const long long row = c_row(mg);
#pragma unroll
            for (int ng = 0; ng < 2; ++ng)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long long col = c_col(ng, e);
                    if (row < p.c_rows && col < p.c_cols && col >= p.peer_col0 && (!upper_only || row <= col)) {
                        double2 v = make_double2(alpha * acc[mg][ng][e][0], alpha * acc[mg][ng][e][1]);
                        if (real_diag && row == col) v.y = 0.0;
                        Cd[row + col * p.ldc] = v;
                    }
                }
        }
    }
}

}  // namespace gs
