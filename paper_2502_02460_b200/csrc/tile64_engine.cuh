// tile64_engine.cuh -- the real-FP64 tile engine with 64 x 64 CTA tiles: every 128 x 128 logical tile of
// tile_engine.cuh (same EngineParams, flags, orders, k-ranges) is computed by 2 x 2 CTAs.
//
// Why a second tile size: a 128 x 128 x 128 block product occupies ONE SM for 17 us, and the POTRF
// panel chain is made of launches with 1-10 such tiles -- four 64 x 64 CTAs finish the same product in
// a quarter of the time on four SMs.  And with 4 consumer warps + 1 TMA warp, ~100 registers and
// 4 x 16 KB stages, three CTAs share an SM (three warps per sub-partition instead of two), which hides
// fragment-load latency and one CTA's prologue / epilogue under the others' main loops.  The price is
// twice the operand traffic from L2 per flop (16 instead of 8 B/clk/SM).
//
// Layouts and fragment mappings are those of tile_engine.cuh restricted to a 32 x 32 warp tile.
#pragma once
#include "tile_engine.cuh"

namespace gs {

constexpr int T64 = 64;
constexpr int k64Stages = 4;
constexpr int k64ConsumerWarps = 4;
constexpr int k64Threads = (k64ConsumerWarps + 1) * 32;
constexpr int k64TileBytes = T64 * BK * 8;                  // 8 KB per operand tile
constexpr int k64StageBytes = 2 * k64TileBytes;             // A + B
constexpr int k64SmemBytes = k64Stages * k64StageBytes + 1024 /*align*/ + 256 /*barriers*/;

// mask_tile of tile_engine.cuh for a 64-wide operand tile (512 16-byte chunks, 128 consumer threads)
template <bool kMContig>
__device__ __forceinline__ void mask_tile64(unsigned char* tile, int k0, int x0, bool half_diag, int ctid, bool lower)
{
#pragma unroll
    for (int it = 0; it < 4; ++it) {
        const int chunk_lin = ctid + it * 128;          // 0..511
        const int row128 = chunk_lin >> 3;
        const int ch = chunk_lin & 7;
        const int phys = ch ^ (row128 & 7);
        double2* ptr = reinterpret_cast<double2*>(tile + row128 * 128 + phys * 16);
        int grow0, gcol0, drow = 1;
        if (!kMContig) { gcol0 = x0 + row128; grow0 = k0 + ch * 2; }
        else { const int mb = row128 >> 4, k = row128 & 15; grow0 = x0 + mb * 16 + ch * 2; gcol0 = k0 + k; }
        if (lower) { const int t0 = grow0; grow0 = gcol0; gcol0 = t0; drow = -1; }
        double2 v = *ptr;
        bool touched = false;
        if (grow0 > gcol0) { v.x = 0.0; touched = true; }
        else if (half_diag && grow0 == gcol0) { v.x *= 0.5; touched = true; }
        if (grow0 + drow > gcol0) { v.y = 0.0; touched = true; }
        else if (half_diag && grow0 + drow == gcol0) { v.y *= 0.5; touched = true; }
        if (touched) *ptr = v;
    }
}

template <bool kANN>
__global__ void __launch_bounds__(k64Threads, 3) tile64_engine_kernel(const __grid_constant__ EngineParams p)
{
    extern __shared__ unsigned char smem_raw[];
    unsigned char* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + k64Stages * k64StageBytes);
    const uint32_t full0 = smem_u32(bars);
    const uint32_t empty0 = smem_u32(bars + k64Stages);

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;

    // logical 128-tile (b, I, J) and the 64 x 64 quarter (qi, qj) of it this CTA computes
    int b, I, J;
    if (!decode_tile(p, blockIdx.x >> 2, b, I, J)) return;
    const int qi = blockIdx.x & 1, qj = (blockIdx.x >> 1) & 1;
    // a tile that lies entirely outside the C bounds stores nothing: skip it (batched launches over a matrix whose
    // block count is not a power of two -- the doubling levels of the triangular inversion -- have many of them)
    if (p.c_row0 + (long long)b * p.c_brow + (long long)BM * I + T64 * qi >= p.c_rows ||
        p.c_col0 + (long long)b * p.c_bcol + (long long)BN * J + T64 * qj >= p.c_cols)
        return;
    int k_lo = p.klo_c + p.klo_i * I + p.klo_j * J;
    int k_hi = p.khi_c + p.khi_i * I + p.khi_j * J;
    if (k_lo < 0) k_lo = 0;
    if (k_hi > p.kmax) k_hi = p.kmax;
    const int nk = k_hi > k_lo ? k_hi - k_lo : 0;
    const bool dual = (p.flags & F_DUAL) != 0;
    const int nsteps = dual ? 2 * nk : nk;

    if (threadIdx.x == 0) {
        for (int s = 0; s < k64Stages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, k64ConsumerWarps);
        }
        mbar_fence_init();
    }
    __syncthreads();
    grid_dep_launch();
    grid_dep_wait();
    if (p.info != nullptr && *p.info != 0) return;

    const int a_x = p.a.x0 + b * p.a.bx + BM * I + T64 * qi, a_k = p.a.k0 + b * p.a.bk;
    const int b_x = p.b.x0 + b * p.b.bx + BN * J + T64 * qj, b_k = p.b.k0 + b * p.b.bk;
    const int a2_x = p.a2.x0 + b * p.a2.bx + BM * I + T64 * qi, a2_k = p.a2.k0 + b * p.a2.bk;
    const int b2_x = p.b2.x0 + b * p.b2.bx + BN * J + T64 * qj, b2_k = p.b2.k0 + b * p.b2.bk;

    if (warp == k64ConsumerWarps) {
        // ===================== TMA producer (one elected lane) =====================
        if (lane == 0) {
            tma_prefetch_desc(&p.mapA);
            tma_prefetch_desc(&p.mapB);
            if (dual) { tma_prefetch_desc(&p.mapA2); tma_prefetch_desc(&p.mapB2); }
            for (int s = 0; s < nsteps; ++s) {
                const int stage = s % k64Stages;
                const uint32_t ph = (s / k64Stages) & 1;
                mbar_wait(empty0 + 8 * stage, ph ^ 1);
                const uint32_t full = full0 + 8 * stage;
                mbar_arrive_expect_tx(full, k64StageBytes);
                const uint32_t dstA = smem_u32(smem + stage * k64StageBytes);
                const uint32_t dstB = dstA + k64TileBytes;
                const bool second = dual && (s & 1);
                const int kt = k_lo + (dual ? (s >> 1) : s);
                const CUtensorMap* mA = second ? &p.mapA2 : &p.mapA;
                const CUtensorMap* mB = second ? &p.mapB2 : &p.mapB;
                const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * BK;
                const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * BK;
                if (kANN) {
#pragma unroll
                    for (int mb = 0; mb < T64 / 16; ++mb)
                        tma_load_2d(dstA + mb * 2048, mA, ax + mb * 16, ak, full);   // 16 x 16 boxes
                } else {
                    tma_load_2d(dstA, mA, ak, ax, full);                              // 16 x 64 box (maps are encoded for this engine)
                }
                tma_load_2d(dstB, mB, bk, bx, full);
            }
        }
        return;
    }

    // ===================== consumers: 4 warps, 2 (m) x 2 (n), warp tile 32 x 32 =====================
    const int wm = warp & 1, wn = warp >> 1;
    const int g = lane >> 2, q = lane & 3;
    const int rho = (g >> 1) + 4 * (g & 1);

    const long long crow0 = p.c_row0 + (long long)b * p.c_brow + (long long)BM * I + T64 * qi + wm * 32;
    const long long ccol0 = p.c_col0 + (long long)b * p.c_bcol + (long long)BN * J + T64 * qj + wn * 32;
    const bool upper_only = (p.flags & F_STORE_UPPER) != 0;
    const double alpha = p.alpha, beta = p.beta;
    auto c_row = [&](int mg) -> long long {
        return crow0 + (kANN ? ((mg >> 1) * 16 + 2 * g + (mg & 1)) : (mg * 8 + rho));
    };
    auto c_col = [&](int ng, int e) -> long long {
        const int gp = 2 * q + e;
        return ccol0 + ng * 8 + ((gp >> 1) + 4 * (gp & 1));
    };

    double acc[4][4][2];
    if (beta != 0.0) {
        const double sc = beta / alpha;
#pragma unroll
        for (int mg = 0; mg < 4; ++mg) {
            const long long row = c_row(mg);
#pragma unroll
            for (int ng = 0; ng < 4; ++ng)
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
            for (int j = 0; j < 4; ++j) { acc[i][j][0] = 0.0; acc[i][j][1] = 0.0; }
    }

    const uint32_t offB = k64TileBytes + (wn * 32 + rho) * 128 + ((q ^ rho) * 16);
    uint32_t offA0, offA1;
    if (kANN) {
        offA0 = (wm * 2) * 2048 + (2 * q) * 128 + ((g ^ (2 * q)) * 16);
        offA1 = (wm * 2) * 2048 + (2 * q + 1) * 128 + ((g ^ (2 * q + 1)) * 16);
    } else {
        offA0 = (wm * 32 + rho) * 128 + ((q ^ rho) * 16);
        offA1 = 0;
    }
    const uint32_t mask_any = p.flags & (F_MASK_A | F_MASK_B | F_MASK_A2 | F_MASK_B2);
    const int ctid = threadIdx.x;   // 0..127 for consumers

    for (int s = 0; s < nsteps; ++s) {
        const int stage = s % k64Stages;
        const uint32_t ph = (s / k64Stages) & 1;
        mbar_wait(full0 + 8 * stage, ph);
        release_previous_stage(s, k64Stages, empty0, lane);
        unsigned char* st = smem + stage * k64StageBytes;

        if (mask_any) {
            const bool second = dual && (s & 1);
            const int kt = k_lo + (dual ? (s >> 1) : s);
            const bool mA = (p.flags & (second ? F_MASK_A2 : F_MASK_A)) != 0;
            const bool mB = (p.flags & (second ? F_MASK_B2 : F_MASK_B)) != 0;
            const int ax = second ? a2_x : a_x, ak = (second ? a2_k : a_k) + kt * BK;
            const int bx = second ? b2_x : b_x, bk = (second ? b2_k : b_k) + kt * BK;
            bool did = false;
            if (mA) {
                const bool lowerA = !second && (p.flags & F_LOWER_A) != 0;
                const bool straddle = lowerA ? (kANN ? (ax <= ak + BK - 1) : (ak <= ax + T64 - 1))
                                             : (kANN ? (ax + T64 - 1 >= ak) : (ak + BK - 1 >= ax));
                if (straddle) {
                    mask_tile64<kANN>(st, ak, ax, !second && (p.flags & F_HALF_DIAG_A), ctid, lowerA);
                    did = true;
                }
            }
            if (mB) {
                if (bk + BK - 1 >= bx) { mask_tile64<false>(st + k64TileBytes, bk, bx, false, ctid, false); did = true; }
            }
            if (did) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                named_bar_sync(1, k64ConsumerWarps * 32);
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
            double bf[4][2];
#pragma unroll
            for (int ng = 0; ng < 4; ++ng) {
                const double2 v = *reinterpret_cast<const double2*>(st + ((offB + ng * 1024) ^ (h * 64)));
                bf[ng][0] = v.x; bf[ng][1] = v.y;
            }
#pragma unroll
            for (int kk = 0; kk < 2; ++kk)
#pragma unroll
                for (int mg = 0; mg < 4; ++mg)
#pragma unroll
                    for (int ng = 0; ng < 4; ++ng)
                        dmma_8x8x4(acc[mg][ng][0], acc[mg][ng][1], af[mg][kk], bf[ng][kk]);
        }
    }

    // ===================== epilogue: C = alpha * acc =====================
#pragma unroll
    for (int mg = 0; mg < 4; ++mg) {
        const long long row = c_row(mg);
#pragma unroll
        for (int ng = 0; ng < 4; ++ng)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const long long col = c_col(ng, e);
                if (row < p.c_rows && col < p.c_cols && (!upper_only || row <= col))
                    p.C[row + col * p.ldc] = alpha * acc[mg][ng][e];
            }
    }
    for (int d = 0; d < p.npeer; ++d) {   // fused exchange (tile_engine.cuh: EngineParams::peer)
        double* Cd = p.peer[d];
#pragma unroll
        for (int mg = 0; mg < 4; ++mg) {
            const long long row = c_row(mg);
#pragma unroll
            for (int ng = 0; ng < 4; ++ng)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const long long col = c_col(ng, e);
                    if (row < p.c_rows && col < p.c_cols && col >= p.peer_col0 && (!upper_only || row <= col))
                        Cd[row + col * p.ldc] = alpha * acc[mg][ng][e];
                }
        }
    }
}

}  // namespace gs
