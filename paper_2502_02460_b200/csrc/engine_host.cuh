// engine_host.cuh -- host side of the tile engine: TMA descriptor construction and launch.
#pragma once
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>

#include <cstring>
#include <mutex>

#include "ctile_engine.cuh"
#include "ctile_half_engine.cuh"
#include "tile64_engine.cuh"
#include "tile_engine.cuh"

namespace gs {

// cuTensorMapEncodeTiled is a driver-API entry point; fetch it through the runtime so libgs does
// not link libcuda directly.
inline PFN_cuTensorMapEncodeTiled tensor_map_encoder()
{
    static std::once_flag once;
    static PFN_cuTensorMapEncodeTiled fn = nullptr;
    std::call_once(once, [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_cuTensorMapEncodeTiled>(p);
    });
    return fn;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is a PER-DEVICE setting: a process that creates plans on
// several devices (gs.Plan(device=...), Batch(device=...)) must opt in on each of them.  `configure` runs once
// per (caller-supplied state, current device), under a mutex (plans may be used from several host threads).
constexpr int kMaxDevices = 64;
struct PerDeviceOnce {
    std::mutex mu;
    bool done[kMaxDevices] = {};
    template <typename F>
    cudaError_t run(F&& configure)
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        std::lock_guard<std::mutex> lock(mu);
        if (dev >= 0 && dev < kMaxDevices && done[dev]) return cudaSuccess;
        e = configure();
        if (e == cudaSuccess && dev >= 0 && dev < kMaxDevices) done[dev] = true;
        return e;
    }
};

// Column-major FP64 matrix view: rows x cols, leading dimension ld (elements).  TMA needs a
// 16-byte aligned base and a row pitch that is a multiple of 16 bytes (even ld).
// (complex128: interleaved (re, im); rows, cols, ld count complex elements.)
struct MatView {
    const void* ptr;
    long long rows, cols, ld;
};

inline bool tma_compatible(const MatView& m)
{
    return (reinterpret_cast<uintptr_t>(m.ptr) % 16 == 0) && (m.ld % 2 == 0);
}

// box = box_rows (contiguous dim, always 16 doubles = 128 B) x box_cols
// A complex matrix is described to TMA as a 2*rows x cols FP64 matrix.
inline bool make_tensor_map(CUtensorMap* out, const MatView& m, int box_cols, bool cplx)
{
    PFN_cuTensorMapEncodeTiled enc = tensor_map_encoder();
    if (enc == nullptr) return false;
    const int w = cplx ? 2 : 1;
    cuuint64_t dims[2] = {static_cast<cuuint64_t>(m.rows) * w, static_cast<cuuint64_t>(m.cols)};
    cuuint64_t strides[1] = {static_cast<cuuint64_t>(m.ld) * 8 * w};
    cuuint32_t box[2] = {static_cast<cuuint32_t>(BK), static_cast<cuuint32_t>(box_cols)};
    cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(m.ptr), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// Launch with the programmatic-stream-serialization attribute (ptx.cuh: grid_dep_wait): only for
// kernels that call grid_dep_wait() before their first global-memory access.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

inline int num_tiles(const EngineParams& p)
{
    int per = p.tiles_m * p.tiles_n;
    if (p.order == ORDER_TRI_ROW_DESC || p.order == ORDER_TRI_DIAG_DESC) {
        const int G = p.super > 1 ? p.super : 1;
        const int ns = (p.tiles_n + G - 1) / G;
        per = ns * (ns + 1) / 2 * G * G;     // padded: CTAs outside the triangle exit at once
    }
    else if (p.order == ORDER_TRAPEZOID) per = p.tiles_m * p.tiles_n - p.tiles_m * (p.tiles_m - 1) / 2;
    return per * p.batch;
}

inline cudaError_t engine_configure_device()
{
    cudaError_t e = cudaFuncSetAttribute(tile_engine_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tile_engine_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tile_engine_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tile_engine_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tile64_engine_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, k64SmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(tile64_engine_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, k64SmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ctile_half_engine_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kHSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ctile_half_engine_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kHSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ctile_engine_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(ctile_engine_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCSmemBytes);
    return e;
}

inline cudaError_t engine_configure()
{
    static PerDeviceOnce once;
    return once.run(engine_configure_device);
}

// a_nn: A operand is m-contiguous (A stored M x K).  Returns cudaSuccess or the launch error.
// use_tma: every operand satisfies tma_compatible() and the tensor maps in p are valid; otherwise
// the plain-load producer reads through p.raw*.
inline cudaError_t engine_launch(const EngineParams& p, bool a_nn, bool use_tma, cudaStream_t stream)
{
    const int grid = num_tiles(p);
    if (grid <= 0) return cudaSuccess;
    cudaError_t e = engine_configure();
    if (e != cudaSuccess) return e;
    if (use_tma) {
        if (a_nn) return launch_pdl(tile_engine_kernel<true, true>, grid, kThreads, kSmemBytes, stream, p);
        return launch_pdl(tile_engine_kernel<false, true>, grid, kThreads, kSmemBytes, stream, p);
    }
    if (a_nn) return launch_pdl(tile_engine_kernel<true, false>, grid, kThreads, kSmemBytes, stream, p);
    return launch_pdl(tile_engine_kernel<false, false>, grid, kThreads, kSmemBytes, stream, p);
}

// real engine with 64 x 64 CTA tiles (tile64_engine.cuh): four CTAs per logical 128-tile; TMA only
inline cudaError_t engine64_launch(const EngineParams& p, bool a_nn, cudaStream_t stream)
{
    const int grid = 4 * num_tiles(p);
    if (grid <= 0) return cudaSuccess;
    cudaError_t e = engine_configure();
    if (e != cudaSuccess) return e;
    if (a_nn) return launch_pdl(tile64_engine_kernel<true>, grid, k64Threads, k64SmemBytes, stream, p);
    return launch_pdl(tile64_engine_kernel<false>, grid, k64Threads, k64SmemBytes, stream, p);
}

// complex128 engine: operands always go through TMA (a complex row pitch is a multiple of 16 bytes)
inline cudaError_t cengine_launch(const EngineParams& p, bool a_nn, bool half, cudaStream_t stream)
{
    if (half) {   // two 64 x 32 CTAs per logical tile (ctile_half_engine.cuh)
        const int g2 = 2 * num_tiles(p);
        if (g2 <= 0) return cudaSuccess;
        const cudaError_t e2 = engine_configure();
        if (e2 != cudaSuccess) return e2;
        if (a_nn) return launch_pdl(ctile_half_engine_kernel<true>, g2, kCThreads, kHSmemBytes, stream, p);
        return launch_pdl(ctile_half_engine_kernel<false>, g2, kCThreads, kHSmemBytes, stream, p);
    }
    const int grid = num_tiles(p);
    if (grid <= 0) return cudaSuccess;
    cudaError_t e = engine_configure();
    if (e != cudaSuccess) return e;
    if (a_nn) return launch_pdl(ctile_engine_kernel<true>, grid, kCThreads, kCSmemBytes, stream, p);
    return launch_pdl(ctile_engine_kernel<false>, grid, kCThreads, kCSmemBytes, stream, p);
}

}  // namespace gs
