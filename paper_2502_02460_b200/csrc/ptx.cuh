// ptx.cuh -- thin inline-PTX wrappers used by the sm_100a kernels of libgs:
// mbarrier (producer/consumer pipeline), TMA tile loads (cp.async.bulk.tensor), FP64 tensor-core
// MMA (mma.sync m8n8k4 f64 -> SASS DMMA.8x8x4, the only FP64 MMA shape sm_100a implements natively).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gs {

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}

__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!mbar_try_wait(bar, parity)) {}
}

// TMA: 2-D tiled load global -> shared, completion signalled on an mbarrier (complete_tx::bytes).
// c0 = coordinate along the contiguous dimension (row index of a column-major matrix),
// c1 = coordinate along the strided dimension (column index).
__device__ __forceinline__ void tma_load_2d(uint32_t dst_smem, const CUtensorMap* map, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst_smem), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}

// The same with an L2 eviction policy for the lines the load brings in (createpolicy): a stream that is read once
// (the triangle of the tridiagonalisation's matrix-vector product) should not push the small, hot vectors out of L2.
__device__ __forceinline__ uint64_t l2_policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst_smem, const CUtensorMap* map, int c0, int c1, uint32_t bar, uint64_t policy)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;"
        ::"r"(dst_smem), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar), "l"(policy)
        : "memory");
}

__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(map)) : "memory");
}

// D(8x8) += A(8x4, row) * B(4x8, col), FP64.  Lane t holds A[t/4][t%4], B[t%4][t/4],
// D[t/4][2*(t%4) + {0,1}].
__device__ __forceinline__ void dmma_8x8x4(double& d0, double& d1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(d0), "+d"(d1)
        : "d"(a), "d"(b));
}

// Consumer release of pipeline stage s-1, performed at the top of iteration s (after the wait on
// stage s).  It must NOT sit right behind the last fragment loads of the stage it releases: an
// mbarrier arrive is not held back by LDS instructions that are still in flight (SASS: the last
// LDS.128 was issued three instructions before SYNCS.ARRIVE, its DMMAs after it), so the producer's
// next TMA fill could overwrite the stage under a pending load -- seen as sporadic wrong tiles with
// two CTAs per SM.  One iteration later every DMMA that consumed those loads has been issued
// (they precede the spin-wait in program order), i.e. the loads have returned.
__device__ __forceinline__ void release_previous_stage(int s, int nstages, uint32_t empty0, int lane)
{
    if (s > 0) {
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * ((s - 1) % nstages));
    }
}

// Programmatic dependent launch: a kernel launched with the programmatic-stream-serialization
// attribute may start while its predecessor in the stream is still running; it must not touch
// global memory before grid_dep_wait() (which returns once the predecessor has completed and its
// writes are visible).  grid_dep_launch() lets the successor's CTAs be scheduled early, so launch
// latency and the prologue (barrier init, descriptor prefetch) hide behind this kernel's tail.
__device__ __forceinline__ void grid_dep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_dep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t nthreads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

}  // namespace gs
