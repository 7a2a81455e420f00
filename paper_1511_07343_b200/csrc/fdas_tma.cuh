// fdas_tma.cuh -- the asynchronous-copy machinery of sm_90+/sm_100 as small device functions: mbarrier
// objects, bulk copies (cp.async.bulk, SASS UBLKCP) and tensor-map box copies (cp.async.bulk.tensor, the TMA,
// SASS UTMALDG / UTMASTG), plus the host side that encodes tensor maps through the driver entry point.
//
// Rules the callers keep (PTX ISA "Asynchronous copy" / "mbarrier"):
//   * an mbarrier lives in shared memory, 8-byte aligned; one thread initialises it, then mbar_fence_init()
//     and a CTA barrier before anybody waits on it or a copy names it;
//   * a load is announced to its mbarrier with mbar_expect_tx(bytes) by the thread that issues it; the phase
//     completes when the announced arrivals AND bytes have come in; every consumer waits on the PARITY of the
//     phase (mbar_wait) before reading the destination;
//   * bulk copies move multiples of 16 bytes between 16-byte aligned addresses; a box destination/source in
//     shared memory is 128-byte aligned; the tensor map fixes the box shape, coordinates are in elements,
//     innermost first, and may lie outside the tensor (loads read zeros there, stores skip it);
//   * a store reads shared memory that ordinary stores wrote: the writers call fence_proxy_async(), then a CTA
//     barrier, then ONE thread issues the store, commits it (tma_store_commit) and, before the buffer is reused
//     or the CTA exits, waits for it (tma_store_wait_read / tma_store_wait_all).
// Waits are BOUNDED: if a phase does not complete within FDAS_MBAR_TIMEOUT_NS the waiter records the fact in the
// status word the kernel was given and returns false, so that a mistake in a byte count shows up as a reported
// error (FDAS_E_CUDA from fdas_plan_status) and not as a hung GPU.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

constexpr unsigned long long FDAS_MBAR_TIMEOUT_NS = 2000000000ull;     // 2 s: five orders of magnitude above any real wait
constexpr uint32_t FDAS_STATUS_MBAR_TIMEOUT = 1u;                      // bit set in the plan's device status word

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t arrivals)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(arrivals) : "memory");
}
// make the initialisation visible to the asynchronous proxy (the copy engines) before the first copy names it
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of asynchronous traffic for the current phase
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t done;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done)
                 : "r"(smem_u32(bar)), "r"(parity)
                 : "memory");
    return done != 0;
}
__device__ __forceinline__ unsigned long long global_timer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Wait for the phase of parity `parity` (0 for the first use of a barrier, then alternating).  false = timed out.
__device__ __forceinline__ bool mbar_wait(uint64_t* bar, uint32_t parity, uint32_t* status)
{
    if (mbar_try_wait(bar, parity)) return true;
    const unsigned long long t0 = global_timer_ns();
    while (!mbar_try_wait(bar, parity)) {
        if (global_timer_ns() - t0 > FDAS_MBAR_TIMEOUT_NS) {
            if (status) atomicOr(status, FDAS_STATUS_MBAR_TIMEOUT);
            return false;
        }
    }
    return true;
}

// global -> shared, `bytes` contiguous bytes, completion counted on `bar`
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// global -> shared, one box of the tensor map at element coordinates (c0 innermost, ...)
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
                 : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
// shared -> global, one box (bulk-group completion)
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, const void* smem_src, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];" ::"l"(map), "r"(smem_u32(smem_src)),
                 "r"(c0), "r"(c1), "r"(c2)
                 : "memory");
}
__device__ __forceinline__ void tma_store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
// the committed stores have finished READING shared memory (the buffer may be overwritten)
__device__ __forceinline__ void tma_store_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// the committed stores are complete (required before the CTA exits)
__device__ __forceinline__ void tma_store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
// order this thread's ordinary shared-memory writes before later asynchronous-proxy reads of them
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tma_prefetch_map(const CUtensorMap* map)
{
    asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// barrier `id` (1..15; 0 is __syncthreads) among `n_threads` threads of the CTA (a multiple of 32: whole warps)
__device__ __forceinline__ void named_bar_sync(int id, int n_threads)
{
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n_threads) : "memory");
}

// ------------------------------------------------------------------ host: tensor-map encoding
// Tensor of 8-byte elements (a float2 / complex value is one element), rank 2 or 3, dims[0] innermost and
// contiguous, strides_bytes[i] = byte stride of dims[i+1] (multiples of 16), box[i] <= 256 elements.
// Returns false if the driver entry point is missing or refuses the description.
bool fdas_encode_tensor_map(CUtensorMap* out, const void* base, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                            const uint32_t* box);
