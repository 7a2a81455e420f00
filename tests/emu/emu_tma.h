// Emulator model of paper_1511_07343_b200/csrc/fdas_tma.cuh (prep.py swaps the include): the same function
// names, implemented on the host in emu_rt.cpp with the hardware's rules ENFORCED rather than assumed --
//   * mbarrier phases: arrival counts, announced bytes, parity waits; a wait that can never be satisfied is
//     reported as a deadlock with the kernel and block named;
//   * copies are DEFERRED: a load moves its bytes only after every runnable thread of the CTA has had its turn (so
//     a read of the destination that is not ordered after the mbarrier wait sees NaN poison), a store reads shared memory only when its group is waited
//     for (so reusing the buffer too early corrupts the output), and a CTA that exits with stores not waited
//     for aborts;
//   * sizes and alignments (16-byte multiples, 128-byte box buffers, box <= 256 elements, 16-byte strides) abort
//     on violation; coordinates outside the tensor read zeros / are not written.
// TEST INFRASTRUCTURE ONLY (tests/emu/README.md).
#pragma once
#include "cuda_runtime.h"

typedef int CUresult;
enum { CUDA_SUCCESS = 0, CUDA_ERROR_INVALID_VALUE = 1 };
typedef unsigned long long cuuint64_t;
typedef unsigned cuuint32_t;
struct alignas(64) CUtensorMap { unsigned long long opaque[16]; };
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_UINT64 = 8, CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 4 };   // value = element bytes here
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0, CU_TENSOR_MAP_L2_PROMOTION_L2_128B = 2 };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };
enum { cudaEnableDefault = 0 };
cudaError_t cudaGetDriverEntryPoint(const char* symbol, void** fn, unsigned long long flags, cudaDriverEntryPointQueryResult* q);
#define __grid_constant__

constexpr unsigned long long FDAS_MBAR_TIMEOUT_NS = 2000000000ull;
constexpr uint32_t FDAS_STATUS_MBAR_TIMEOUT = 1u;

void mbar_init(uint64_t* bar, uint32_t arrivals);
static inline void mbar_fence_init() {}
void mbar_expect_tx(uint64_t* bar, uint32_t bytes);
void mbar_arrive(uint64_t* bar);
bool mbar_try_wait(uint64_t* bar, uint32_t parity);
bool mbar_wait(uint64_t* bar, uint32_t parity, uint32_t* status);
void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar);
void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar);
void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar);
void tma_store_3d(const CUtensorMap* map, const void* smem_src, int c0, int c1, int c2);
void tma_store_commit();
void tma_store_wait_read();
void tma_store_wait_all();
static inline void fence_proxy_async() {}
void named_bar_sync(int id, int n_threads);
static inline void tma_prefetch_map(const CUtensorMap*) {}

bool fdas_encode_tensor_map(CUtensorMap* out, const void* base, int rank, const uint64_t* dims, const uint64_t* strides_bytes,
                            const uint32_t* box);
