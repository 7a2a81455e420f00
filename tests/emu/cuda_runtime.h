// Host emulation shim for CUDA device code: committed TEST INFRASTRUCTURE (tests/emu/README.md), never on the product path.
#pragma once
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>
#include <functional>

#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __noinline__ __attribute__((noinline))
#define __restrict__ __restrict
#define __launch_bounds__(...)
#define __shared__ thread_local
#define __align__(n) __attribute__((aligned(n)))

struct alignas(8) float2 { float x, y; };          // CUDA's alignments: the emu build runs with -fsanitize=alignment
struct alignas(16) float4 { float x, y, z, w; };
struct alignas(16) double2 { double x, y; };
struct uint3 { unsigned x, y, z; };
struct dim3 {
    unsigned x, y, z;
    dim3(unsigned a = 1, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {}
};
static inline float2 make_float2(float x, float y) { return float2{x, y}; }
static inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }

extern thread_local uint3 threadIdx, blockIdx;
extern thread_local dim3 blockDim, gridDim;

typedef int cudaError_t;
typedef void* cudaStream_t;
enum { cudaSuccess = 0, cudaErrorMemoryAllocation = 2 };
enum cudaMemcpyKind { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributePreferredSharedMemoryCarveout = 9 };

cudaError_t cudaMalloc(void** p, size_t n);
template <class T> static inline cudaError_t cudaMalloc(T** p, size_t n) { return cudaMalloc((void**)p, n); }
cudaError_t cudaFree(void* p);
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind k);
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind k, cudaStream_t st);
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t st);
// every stream / event operation is logged (EMU_STREAM_TRACE=<file>) so that a test can rebuild the happens-before graph
void emu_trace(const char* op, const void* a, const void* b, const void* c, size_t n);
static inline cudaError_t cudaStreamSynchronize(cudaStream_t s) { emu_trace("streamsync", s, 0, 0, 0); return cudaSuccess; }
// streams and events: every enqueue runs to completion before it returns, so ordering is trivially kept
typedef void* cudaEvent_t;
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };
uintptr_t emu_new_id();
static inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = (cudaStream_t)(0x5000 + emu_new_id()); return cudaSuccess; }
static inline cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned) { *e = (cudaEvent_t)(0xE000 + emu_new_id()); return cudaSuccess; }
static inline cudaError_t cudaEventDestroy(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = (cudaEvent_t)(0xE000 + emu_new_id()); return cudaSuccess; }
static inline cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t, cudaEvent_t) { *ms = 1.0f; return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s) { emu_trace("record", s, e, 0, 0); return cudaSuccess; }
static inline cudaError_t cudaEventSynchronize(cudaEvent_t e) { emu_trace("eventsync", 0, e, 0, 0); return cudaSuccess; }
static inline cudaError_t cudaStreamWaitEvent(cudaStream_t s, cudaEvent_t e, unsigned) { emu_trace("wait", s, e, 0, 0); return cudaSuccess; }
template <class T> static inline cudaError_t cudaMallocHost(T** p, size_t n) { *p = (T*)malloc(n); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
static inline cudaError_t cudaFreeHost(void* p) { free(p); return cudaSuccess; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaSetDevice(int) { return cudaSuccess; }
// the pretend device: EMU_SMS SMs (default 3) with EMU_CTAS_PER_SM resident CTAs each (default 2), so that persistent
// kernels loop over several items per CTA; EMU_SMS=148 with the real occupancy exercises the B200 geometry
enum cudaDeviceAttr { cudaDevAttrMultiProcessorCount = 16 };
int emu_env_int(const char* name, int dflt);
static inline cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaDeviceGetAttribute(int* v, cudaDeviceAttr, int) { *v = emu_env_int("EMU_SMS", 3); return cudaSuccess; }
template <class F> static inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int* n, F, int, size_t) { *n = emu_env_int("EMU_CTAS_PER_SM", 2); return cudaSuccess; }
struct cudaFuncAttributes { int numRegs; size_t sharedSizeBytes; };
template <class F> static inline cudaError_t cudaFuncGetAttributes(cudaFuncAttributes* a, F) { a->numRegs = 0; a->sharedSizeBytes = 0; return cudaSuccess; }
static inline const char* cudaGetErrorString(cudaError_t) { return "emu"; }
template <class F> static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int) { return cudaSuccess; }

// ---- device runtime
void emu_syncthreads();
void emu_syncwarp();
void* emu_dyn_smem();
void emu_check_ptr(const void* p, size_t n, const char* what);
void emu_launch(dim3 grid, dim3 block, size_t smem, const char* name, const std::function<void()>& body, cudaStream_t st = 0);
unsigned emu_ballot(int pred);
static inline unsigned __ballot_sync(unsigned mask, int pred)
{
    if (mask != 0xffffffffu) { fprintf(stderr, "EMU: __ballot_sync with a partial mask is not modelled\n"); abort(); }
    return emu_ballot(pred);
}
unsigned emu_shfl(unsigned v, int src_lane);
static inline unsigned __shfl_sync(unsigned mask, unsigned v, int src_lane)
{
    if (mask != 0xffffffffu) { fprintf(stderr, "EMU: __shfl_sync with a partial mask is not modelled\n"); abort(); }
    return emu_shfl(v, src_lane);
}
static inline int __any_sync(unsigned mask, int pred) { return __ballot_sync(mask, pred) != 0; }
static inline int __ffs(int x) { return __builtin_ffs(x); }
static inline int __popc(unsigned x) { return __builtin_popcount(x); }
static inline int __clz(int x) { return x ? __builtin_clz((unsigned)x) : 32; }
#define __syncthreads() emu_syncthreads()
#define __syncwarp() emu_syncwarp()

template <class T> static inline T __ldg(const T* p)
{
    emu_check_ptr(p, sizeof(T), "__ldg");
    return *p;
}
template <class T> static inline T __ldcs(const T* p)
{
    emu_check_ptr(p, sizeof(T), "__ldcs");
    return *p;
}
static inline unsigned atomicAdd(unsigned* p, unsigned v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned atomicMax(unsigned* p, unsigned v) { unsigned o = __atomic_load_n(p, __ATOMIC_RELAXED); while (o < v && !__atomic_compare_exchange_n(p, &o, v, false, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {} return o; }
static inline unsigned __float_as_uint(float x) { unsigned i; memcpy(&i, &x, 4); return i; }
static inline unsigned atomicOr(unsigned* p, unsigned v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }

static inline void sincospif(float x, float* s, float* c)
{
    double r = (double)x - 2.0 * floor((double)x * 0.5);
    *s = (float)sin(M_PI * r);
    *c = (float)cos(M_PI * r);
}
static inline void sincospi(double x, double* s, double* c)
{
    double r = x - 2.0 * floor(x * 0.5);
    *s = sin(M_PI * r);
    *c = cos(M_PI * r);
}
// separately rounded fp64 operations (the emu build has no FMA contraction: plain x86-64, -ffp-contract=off)
static inline double __dadd_rn(double a, double b) { volatile double r = a + b; return r; }
static inline double __dsub_rn(double a, double b) { volatile double r = a - b; return r; }
static inline double __dmul_rn(double a, double b) { volatile double r = a * b; return r; }
static inline double __ddiv_rn(double a, double b) { volatile double r = a / b; return r; }
static inline double __dsqrt_rn(double a) { volatile double r = sqrt(a); return r; }
static inline float2 __ffma2_rn(float2 a, float2 b, float2 c) { return float2{fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)}; }
static inline int __float_as_int(float x) { int i; memcpy(&i, &x, 4); return i; }
static inline float __int_as_float(int i) { float x; memcpy(&x, &i, 4); return x; }
static inline float2 __fmul2_rn(float2 a, float2 b) { return float2{a.x * b.x, a.y * b.y}; }
static inline float2 __fadd2_rn(float2 a, float2 b) { return float2{a.x + b.x, a.y + b.y}; }
static inline int min(int a, int b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }
static inline long long min(long long a, long long b) { return a < b ? a : b; }
static inline long long max(long long a, long long b) { return a > b ? a : b; }
static inline unsigned min(unsigned a, unsigned b) { return a < b ? a : b; }
static inline float min(float a, float b) { return fminf(a, b); }
static inline float max(float a, float b) { return fmaxf(a, b); }
