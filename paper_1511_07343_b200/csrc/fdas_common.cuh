// fdas_common.cuh -- plan object, error plumbing and small device helpers shared by the
// kernels of libfdas.so (include/fdas.h is the public boundary).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/fdas.h"

struct fdas_plan {
    int64_t n_samples, n_bins, n_cols;
    int32_t bin0, n_z, n_t, m, L, step, n_seg, interbin, nset;
    double  z_max, dz;
    int32_t max_batch, quad_points;
    int32_t built;
    int32_t n_sms;                     // SMs of the device the bank was built on (launch geometry)
    // tuning keys (FDAS_OPT_TUNE_*; 0 = default), read by the launchers
    int32_t tune_scalar, tune_t_chunks, tune_hs_sectors, tune_hs_rows, tune_hs_variant, tune_spec_generic, tune_stage_templates, tune_spec_selftest;
    // big FFT split of the packed half-length transform: M = n_samples/2 = R1*R2
    int32_t M, R1, R2, C1, C2, n_part;
    size_t  ws_inter_bytes, ws_part_bytes, workspace_bytes;
    // TMA-staged multi-pass spectrum (fdas_spectrum_tma.cu): M = 2^(la+lb+lc), 0 passes = series too short for it
    int32_t sp_npass, sp_la, sp_lb, sp_lc;
    uint32_t* d_status;                // device status word (bit 0: an mbarrier wait timed out), allocated with the bank
    // template bank (device, owned)
    float2* d_taps;   // [n_t][m]  conj R_z(d_j), fp32
    float2* d_W;      // [n_t][L]  FFT_L(index-reversed taps)/L, natural order
    float2* d_Wr;     // the same spectra in the register layout of k_correlate_2048 (L = 2048 only)
    float2* d_segtw;  // per-thread twiddle table of the L = 2048 segment kernels (46 x 128 float2, fdas_correlate.cu)
    // scratch arena of fdas_search_host (device, owned, lazily allocated)
    void*   arena;
    size_t  arena_bytes;
    uint32_t* pinned_counts;           // pinned host staging for the candidate counts
    size_t  pinned_counts_n;
    int32_t pipe_ready;                // copy streams + events of the host pipeline exist
    cudaStream_t st_h2d, st_d2h;
    cudaEvent_t ev_in[2], ev_free[2], ev_done[2];
};

void fdas_set_cuda_error(cudaError_t e, const char* where);

#define FDAS_CUDA(call)                                          \
    do {                                                         \
        cudaError_t _e = (call);                                 \
        if (_e != cudaSuccess) {                                 \
            fdas_set_cuda_error(_e, #call);                      \
            return FDAS_E_CUDA;                                  \
        }                                                        \
    } while (0)

#define FDAS_LAUNCH_CHECK() FDAS_CUDA(cudaGetLastError())

// kernel launchers (one per .cu file); all enqueue on `st` and return an FDAS code
int fdas_launch_templates(fdas_plan* p, cudaStream_t st);
int fdas_permute_templates(fdas_plan* p, cudaStream_t st);
int fdas_launch_spectrum(fdas_plan* p, const float* d_series, int n_batch, float2* d_spec,
                         float* d_meanpow, void* d_ws, cudaStream_t st);
void fdas_spectrum_tma_plan(fdas_plan* p);
int fdas_spectrum_selftest(fdas_plan* p, int mode, cudaStream_t st);
int fdas_launch_spectrum_tma(fdas_plan* p, const float* d_series, int n_batch, float2* d_spec,
                             float* d_meanpow, void* d_ws, cudaStream_t st);
// series of 2^13 samples and more take the TMA-staged multi-pass transform (tensor maps need 16-byte bases)
inline int fdas_run_spectrum(fdas_plan* p, const float* d_series, int n_batch, float2* d_spec, float* d_meanpow, void* d_ws,
                             cudaStream_t st)
{
    const bool aligned = ((reinterpret_cast<uintptr_t>(d_series) | reinterpret_cast<uintptr_t>(d_spec)) & 15) == 0;
    if (p->sp_npass && !p->tune_spec_generic && aligned)
        return fdas_launch_spectrum_tma(p, d_series, n_batch, d_spec, d_meanpow, d_ws, st);
    return fdas_launch_spectrum(p, d_series, n_batch, d_spec, d_meanpow, d_ws, st);
}
int fdas_launch_correlate(fdas_plan* p, const float2* d_spec, int n_batch, float* d_plane, float thr,
                          fdas_cand* d_cands, uint32_t* d_counts, uint32_t cap, cudaStream_t st);
int fdas_launch_harmsum(fdas_plan* p, const float* d_plane, int max_harm, const float* h_thr,
                        fdas_cand* d_cands, uint32_t* d_count, uint32_t cap, cudaStream_t st);
int fdas_launch_resample(fdas_plan* p, const float* d_series, double beta, float* d_out, cudaStream_t st);
int fdas_launch_candidates(fdas_plan* p, const float* d_plane, float thr, fdas_cand* d_cands,
                           uint32_t* d_count, uint32_t cap, cudaStream_t st);

// occupancy of the configs[2] instance of a kernel family (fdas_kernel_occupancy): resident CTAs per SM, registers
// per thread, static + dynamic shared memory per CTA
template <class K>
inline int fdas_occupancy_of(K kernel, int threads, size_t dyn_smem, int32_t* ctas, int32_t* regs, int32_t* smem)
{
    cudaFuncAttributes fa;
    int n = 0;
    if (dyn_smem > 48 * 1024) FDAS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem));
    FDAS_CUDA(cudaFuncGetAttributes(&fa, kernel));
    FDAS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kernel, threads, dyn_smem));
    *ctas = n; *regs = fa.numRegs; *smem = (int32_t)(fa.sharedSizeBytes + dyn_smem);
    return FDAS_OK;
}
int fdas_occupancy_spectrum(int which, int32_t* ctas, int32_t* regs, int32_t* smem);
int fdas_occupancy_correlate(int which, int32_t* ctas, int32_t* regs, int32_t* smem);
int fdas_occupancy_harmsum(int32_t* ctas, int32_t* regs, int32_t* smem);

// ------------------------------------------------------------------ device helpers
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// The same product with the packed f32x2 instructions of sm_100 (FMUL2 + FFMA2): per component the same two
// operations in the same order as cmul, so the result is bit-identical; half the FMA-pipe issue slots.
__device__ __forceinline__ float2 cmul_pk(float2 a, float2 b)
{
    const float2 m = __fmul2_rn(make_float2(a.y, a.y), make_float2(-b.y, b.x));      // (-a.y b.y, a.y b.x)
    return __ffma2_rn(make_float2(a.x, a.x), b, m);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

// exp(sign * 2 pi i * num / den), num/den exact in fp32 (den a power of two)
__device__ __forceinline__ float2 twiddle(int num, int den, float sign)
{
    float s, c;
    sincospif(2.0f * (float)num / (float)den, &s, &c);
    return make_float2(c, sign * s);
}

// Append one candidate; the slot counter receives the true count (include/fdas.h).
__device__ __forceinline__ void store_cand(fdas_cand* list, uint32_t slot, uint32_t cap, int col, int zi, int nharm, float power)
{
    if (slot < cap) {
        fdas_cand c;
        c.col = col; c.zi = (int16_t)zi; c.nharm = (int16_t)nharm; c.power = power;
        list[slot] = c;
    }
}

// Warp-ballot compaction: called by ALL 32 lanes of a converged warp, each with its own
// predicate.  One ballot, ONE atomicAdd per warp (by the first lane that has a hit) for the warp's whole group
// of records, the base handed round with a shuffle, lane-rank offsets inside the group.  The counter still
// receives the true number found; records beyond `cap` are dropped.
__device__ __forceinline__ void push_cand_warp(fdas_cand* list, uint32_t* count, uint32_t cap, bool hit,
                                               int col, int zi, int nharm, float power)
{
    const unsigned m = __ballot_sync(0xffffffffu, hit);
    if (m == 0) return;                                                  // warp-uniform
    const unsigned lane = (threadIdx.x + threadIdx.y * blockDim.x) & 31u;
    const int leader = __ffs((int)m) - 1;
    uint32_t base = 0;
    if ((int)lane == leader) base = atomicAdd(count, (uint32_t)__popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (hit) store_cand(list, base + (uint32_t)__popc(m & ((1u << lane) - 1u)), cap, col, zi, nharm, power);
}
