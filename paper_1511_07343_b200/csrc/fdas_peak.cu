// fdas_peak.cu -- FP32 FMA-rate microbenchmark ("the builder must add an
// FFMA-chain microbenchmark, record the measured FP32 peak").  It gives bench.py a MEASURED
// denominator for the ALU-bound fused correlate kernel beside the nominal 148 x 128 x 2 x clock.
// Measurement aid only: nothing on the search path calls it.
#include "fdas_common.cuh"

constexpr int PEAK_ACC = 16;           // independent accumulators per thread (FMA latency 4 x 4 warps per scheduler)

// Every thread runs `iters` rounds of PEAK_ACC fused multiply-adds a <- a*x + y with loop-invariant x, y
// (the operand pattern of the FFT butterflies: two invariant twiddle registers, one running value).
__global__ void __launch_bounds__(256)
k_ffma_peak(float* __restrict__ sink, float x, float y, int iters)
{
    float a[PEAK_ACC];
#pragma unroll
    for (int i = 0; i < PEAK_ACC; i++) a[i] = (float)(threadIdx.x + i) * 1.0e-3f;
#pragma unroll 1
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++) {
#pragma unroll
            for (int i = 0; i < PEAK_ACC; i++) a[i] = fmaf(a[i], x, y);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < PEAK_ACC; i++) s += a[i];
    if (s == 123.456f) sink[0] = s;    // never true for the x, y used; keeps the chain alive
}

// The same chains with the packed f32x2 instruction of sm_100 (FFMA2: two FMAs per lane and issue slot).
__global__ void __launch_bounds__(256)
k_ffma2_peak(float* __restrict__ sink, float x, float y, int iters)
{
    float2 a[PEAK_ACC / 2];
    const float2 x2 = make_float2(x, x), y2 = make_float2(y, y);
#pragma unroll
    for (int i = 0; i < PEAK_ACC / 2; i++) a[i] = make_float2((float)(threadIdx.x + i) * 1.0e-3f, (float)(threadIdx.x + i) * 2.0e-3f);
#pragma unroll 1
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < 4; r++) {
#pragma unroll
            for (int i = 0; i < PEAK_ACC / 2; i++) a[i] = __ffma2_rn(a[i], x2, y2);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < PEAK_ACC / 2; i++) s += a[i].x + a[i].y;
    if (s == 123.456f) sink[0] = s;
}

extern "C" int fdas_measure_fp32_tflops(double* out_tflops, double* out_ms, int32_t packed, void* stream)
{
    if (!out_tflops) return FDAS_E_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    FDAS_CUDA(cudaGetDevice(&dev));
    FDAS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    const int iters = 4096, grid = sms * 8, block = 256;
    double best_ms = 1.0e30;
    cudaError_t err = cudaMalloc(&sink, sizeof(float));
    if (err == cudaSuccess) err = cudaEventCreate(&e0);
    if (err == cudaSuccess) err = cudaEventCreate(&e1);
    for (int rep = 0; rep < 5 && err == cudaSuccess; rep++) {   // rep 0 warms up; best of the rest (burst figure)
        err = cudaEventRecord(e0, st);
        if (err != cudaSuccess) break;
        if (packed) k_ffma2_peak<<<grid, block, 0, st>>>(sink, 0.999f, 1.0e-3f, iters);
        else k_ffma_peak<<<grid, block, 0, st>>>(sink, 0.999f, 1.0e-3f, iters);
        err = cudaGetLastError();
        if (err == cudaSuccess) err = cudaEventRecord(e1, st);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
        if (err == cudaSuccess && rep > 0 && ms < best_ms) best_ms = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (sink) cudaFree(sink);
    if (err != cudaSuccess) { fdas_set_cuda_error(err, "fdas_measure_fp32_tflops"); return FDAS_E_CUDA; }
    const double flops = 2.0 * 4.0 * PEAK_ACC * (double)iters * (double)grid * (double)block;
    *out_tflops = flops / (best_ms * 1.0e-3) / 1.0e12;
    if (out_ms) *out_ms = best_ms;
    return FDAS_OK;
}

// L2 -> SM read bandwidth (measurement aid for the harmonic sum, whose inherent cost is an L2 -> SM stream of 5.84
// planes): EVERY CTA streams the whole buffer -- small enough to stay in the 126 MB L2, far too
// large for L1 -- once, with coalesced 16-byte loads, each CTA starting at a different place.  Bytes moved from L2
// = grid x buffer; DRAM is touched on the first pass of the first launch only.
__global__ void __launch_bounds__(256)
k_l2_read(const float4* __restrict__ buf, size_t n4, float* __restrict__ sink)
{
    float acc = 0.0f;
    const size_t start = ((size_t)blockIdx.x * 9973u * 256u) % n4;
    for (size_t i = threadIdx.x; i < n4; i += 256) {
        size_t j = start + i;
        if (j >= n4) j -= n4;
        const float4 v = __ldg(buf + j);
        acc += v.x + v.y + v.z + v.w;
    }
    if (acc == 123.456f) sink[0] = acc;       // never true for a zeroed buffer; keeps the loads alive
}

extern "C" int fdas_measure_l2_gbs(double* out_gbs, size_t bytes, void* stream)
{
    if (!out_gbs || bytes < ((size_t)1 << 20) || bytes > ((size_t)96 << 20)) return FDAS_E_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    FDAS_CUDA(cudaGetDevice(&dev));
    FDAS_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t n4 = bytes / 16;
    const int grid = sms * 4;
    float4* buf = nullptr;
    float* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t err = cudaMalloc(&buf, n4 * 16);
    if (err == cudaSuccess) err = cudaMalloc(&sink, sizeof(float));
    if (err == cudaSuccess) err = cudaMemsetAsync(buf, 0, n4 * 16, st);
    if (err == cudaSuccess) err = cudaEventCreate(&e0);
    if (err == cudaSuccess) err = cudaEventCreate(&e1);
    double best_ms = 1.0e30;
    for (int rep = 0; rep < 4 && err == cudaSuccess; rep++) {                 // rep 0 warms up
        err = cudaEventRecord(e0, st);
        if (err != cudaSuccess) break;
        k_l2_read<<<grid, 256, 0, st>>>(buf, n4, sink);
        err = cudaGetLastError();
        if (err == cudaSuccess) err = cudaEventRecord(e1, st);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float ms = 0.0f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
        if (err == cudaSuccess && rep > 0 && ms < best_ms) best_ms = ms;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (buf) cudaFree(buf);
    if (sink) cudaFree(sink);
    if (err != cudaSuccess) { fdas_set_cuda_error(err, "fdas_measure_l2_gbs"); return FDAS_E_CUDA; }
    *out_gbs = (double)grid * (double)n4 * 16.0 / (best_ms * 1.0e-3) / 1.0e9;
    return FDAS_OK;
}
