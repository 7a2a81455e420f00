// fdas_resample.cu -- time-domain acceleration trial ("resampling
// the time series according to a time offset caused by the constant acceleration, followed by a standard
// periodicity search for each acceleration value").  The periodicity search of a resampled series is the
// existing path: fdas_spectrum, then a plan with z_max = 0 (one delta template) gives |S|^2 and candidates.
#include "fdas_common.cuh"

// y[m] = x[nearest sample to u N],  u = 2u' / [(1-beta) + sqrt((1-beta)^2 + 4 beta u')],  u' = m/N:
// the root of u + beta (u^2 - u) = u' (include/fdas.h).  The index is decided in fp64 with separately
// rounded operations (__d*_rn are never contracted into FMAs), the same sequence as the reference.
// One thread per 4 consecutive outputs (a 16-byte store); the gathers of a warp fall in <= 2 lines.
__global__ void __launch_bounds__(256)
k_resample(const float* __restrict__ x, float* __restrict__ y, long long N, double beta)
{
    const long long m0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (m0 >= N) return;
    const double omb = __dsub_rn(1.0, beta), omb2 = __dmul_rn(omb, omb), fb = __dmul_rn(4.0, beta), dN = (double)N;
    float out[4];
#pragma unroll
    for (int i = 0; i < 4; i++) {
        const double up = __ddiv_rn((double)(m0 + i), dN);
        const double disc = __dadd_rn(omb2, __dmul_rn(fb, up));
        const double u = __ddiv_rn(__dmul_rn(2.0, up), __dadd_rn(omb, __dsqrt_rn(disc)));
        long long n = (long long)floor(__dadd_rn(__dmul_rn(u, dN), 0.5));
        n = n > N - 1 ? N - 1 : (n < 0 ? 0 : n);
        out[i] = m0 + i < N ? __ldg(x + n) : 0.0f;
    }
    if (m0 + 3 < N) *reinterpret_cast<float4*>(y + m0) = make_float4(out[0], out[1], out[2], out[3]);
    else
        for (int i = 0; i < 4 && m0 + i < N; i++) y[m0 + i] = out[i];
}

int fdas_launch_resample(fdas_plan* p, const float* d_series, double beta, float* d_out, cudaStream_t st)
{
    const long long N = p->n_samples;
    const unsigned grid = (unsigned)((N / 4 + 255) / 256);
    k_resample<<<grid, 256, 0, st>>>(d_series, d_out, N, beta);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}
