// fdas_spectrum.cu -- PAPER.md:49 step 2, "Real to complex DFT of the time series", plus the
// mean-power normalisation of BASELINE.json configs[0].
//
// The N real samples are packed as M = N/2 complex numbers z[n] = x[2n] + i x[2n+1] and
// transformed by a four-step FFT with M = R1*R2 (n = n1*R2 + n2, k = k1 + R1*k2):
//   pass 1  column FFTs over n1 (length R1) for every n2, times W_M^{n2 k1}   -> workspace
//   pass 2  row FFTs over n2 (length R2) for rows k1 and R1-k1 together, then the real-input
//           untangle F_k = E_k + e^{-2 pi i k/N} O_k, scaling by 1/sqrt(mu), write S.
// mu = mean_{k=1..N/2}|F_k|^2 is obtained in pass 1 from the time domain by Parseval:
//   sum_{k=1}^{N/2}|F_k|^2 = (N sum x^2 - F_0^2 + F_{N/2}^2)/2, F_0 = sum x, F_{N/2} = sum (-1)^n x_n,
// accumulated in fp64 per CTA and reduced in a fixed order (deterministic, no atomics).
#include "fdas_common.cuh"
#include "fdas_smemfft.cuh"

// threads per CTA of both passes: the 131 KB tiles allow one CTA per SM, so the CTA itself must carry
// enough warps (16) to keep loads in flight while others compute
constexpr int SPEC_THREADS = 512;

// pass 1: grid = (R2/C, n_batch), block SPEC_THREADS, smem 2*C*(R1+1) float2.
__global__ void __launch_bounds__(SPEC_THREADS)
k_spec_pass1(const float* __restrict__ series, float2* __restrict__ inter, double* __restrict__ part,
             int M, int R1, int R2, int C)
{
    extern __shared__ float2 sm[];
    const int pitch = R1 + 1;
    float2* a = sm;
    float2* b = sm + C * pitch;
    const int n2_0 = blockIdx.x * C, bt = blockIdx.y;
    const float2* z = reinterpret_cast<const float2*>(series) + (size_t)bt * M;
    double s1 = 0.0, s2 = 0.0, sa = 0.0;
    for (int idx = threadIdx.x; idx < C * R1; idx += blockDim.x) {
        int n1 = idx / C, cc = idx - n1 * C;
        float2 v = z[(size_t)n1 * R2 + n2_0 + cc];
        a[cc * pitch + n1] = v;
        double x = v.x, y = v.y;
        s1 += x + y;
        sa += x - y;
        s2 = fma(x, x, fma(y, y, s2));
    }
    float2* r = smem_fft(a, b, R1, C, pitch, -1.0f);
    for (int idx = threadIdx.x; idx < C * R1; idx += blockDim.x) {
        int k1 = idx / C, cc = idx - k1 * C;
        int n2 = n2_0 + cc;
        int ph = (int)(((long long)n2 * k1) & (M - 1));
        float2 v = cmul_pk(r[cc * pitch + k1], twiddle(ph, M, -1.0f));
        inter[(size_t)bt * M + (size_t)k1 * R2 + n2] = v;
    }
    // block reduction of the three sums (fixed tree)
    __shared__ double red[3][SPEC_THREADS];
    red[0][threadIdx.x] = s1; red[1][threadIdx.x] = s2; red[2][threadIdx.x] = sa;
    __syncthreads();
    for (int o = SPEC_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int q = 0; q < 3; q++) red[q][threadIdx.x] += red[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x < 3) part[((size_t)bt * gridDim.x + blockIdx.x) * 3 + threadIdx.x] = red[threadIdx.x][0];
}

// pass 2: grid = (ceil((R1/2+1)/C), n_batch), block SPEC_THREADS, smem 2*(2C)*(R2+1) float2.
// Rows [0,C): k1 = g*C + i ("low"), rows [C,2C): the mirrors (R1 - k1) mod R1.
__global__ void __launch_bounds__(SPEC_THREADS)
k_spec_pass2(const float2* __restrict__ inter, const double* __restrict__ part, int n_part,
             float2* __restrict__ spec, float* __restrict__ meanpow, int M, int R1, int R2, int C)
{
    extern __shared__ float2 sm[];
    __shared__ double red[3][SPEC_THREADS];
    __shared__ float s_scale;
    const int pitch = R2 + 1;
    float2* a = sm;
    float2* b = sm + 2 * C * pitch;
    const int bt = blockIdx.y, k1_0 = blockIdx.x * C;
    // mu from the pass-1 partial sums, same order in every CTA
    double acc[3] = {0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < n_part; i += blockDim.x)
        for (int q = 0; q < 3; q++) acc[q] += part[((size_t)bt * n_part + i) * 3 + q];
    for (int q = 0; q < 3; q++) red[q][threadIdx.x] = acc[q];
    __syncthreads();
    for (int o = SPEC_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int q = 0; q < 3; q++) red[q][threadIdx.x] += red[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double N = 2.0 * (double)M;
        double tot = 0.5 * (N * red[1][0] - red[0][0] * red[0][0] + red[2][0] * red[2][0]);
        double mu = tot / (double)M;
        s_scale = mu > 0.0 ? (float)(1.0 / sqrt(mu)) : 0.0f;      // all-zero series: S := 0 (G22)
        if (meanpow && blockIdx.x == 0) meanpow[bt] = (float)mu;
    }
    // load rows
    for (int idx = threadIdx.x; idx < 2 * C * R2; idx += blockDim.x) {
        int row = idx / R2, n2 = idx - row * R2;
        int k1 = k1_0 + (row < C ? row : row - C);
        if (k1 > R1 / 2) k1 = R1 / 2;                        // padding rows of the last CTA (never stored)
        if (row >= C) k1 = (R1 - k1) & (R1 - 1);
        a[row * pitch + n2] = inter[(size_t)bt * M + (size_t)k1 * R2 + n2];
    }
    float2* r = smem_fft(a, b, R2, 2 * C, pitch, -1.0f);
    const float sc = s_scale;
    float2* out = spec + (size_t)bt * M;
    // untangle: for (row, k2): k = k1 + R1*k2 ; partner (M - k) mod M
    for (int idx = threadIdx.x; idx < 2 * C * R2; idx += blockDim.x) {
        int k2 = idx / (2 * C), row = idx - k2 * (2 * C);
        int i = row < C ? row : row - C;
        int k1l = k1_0 + i;
        if (k1l > R1 / 2) continue;
        int k1 = row < C ? k1l : ((R1 - k1l) & (R1 - 1));
        if (row >= C && (k1l == 0 || 2 * k1l == R1)) continue;   // self-mirrored rows: stored once
        int prow = row < C ? row + C : row - C;
        int pk2 = (k1 == 0) ? ((R2 - k2) & (R2 - 1)) : (R2 - 1 - k2);
        float2 zk = r[row * pitch + k2];
        float2 zp = r[prow * pitch + pk2];
        int k = k1 + R1 * k2;
        if (k == 0) {                                        // DC dropped; Nyquist -> last column
            out[M - 1] = make_float2((zk.x - zk.y) * sc, 0.0f);
            continue;
        }
        float2 e = make_float2(0.5f * (zk.x + zp.x), 0.5f * (zk.y - zp.y));      // (Z_k + conj Z_{M-k})/2
        float2 dd = make_float2(0.5f * (zk.x - zp.x), 0.5f * (zk.y + zp.y));     // (Z_k - conj Z_{M-k})/2
        float2 o = make_float2(dd.y, -dd.x);                                      // * (-i)
        float2 w = twiddle(k, 2 * M, -1.0f);
        float2 f = cadd(e, cmul_pk(o, w));
        out[k - 1] = make_float2(f.x * sc, f.y * sc);
    }
}

int fdas_launch_spectrum(fdas_plan* p, const float* d_series, int n_batch, float2* d_spec,
                         float* d_meanpow, void* d_ws, cudaStream_t st)
{
    float2* inter = reinterpret_cast<float2*>(d_ws);
    double* part = reinterpret_cast<double*>(reinterpret_cast<char*>(d_ws) + p->ws_inter_bytes);
    size_t sm1 = 2 * (size_t)p->C1 * (p->R1 + 1) * sizeof(float2);
    size_t sm2 = 2 * (size_t)(2 * p->C2) * (p->R2 + 1) * sizeof(float2);
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_pass1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm1));
    FDAS_CUDA(cudaFuncSetAttribute(k_spec_pass2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm2));
    k_spec_pass1<<<dim3(p->R2 / p->C1, n_batch), SPEC_THREADS, sm1, st>>>(d_series, inter, part, p->M, p->R1, p->R2, p->C1);
    FDAS_LAUNCH_CHECK();
    int g2 = (p->R1 / 2 + 1 + p->C2 - 1) / p->C2;
    k_spec_pass2<<<dim3(g2, n_batch), SPEC_THREADS, sm2, st>>>(inter, part, p->n_part, d_spec, d_meanpow,
                                                      p->M, p->R1, p->R2, p->C2);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}
