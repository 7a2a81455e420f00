// fdas_correlate.cu -- PAPER.md:49 steps 3-7 fused in one kernel (SURVEY §8 rows a2-a6, a6'):
// overlap-save window of the spectrum -> forward FFT_L -> for every template: pointwise
// multiply by its spectrum (1/L folded in), inverse FFT_L, |.|^2, keep the first `step`
// outputs -> plane row and/or thresholded candidates.  Computes Eq. (1).
#include "fdas_common.cuh"
#include "fdas_smemfft.cuh"

// v0 (generic L, natural-order smem Stockham): one CTA per (segment, batch entry).
// smem: X[L] | A[L] | B[L].
__global__ void __launch_bounds__(256)
k_correlate_smem(const float2* __restrict__ spec, const float2* __restrict__ W, float* __restrict__ plane,
                 fdas_cand* __restrict__ cands, uint32_t* __restrict__ counts, uint32_t cap, float thr,
                 int n_bins, int n_z, int nset, int m, int L, int step)
{
    extern __shared__ float2 sm[];
    float2* X = sm;
    float2* A = sm + L;
    float2* B = sm + 2 * L;
    const int seg = blockIdx.x, bt = blockIdx.y;
    const long long base = (long long)seg * step - m / 2;
    const float2* S = spec + (size_t)bt * n_bins;
    for (int i = threadIdx.x; i < L; i += blockDim.x) {
        long long c = base + i;
        A[i] = (c >= 0 && c < n_bins) ? S[c] : make_float2(0.f, 0.f);
    }
    float2* r = smem_fft(A, B, L, 1, L, -1.0f);
    for (int i = threadIdx.x; i < L; i += blockDim.x) X[i] = r[i];
    const int n_t = n_z * nset;
    const size_t n_cols = (size_t)n_bins * nset;
    const int c0 = seg * step;
    const int nvalid = min(step, n_bins - c0);
    for (int t = 0; t < n_t; t++) {
        __syncthreads();
        const float2* Wt = W + (size_t)t * L;
        for (int i = threadIdx.x; i < L; i += blockDim.x) A[i] = cmul(X[i], Wt[i]);
        float2* y = smem_fft(A, B, L, 1, L, +1.0f);
        const int zi = t / nset, s = t - zi * nset;
        for (int o = threadIdx.x; o < nvalid; o += blockDim.x) {
            float2 v = y[o];
            float pw = fmaf(v.x, v.x, v.y * v.y);
            int col = (c0 + o) * nset + s;
            if (plane) plane[((size_t)bt * n_z + zi) * n_cols + col] = pw;
            if (cands && pw > thr) push_cand(cands + (size_t)bt * cap, counts + bt, cap, col, zi, 1, pw);
        }
    }
}

int fdas_launch_correlate(fdas_plan* p, const float2* d_spec, int n_batch, float* d_plane, float thr,
                          fdas_cand* d_cands, uint32_t* d_counts, uint32_t cap, cudaStream_t st)
{
    if (d_cands) FDAS_CUDA(cudaMemsetAsync(d_counts, 0, sizeof(uint32_t) * n_batch, st));
    size_t smem = 3 * (size_t)p->L * sizeof(float2);
    FDAS_CUDA(cudaFuncSetAttribute(k_correlate_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_correlate_smem<<<dim3(p->n_seg, n_batch), 256, smem, st>>>(d_spec, p->d_W, d_plane, d_cands, d_counts, cap, thr,
                                                                  (int)p->n_bins, p->n_z, p->nset, p->m, p->L, p->step);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}
