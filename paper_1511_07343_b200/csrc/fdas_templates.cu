// fdas_templates.cu -- template bank build ("initialization
// stage that includes computation of the templates").
#include "fdas_common.cuh"
#include "fdas_smemfft.cuh"

// T_z[j] = conj R_z(d_j),  R_z(d) = int_0^1 exp(2 pi i [(-d - z/2) u + (z/2) u^2]) du
// (the constant-fdot Fourier response the paper cites from Ransom et al.).
// fp64 composite Simpson rule over `nq` (even) intervals; one CTA per tap.
// grid = (m, n_t), block = 256.
__global__ void __launch_bounds__(256)
k_gen_taps(float2* __restrict__ taps, int m, int nset, double z_max, double dz, int nq)
{
    const int j = blockIdx.x, t = blockIdx.y;
    const int zi = t / nset, s = t - zi * nset;
    const double z = -z_max + zi * dz;
    const double d = (double)(j - m / 2) + 0.5 * s;
    const double a = -d - 0.5 * z, b = 0.5 * z;
    double sr = 0.0, si = 0.0;
    for (int n = threadIdx.x; n <= nq; n += blockDim.x) {
        double u = (double)n / (double)nq;
        double cyc = fma(b * u, u, a * u);
        cyc -= floor(cyc);
        double sn, cs;
        sincospi(2.0 * cyc, &sn, &cs);
        double w = (n == 0 || n == nq) ? 1.0 : ((n & 1) ? 4.0 : 2.0);
        sr += w * cs;
        si += w * sn;
    }
    __shared__ double red[2][256];
    red[0][threadIdx.x] = sr;
    red[1][threadIdx.x] = si;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            red[0][threadIdx.x] += red[0][threadIdx.x + o];
            red[1][threadIdx.x] += red[1][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        double sc = 1.0 / (3.0 * (double)nq);
        taps[(size_t)t * m + j] = make_float2((float)(red[0][0] * sc), (float)(-red[1][0] * sc));   // conj
    }
}

// W_t = FFT_L(g_t)/L with g[(-(j+s)) mod L] = T_t[j] (index-reversed taps; the half-bin set
// s=1 sits one bin later in the window, reading G12/G13), stored in natural order [n_t][L].
// grid = n_t, block = 256, dynamic smem = 2*L*sizeof(float2).
__global__ void __launch_bounds__(256)
k_template_spectrum(const float2* __restrict__ taps, float2* __restrict__ W, int m, int L, int nset)
{
    extern __shared__ float2 sm[];
    float2* a = sm;
    float2* b = sm + L;
    const int t = blockIdx.x, s = t % nset;
    for (int i = threadIdx.x; i < L; i += blockDim.x) a[i] = make_float2(0.f, 0.f);
    __syncthreads();
    for (int j = threadIdx.x; j < m; j += blockDim.x) a[(2 * L - j - s) % L] = taps[(size_t)t * m + j];
    float2* r = smem_fft(a, b, L, 1, L, -1.0f);
    const float sc = 1.0f / (float)L;
    for (int i = threadIdx.x; i < L; i += blockDim.x)
        W[(size_t)t * L + i] = make_float2(r[i].x * sc, r[i].y * sc);
}

int fdas_launch_templates(fdas_plan* p, cudaStream_t st)
{
    int nq = p->quad_points & ~1;
    k_gen_taps<<<dim3(p->m, p->n_t), 256, 0, st>>>(p->d_taps, p->m, p->nset, p->z_max, p->dz, nq);
    FDAS_LAUNCH_CHECK();
    size_t smem = 2 * (size_t)p->L * sizeof(float2);
    FDAS_CUDA(cudaFuncSetAttribute(k_template_spectrum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_template_spectrum<<<p->n_t, 256, smem, st>>>(p->d_taps, p->d_W, p->m, p->L, p->nset);
    FDAS_LAUNCH_CHECK();
    return fdas_permute_templates(p, st);
}
