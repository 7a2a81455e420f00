// fdas_smemfft.cuh -- generic shared-memory Stockham (autosort, natural order in and out)
// FFT used by the big real-to-complex transform and by the template-spectrum kernel.
// Radix-8 passes with one radix-4 or radix-2 pass for the remainder; ping-pong buffers.
#pragma once
#include "fdas_common.cuh"

// In-place DFT of R points in registers, natural order out. sign = -1 forward, +1 inverse.
__device__ __forceinline__ void dft2(float2& a, float2& b)
{
    float2 t = a;
    a = cadd(t, b);
    b = csub(t, b);
}
// multiply by sign*i : (x,y) -> (-sign*y, sign*x)
__device__ __forceinline__ float2 mul_i(float2 a, float sign) { return make_float2(-sign * a.y, sign * a.x); }

__device__ __forceinline__ void dft4(float2* u, float sign)
{
    dft2(u[0], u[2]);
    dft2(u[1], u[3]);
    u[3] = mul_i(u[3], sign);
    dft2(u[0], u[1]);
    dft2(u[2], u[3]);
    float2 t = u[1]; u[1] = u[2]; u[2] = t;          // bit reversal -> natural order
}

__device__ __forceinline__ void dft8(float2* u, float sign)
{
    const float h = 0.70710678118654752440f;
    dft2(u[0], u[4]); dft2(u[1], u[5]); dft2(u[2], u[6]); dft2(u[3], u[7]);
    // twiddles W8^k (sign): k=1: (1+sign*i)/sqrt2, k=2: sign*i, k=3: (-1+sign*i)/sqrt2
    u[5] = make_float2(h * (u[5].x - sign * u[5].y), h * (u[5].y + sign * u[5].x));
    u[6] = mul_i(u[6], sign);
    u[7] = make_float2(h * (-u[7].x - sign * u[7].y), h * (-u[7].y + sign * u[7].x));
    dft2(u[0], u[2]); dft2(u[1], u[3]);
    u[3] = mul_i(u[3], sign);
    dft2(u[4], u[6]); dft2(u[5], u[7]);
    u[7] = mul_i(u[7], sign);
    dft2(u[0], u[1]); dft2(u[2], u[3]); dft2(u[4], u[5]); dft2(u[6], u[7]);
    float2 t;
    t = u[1]; u[1] = u[4]; u[4] = t;                 // bit reversal 1<->4, 3<->6
    t = u[3]; u[3] = u[6]; u[6] = t;
}

template <int R>
__device__ __forceinline__ void dftR(float2* u, float sign)
{
    if (R == 2) dft2(u[0], u[1]);
    else if (R == 4) dft4(u, sign);
    else dft8(u, sign);
}

// One Stockham pass of radix R over `nfft` sequences of length N (rows of `pitch` float2):
// butterfly i of a row: k = i mod p, inputs in[i + j*N/R] * W_{pR}^{jk}, outputs out[(i-k)R + k + j p].
template <int R>
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ in, float2* __restrict__ out,
                                              int N, int p, int nfft, int pitch, float sign)
{
    const int T = N / R;
    for (int idx = threadIdx.x; idx < nfft * T; idx += blockDim.x) {
        int row = idx / T, i = idx - row * T;
        int k = i & (p - 1);
        const float2* src = in + row * pitch;
        float2* dst = out + row * pitch;
        float2 u[R];
#pragma unroll
        for (int j = 0; j < R; j++) u[j] = src[i + j * T];
        if (p > 1) {
            // W^{jk}, j = 1..R-1, from one sincospif and products of depth <= 3 (w2 = w1 w1, w3 = w2 w1,
            // w4 = w2 w2, w5 = w4 w1, w6 = w3 w3, w7 = w4 w3): a few 1e-8 of extra error, 6 fewer sincospif
            float2 w[R];
            w[1] = twiddle(k, p * R, sign);
            if (R > 2) { w[2] = cmul_pk(w[1], w[1]); w[3] = cmul_pk(w[2], w[1]); }
            if (R > 4) { w[4] = cmul_pk(w[2], w[2]); w[5] = cmul_pk(w[4], w[1]); w[6] = cmul_pk(w[3], w[3]); w[7] = cmul_pk(w[4], w[3]); }
#pragma unroll
            for (int j = 1; j < R; j++) u[j] = cmul_pk(u[j], w[j]);
        }
        dftR<R>(u, sign);
        int j0 = (i - k) * R + k;
#pragma unroll
        for (int j = 0; j < R; j++) dst[j0 + j * p] = u[j];
    }
}

// FFT of `nfft` rows of length N (power of two >= 2) held in smem buffer `a`; `b` is a second
// buffer of the same size. Returns the buffer holding the result. All threads must call.
__device__ __forceinline__ float2* smem_fft(float2* a, float2* b, int N, int nfft, int pitch, float sign)
{
    int p = 1;
    while (N / p >= 8) {
        __syncthreads();
        stockham_pass<8>(a, b, N, p, nfft, pitch, sign);
        p *= 8;
        float2* t = a; a = b; b = t;
    }
    if (N / p == 4) {
        __syncthreads();
        stockham_pass<4>(a, b, N, p, nfft, pitch, sign);
        float2* t = a; a = b; b = t;
    } else if (N / p == 2) {
        __syncthreads();
        stockham_pass<2>(a, b, N, p, nfft, pitch, sign);
        float2* t = a; a = b; b = t;
    }
    __syncthreads();
    return a;
}
