// fdas_regfft.cuh -- register-resident radix-8/16 DIT butterflies for the fused segment kernel.
//
// All transforms here are decimation-in-time on R = 2^s points held in registers v[0..R):
// the caller places input j in v[bitrev_s(j)] (a compile-time register renaming), the routine
// leaves output q in v[q].  Stage `span` combines (v[b+q], v[b+q+span/2]) with the twiddle
//   tau = w^(R/span) * omega_span^q ,  omega_n = exp(SIGN 2 pi i / n),
// where w is the per-thread inter-pass twiddle base (w = 1 for the first pass).  Every
// butterfly a +- tau b is 6 FMAs:  o0 = a + tau b (4 FMA),  o1 = 2a - o0 (2 FMA); twiddles
// 1 and +-i cost 4 adds.  Multiplication by i is folded into operand signs, so a radix-16
// pass needs only 8 independent twiddle values per thread (1+1+2+4), a radix-8 pass 4.
#pragma once
#include "fdas_common.cuh"

// bit reversal of a 3- or 4-bit index, written without a loop so that it folds after unrolling
__host__ __device__ constexpr int bitrev(int j, int bits)
{
    return bits == 4 ? (((j & 1) << 3) | ((j & 2) << 1) | ((j & 4) >> 1) | ((j & 8) >> 3))
                     : (((j & 1) << 2) | (j & 2) | ((j & 4) >> 2));
}

// cos / sin of 2 pi e / 16, e = 0..7
__device__ __forceinline__ constexpr float cos16(int e)
{
    return e == 0 ? 1.0f : e == 1 ? 0.92387953251128674f : e == 2 ? 0.70710678118654752f
         : e == 3 ? 0.38268343236508977f : e == 4 ? 0.0f : e == 5 ? -0.38268343236508977f
         : e == 6 ? -0.70710678118654752f : -0.92387953251128674f;
}
__device__ __forceinline__ constexpr float sin16(int e)
{
    return e == 0 ? 0.0f : e == 1 ? 0.38268343236508977f : e == 2 ? 0.70710678118654752f
         : e == 3 ? 0.92387953251128674f : e == 4 ? 1.0f : e == 5 ? 0.92387953251128674f
         : e == 6 ? 0.70710678118654752f : 0.38268343236508977f;
}

// (a, b) <- (a + tau b, a - tau b), tau = (c, s)
__device__ __forceinline__ void bfly(float2& a, float2& b, float c, float s)
{
    float r0 = fmaf(-s, b.y, fmaf(c, b.x, a.x));
    float i0 = fmaf(s, b.x, fmaf(c, b.y, a.y));
    b.x = fmaf(2.0f, a.x, -r0);
    b.y = fmaf(2.0f, a.y, -i0);
    a.x = r0;
    a.y = i0;
}
// tau = i * (c, s) = (-s, c)
__device__ __forceinline__ void bfly_i(float2& a, float2& b, float c, float s)
{
    float r0 = fmaf(-c, b.y, fmaf(-s, b.x, a.x));
    float i0 = fmaf(c, b.x, fmaf(-s, b.y, a.y));
    b.x = fmaf(2.0f, a.x, -r0);
    b.y = fmaf(2.0f, a.y, -i0);
    a.x = r0;
    a.y = i0;
}
__device__ __forceinline__ void bfly_1(float2& a, float2& b)
{
    float2 t = b;
    b = make_float2(a.x - t.x, a.y - t.y);
    a = make_float2(a.x + t.x, a.y + t.y);
}
// tau = SIGN * i
template <int SIGN>
__device__ __forceinline__ void bfly_pmi(float2& a, float2& b)
{
    float2 t = (SIGN > 0) ? make_float2(-b.y, b.x) : make_float2(b.y, -b.x);
    b = make_float2(a.x - t.x, a.y - t.y);
    a = make_float2(a.x + t.x, a.y + t.y);
}

// ---- the same butterflies with the packed f32x2 instructions of sm_100 (FFMA2 / FADD2 / FMUL2): a complex
// value is a natural (re, im) register pair, the twiddle components are broadcast (the .F32 operand form),
// i*b = (-b.y, b.x) is an operand swizzle + sign pattern, so a +- tau b is 3 issue slots instead of 6 and
// every component sees exactly the operations, in the order, of the scalar version (bit-identical results).
__device__ __forceinline__ float2 f2(float x, float y) { return make_float2(x, y); }
// -x by flipping the sign bit on the integer pipe: building i*b = (-b.y, b.x) then costs the FMA pipe nothing
// (a float negation would be an FADD there); exact, so results do not change.
__device__ __forceinline__ float negi(float x) { return __int_as_float(__float_as_int(x) ^ 0x80000000); }
__device__ __forceinline__ void bfly_pk(float2& a, float2& b, float c, float s)
{
    const float2 t = __ffma2_rn(f2(c, c), b, a);                               // a + c b
    const float2 o0 = __ffma2_rn(f2(s, s), f2(negi(b.y), b.x), t);             // + s (i b)
    b = __ffma2_rn(f2(2.0f, 2.0f), a, f2(-o0.x, -o0.y));
    a = o0;
}
__device__ __forceinline__ void bfly_i_pk(float2& a, float2& b, float c, float s)     // tau = i (c, s)
{
    const float2 t = __ffma2_rn(f2(-s, -s), b, a);
    const float2 o0 = __ffma2_rn(f2(c, c), f2(negi(b.y), b.x), t);
    b = __ffma2_rn(f2(2.0f, 2.0f), a, f2(-o0.x, -o0.y));
    a = o0;
}
__device__ __forceinline__ void bfly_1_pk(float2& a, float2& b)
{
    const float2 t = b;
    b = __fadd2_rn(a, f2(-t.x, -t.y));
    a = __fadd2_rn(a, t);
}
template <int SIGN>
__device__ __forceinline__ void bfly_pmi_pk(float2& a, float2& b)
{
    const float2 t = (SIGN > 0) ? f2(-b.y, b.x) : f2(b.y, -b.x);
    b = __fadd2_rn(a, f2(-t.x, -t.y));
    a = __fadd2_rn(a, t);
}

// one DIT stage (span = 2^ST) with constant twiddles omega_span^q
template <int R, int SIGN, int ST, bool PK = false>
__device__ __forceinline__ void dit_const_stage(float2* v)
{
    constexpr int span = 1 << ST, half = span >> 1;
#pragma unroll
    for (int b = 0; b < R; b += span) {
#pragma unroll
        for (int q = 0; q < half; q++) {
            const int e = q * (16 / span);           // omega_span^q = exp(SIGN 2 pi i e / 16), e in [0, 8)
            if (PK) {
                if (e == 0) bfly_1_pk(v[b + q], v[b + q + half]);
                else if (e == 4) bfly_pmi_pk<SIGN>(v[b + q], v[b + q + half]);
                else bfly_pk(v[b + q], v[b + q + half], cos16(e), SIGN > 0 ? sin16(e) : -sin16(e));
            } else {
                if (e == 0) bfly_1(v[b + q], v[b + q + half]);
                else if (e == 4) bfly_pmi<SIGN>(v[b + q], v[b + q + half]);
                else bfly(v[b + q], v[b + q + half], cos16(e), SIGN > 0 ? sin16(e) : -sin16(e));
            }
        }
    }
}

// DIT on R points (8 or 16), no inter-pass twiddle (w = 1): constants only.
template <int R, int SIGN, bool PK = false>
__device__ __forceinline__ void dit_const(float2* v)
{
    dit_const_stage<R, SIGN, 1, PK>(v);
    dit_const_stage<R, SIGN, 2, PK>(v);
    dit_const_stage<R, SIGN, 3, PK>(v);
    if constexpr (R >= 16) dit_const_stage<R, SIGN, 4, PK>(v);
}

// Template multiply folded into the first (span 2) stage of the 16-point inverse DIT:
//   v[bitrev(k1)], v[bitrev(k1 + 8)] <- X[k1] W[k1] +- X[k1+8] W[k1+8],  k1 = 0..7,
// with W[2j], W[2j+1] = (w4[j].xy, w4[j].zw).  p = X_a W_a (4 ops), o0 = p + X_b W_b (4 FMA),
// o1 = 2p - o0 (2 FMA): 10 ops per pair instead of 12.  Continue with stages 2..4 of dit_const<16, +1>.
__device__ __forceinline__ void mul_first_stage16(float2* v, const float2* X, const float4* w4)
{
#pragma unroll
    for (int k1 = 0; k1 < 8; k1++) {
        const float4 wa4 = w4[k1 >> 1], wb4 = w4[(k1 >> 1) + 4];
        const float2 wa = (k1 & 1) ? make_float2(wa4.z, wa4.w) : make_float2(wa4.x, wa4.y);
        const float2 wb = (k1 & 1) ? make_float2(wb4.z, wb4.w) : make_float2(wb4.x, wb4.y);
        const float2 a = X[k1], b = X[k1 + 8];
        const float pr = fmaf(a.x, wa.x, -a.y * wa.y);
        const float pi = fmaf(a.x, wa.y, a.y * wa.x);
        const float r0 = fmaf(-b.y, wb.y, fmaf(b.x, wb.x, pr));
        const float i0 = fmaf(b.y, wb.x, fmaf(b.x, wb.y, pi));
        const int o = bitrev(k1, 4);                 // even; bitrev(k1 + 8) = o + 1
        v[o] = make_float2(r0, i0);
        v[o + 1] = make_float2(fmaf(2.0f, pr, -r0), fmaf(2.0f, pi, -i0));
    }
}

// mul_first_stage16 with packed instructions (same operations per component, in the same order)
__device__ __forceinline__ void mul_first_stage16_pk(float2* v, const float2* X, const float4* w4)
{
#pragma unroll
    for (int k1 = 0; k1 < 8; k1++) {
        const float4 wa4 = w4[k1 >> 1], wb4 = w4[(k1 >> 1) + 4];
        const float2 wa = (k1 & 1) ? f2(wa4.z, wa4.w) : f2(wa4.x, wa4.y);
        const float2 wb = (k1 & 1) ? f2(wb4.z, wb4.w) : f2(wb4.x, wb4.y);
        const float2 a = X[k1], b = X[k1 + 8];
        const float2 m = __fmul2_rn(f2(a.y, a.y), f2(negi(wa.y), wa.x));       // (-a.y wa.y, a.y wa.x)
        const float2 pp = __ffma2_rn(f2(a.x, a.x), wa, m);                      // p = X_a W_a
        const float2 t = __ffma2_rn(f2(b.x, b.x), wb, pp);
        const float2 o0 = __ffma2_rn(f2(b.y, b.y), f2(negi(wb.y), wb.x), t);    // p + X_b W_b
        const int o = bitrev(k1, 4);
        v[o] = o0;
        v[o + 1] = __ffma2_rn(f2(2.0f, 2.0f), pp, f2(-o0.x, -o0.y));
    }
}

template <int R, int ST, bool PK = false>
__device__ __forceinline__ void dit_tw_stage(float2* v, const float2* tw)
{
    constexpr int span = 1 << ST, half = span >> 1;
    constexpr int nind = half >= 2 ? half / 2 : 1;
    constexpr int base = span == 2 ? 0 : half / 2;
#pragma unroll
    for (int b = 0; b < R; b += span) {
#pragma unroll
        for (int q = 0; q < half; q++) {
            if (PK) {
                if (q < nind) bfly_pk(v[b + q], v[b + q + half], tw[base + q].x, tw[base + q].y);
                else bfly_i_pk(v[b + q], v[b + q + half], tw[base + q - nind].x, tw[base + q - nind].y);
            } else {
                if (q < nind) bfly(v[b + q], v[b + q + half], tw[base + q].x, tw[base + q].y);
                else bfly_i(v[b + q], v[b + q + half], tw[base + q - nind].x, tw[base + q - nind].y);
            }
        }
    }
}

// DIT on R points with inter-pass twiddle base w (inverse sign, SIGN = +1).
// tw[] holds, for stage span = 2, 4, 8, 16: w^(R/span) * omega_span^q for q in [0, max(1, span/4)):
//   index 0: span 2;  1: span 4;  2..3: span 8;  4..7: span 16.   (the other q are i * these)
template <int R, bool PK = false>
__device__ __forceinline__ void dit_tw(float2* v, const float2* tw)
{
    dit_tw_stage<R, 1, PK>(v, tw);
    dit_tw_stage<R, 2, PK>(v, tw);
    dit_tw_stage<R, 3, PK>(v, tw);
    if constexpr (R >= 16) dit_tw_stage<R, 4, PK>(v, tw);
}

// Fill tw[] for dit_tw<R>: w = exp(2 pi i num / den)  (num/den exact in fp32).
template <int R>
__device__ __forceinline__ void make_tw(float2* tw, int num, int den)
{
#pragma unroll
    for (int st = 1; (1 << st) <= R; st++) {
        const int span = 1 << st;
        const int half = span >> 1;
        const int nind = half >= 2 ? half / 2 : 1;
        const int base = span == 2 ? 0 : half / 2;
#pragma unroll
        for (int q = 0; q < nind; q++) {
            // w^(R/span) * omega_span^q = exp(2 pi i (num (R/span)/den + q/span))
            float ph = (float)(num * (R / span)) / (float)den + (float)q / (float)span;
            float s, c;
            sincospif(2.0f * ph, &s, &c);
            tw[base + q] = make_float2(c, s);
        }
    }
}
