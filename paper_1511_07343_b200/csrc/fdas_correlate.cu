// fdas_correlate.cu -- PAPER.md:49 steps 3-7 fused in one kernel (SURVEY §8 rows a2-a6, a6'):
// overlap-save window of the spectrum -> forward FFT_L -> for every template: pointwise
// multiply by its spectrum (1/L folded in), inverse FFT_L, |.|^2, keep the first `step`
// outputs -> plane row and/or thresholded candidates.  Computes Eq. (1).
#include "fdas_common.cuh"
#include "fdas_smemfft.cuh"
#include "fdas_regfft.cuh"
#include "fdas_tma.cuh"

// Generic segment length (L != 2048; natural-order smem Stockham): one CTA per (segment, batch entry).
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
        for (int o0 = 0; o0 < nvalid; o0 += blockDim.x) {                 // every warp stays converged (ballot below)
            const int o = o0 + threadIdx.x;
            const bool in = o < nvalid;
            float2 v = in ? y[o] : make_float2(0.f, 0.f);
            float pw = fmaf(v.x, v.x, v.y * v.y);
            int col = (c0 + o) * nset + s;
            if (plane && in) plane[((size_t)bt * n_z + zi) * n_cols + col] = pw;
            if (cands) push_cand_warp(cands + (size_t)bt * cap, counts + bt, cap, in && pw > thr, col, zi, 1, pw);
        }
    }
}


// ---------------------------------------------------------------------------------------------
// L = 2048: register-resident 16 x 16 x 8 FFTs, 128 threads (4 warps) per CTA, 16 points per
// thread.  Index split (inverse, DIT):  k = 128 k1 + 8 k2 + k3,  t = t1 + 16 t2 + 256 t3:
//   pass 1  thread (k2,k3): Y[k1] = X[k1] W[k1], 16-point DFT over k1 -> t1          (no twiddles)
//   ex1     [k3][t1][k2], intra-warp (a warp owns two k3 values)
//   pass 2  thread (t1,k3): twiddle exp(2 pi i k2 t1/256), 16-point DFT over k2 -> t2
//   ex2     [k3][t2][t1], block barrier
//   pass 3  two adjacent outputs p per thread: twiddle exp(2 pi i k3 p/2048), 8-point DFT
//           over k3 -> t3;  |.|^2;  coalesced store of t = p + 256 t3 < step.
// The forward transform of the window runs the same passes in reverse (once per segment) and
// leaves X[128 k1 + 8 k2 + k3] in the registers pass 1 needs; the template spectra are stored
// in that same register layout (Wr), so nothing is reordered in the template loop.
// The segment spectrum X stays in registers across all templates ("data reuse").
constexpr int SEG_THREADS = 128;

// out of line: the fused-threshold append is rare (called by all 32 lanes of a warp, see push_cand_warp)
__device__ __noinline__ void push_cand_seg(fdas_cand* list, uint32_t* count, uint32_t cap, bool hit,
                                           int col, int zi, float power)
{
    push_cand_warp(list, count, cap, hit, col, zi, 1, power);
}

// Instruction economy of the template loop (cuobjdump: see DESIGN.md section 6.1):
//   * the template multiply is folded into the first butterfly stage (mul_first_stage16);
//   * exchange 1 rows have pitch 18 float2 (16-byte aligned), so pass 2 reads its 16 inputs with
//     8 LDS.128 (quarter-warp bank pattern 4 lo + 4 j: conflict-free);
//   * pass 3 owns the ADJACENT outputs p = 2 tid, 2 tid + 1: 8 LDS.128 from exchange 2, and for
//     integer-bin planes 8-byte stores of two neighbouring columns;
//   * PK: the butterflies use the packed f32x2 instructions of sm_100 (FFMA2/FADD2/FMUL2, fdas_regfft.cuh): the
//     same operations per component in the same order (bit-identical planes), ~15 % fewer issue slots;
//   * FAST (launched when step is a multiple of 256): a full segment keeps exactly t3 < step/256
//     for every thread, so its stores are unpredicated and the butterflies feeding the discarded
//     t3 = 7 outputs are dead code; the ragged last segment takes the predicated path.
constexpr int SEG_PITCH3 = 288;                 // float2 per k3 region: 16 rows of pitch 18
constexpr int SEG_BUF = 8 * SEG_PITCH3;

// Pass 3 of one template for this thread's outputs p = 2 tid (u0) and 2 tid + 1 (u1), t = p + 256 t3:
// 8 LDS.128 from exchange 2, two 8-point DITs over k3, |.|^2, store / threshold.
// FULL (CTA-uniform): every thread keeps exactly t3 < NKEEP, so nothing is predicated and the work
// feeding t3 >= NKEEP is dead code; otherwise t3 < nv (ragged last segment, or step not a multiple of 256).
template <bool HAS_PLANE, bool HAS_CANDS, int NSET, int NKEEP, bool FULL, bool PK>
__device__ __forceinline__ void seg_pass3(const float2* buf, const float2* tw_a, const float2* tw_b, int tid,
                                         float* prow, int nv, fdas_cand* cands, uint32_t* counts, uint32_t cap,
                                         float thr, int col0, int zi)
{
    float2 u0[8], u1[8];
#pragma unroll
    for (int k3 = 0; k3 < 8; k3++) {
        const float4 q = *reinterpret_cast<const float4*>(buf + 2 * tid + SEG_PITCH3 * k3);
        u0[bitrev(k3, 3)] = make_float2(q.x, q.y);
        u1[bitrev(k3, 3)] = make_float2(q.z, q.w);
    }
    dit_tw<8, PK>(u0, tw_a);
    dit_tw<8, PK>(u1, tw_b);
    float pa[8], pb[8];
    float mx = 0.0f;                                   // largest kept power of this thread (fused threshold: one test)
#pragma unroll
    for (int t3 = 0; t3 < 8; t3++) {
        if (FULL && t3 >= NKEEP) continue;             // compile time: the butterflies feeding these outputs are dead code
        const bool kept = FULL || t3 < nv;
        pa[t3] = fmaf(u0[t3].x, u0[t3].x, u0[t3].y * u0[t3].y);
        pb[t3] = fmaf(u1[t3].x, u1[t3].x, u1[t3].y * u1[t3].y);
        if (HAS_PLANE && kept) {
            if (NSET == 1) *reinterpret_cast<float2*>(prow + 256 * t3) = make_float2(pa[t3], pb[t3]);
            else { prow[(256 * t3) * NSET] = pa[t3]; prow[(256 * t3 + 1) * NSET] = pb[t3]; }
        }
        if (HAS_CANDS && kept) mx = fmaxf(mx, fmaxf(pa[t3], pb[t3]));
    }
    if (HAS_CANDS && __any_sync(0xffffffffu, mx > thr)) {      // rare; warp-uniform, so the ballots below see all 32 lanes
#pragma unroll
        for (int t3 = 0; t3 < 8; t3++) {
            if (FULL && t3 >= NKEEP) continue;
            const bool kept = FULL || t3 < nv;
            push_cand_seg(cands, counts, cap, kept && pa[t3] > thr, col0 + 256 * t3 * NSET, zi, pa[t3]);
            push_cand_seg(cands, counts, cap, kept && pb[t3] > thr, col0 + (256 * t3 + 1) * NSET, zi, pb[t3]);
        }
    }
}

// Per-thread constants of the segment kernels: the 14 + 15 twiddles of the forward transform and the 16 of the inverse
// passes depend on the thread index only, so they are computed ONCE with the bank (same device functions: the planes do
// not change by a bit) instead of 45 sincospif per thread in the prologue of every CTA (~1350 of its ~2000 instructions,
// i.e. ~8 % of a 29-template CTA).  Entry e of thread tid is the float2 half (e & 1) of table[(e >> 1) * 128 + tid]:
//   e =  0..6   exp(-2 pi i k3 tid / 2048),         k3 = 1..7        (forward pass over n3, p = tid)
//   e =  7..13  exp(-2 pi i k3 (tid + 128) / 2048)                    (p = tid + 128)
//   e = 14..28  exp(-2 pi i k2 lo / 256),           k2 = 1..15, lo = tid & 15
//   e = 29..36  make_tw<16>(lo, 256);  e = 37..40  make_tw<8>(2 tid, 2048);  e = 41..44  make_tw<8>(2 tid + 1, 2048)
constexpr int SEG_TW_ENTRIES = 46;                 // 45 used, padded to whole float4
constexpr int SEG_TW_FLOAT4 = SEG_TW_ENTRIES / 2 * SEG_THREADS;

__global__ void __launch_bounds__(SEG_THREADS)
k_segment_twiddles(float4* __restrict__ table)
{
    const int tid = threadIdx.x, lo = tid & 15;
    float2 e[SEG_TW_ENTRIES];
#pragma unroll
    for (int k3 = 1; k3 < 8; k3++) {
        e[k3 - 1] = twiddle(k3 * tid, 2048, -1.0f);
        e[6 + k3] = twiddle(k3 * (tid + 128), 2048, -1.0f);
    }
#pragma unroll
    for (int k2 = 1; k2 < 16; k2++) e[13 + k2] = twiddle(k2 * lo, 256, -1.0f);
    make_tw<16>(e + 29, lo, 256);
    make_tw<8>(e + 37, 2 * tid, 2048);
    make_tw<8>(e + 41, 2 * tid + 1, 2048);
    e[45] = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int j = 0; j < SEG_TW_ENTRIES / 2; j++) table[j * SEG_THREADS + tid] = make_float4(e[2 * j].x, e[2 * j].y, e[2 * j + 1].x, e[2 * j + 1].y);
}

// entry e (compile time after unrolling) of this thread; the two halves of a float4 share one load
__device__ __forceinline__ float2 seg_tw(const float4* __restrict__ table, int tid, int e)
{
    const float4 q = __ldg(table + (e >> 1) * SEG_THREADS + tid);
    return (e & 1) ? make_float2(q.z, q.w) : make_float2(q.x, q.y);
}

// Shared state of the STAGED variant (k_correlate_2048_staged): NG segments ("groups" of 128 threads) per CTA take
// every template spectrum from a two-slot ring in shared memory that ONE thread fills with 16 KB bulk copies
// (cp.async.bulk, fdas_tma.cuh).  full[b]: the copy into slot b has landed (1 arrival + 16384 bytes);
// empty[b]: every warp of the CTA has copied slot b into its registers (4 NG arrivals).
struct SegStage {
    const float4* wbuf;       // [2][8 * SEG_THREADS]
    uint64_t* full;           // [2]
    uint64_t* empty;          // [2]
    uint32_t* status;
    int group;                // 0 .. NG-1 (the named barrier of the group is 1 + group)
    bool producer;            // thread 0 of the CTA
};

// One overlap-save segment against the templates [t_begin, t_end): the body of both kernels.  NG == 1: the
// 128-thread CTA of k_correlate_2048 (template spectra by LDG from L2/L1, __syncthreads).  NG > 1: one group of
// the staged kernel (template spectra from the ring, group barriers).  `tid` is the thread's index in its group.
template <bool HAS_PLANE, bool HAS_CANDS, int NSET, int NKEEP, bool PK, int NG>
__device__ __forceinline__ void correlate_segment(float2* sm, const int tid, const int seg, const int bt, const int t_begin,
                                                  const int t_end, const float2* __restrict__ spec,
                                                  const float4* __restrict__ Wr, const float4* __restrict__ twt,
                                                  float* __restrict__ plane, fdas_cand* __restrict__ cands,
                                                  uint32_t* __restrict__ counts, uint32_t cap, float thr, int n_bins, int n_z,
                                                  int m, int step, const SegStage& stg)
{
    constexpr int L = 2048;
    constexpr int nset = NSET;
    const int lo = tid & 15, k3A = tid >> 4;
    auto group_barrier = [&]() {
        if constexpr (NG == 1) __syncthreads();
        else named_bar_sync(1 + stg.group, SEG_THREADS);
    };
    const int c0 = seg * step;
    const float2* S = spec + (size_t)bt * n_bins;

    float2 X[16];
    {   // ---- forward FFT of the window (sign -), reverse pass order
        float2* buf = sm;
#pragma unroll
        for (int g = 0; g < 2; g++) {
            const int p = tid + 128 * g;
            float2 u[8];
#pragma unroll
            for (int n3 = 0; n3 < 8; n3++) {
                long long c = (long long)c0 - m / 2 + p + 256 * n3;
                u[bitrev(n3, 3)] = (c >= 0 && c < n_bins) ? S[c] : make_float2(0.f, 0.f);
            }
            dit_const<8, -1, PK>(u);
#pragma unroll
            for (int k3 = 0; k3 < 8; k3++) {
                float2 val = k3 ? cmul(u[k3], seg_tw(twt, tid, 7 * g + k3 - 1)) : u[0];
                buf[p + SEG_PITCH3 * k3] = val;
            }
        }
        group_barrier();
        float2 v[16];
#pragma unroll
        for (int n2 = 0; n2 < 16; n2++) v[bitrev(n2, 4)] = buf[lo + 16 * n2 + SEG_PITCH3 * k3A];
        dit_const<16, -1, PK>(v);
#pragma unroll
        for (int k2 = 1; k2 < 16; k2++) v[k2] = cmul(v[k2], seg_tw(twt, tid, 13 + k2));
        __syncwarp();
#pragma unroll
        for (int k2 = 0; k2 < 16; k2++) buf[k2 + 18 * lo + SEG_PITCH3 * k3A] = v[k2];
        __syncwarp();
#pragma unroll
        for (int n1 = 0; n1 < 16; n1++) v[bitrev(n1, 4)] = buf[lo + 18 * n1 + SEG_PITCH3 * k3A];
        dit_const<16, -1, PK>(v);
#pragma unroll
        for (int k1 = 0; k1 < 16; k1++) X[k1] = v[k1];
        group_barrier();
    }

    float2 tw2[8], tw3[2][4];                                      // inverse-pass twiddles (loop invariant), from the table
#pragma unroll
    for (int i = 0; i < 8; i++) tw2[i] = seg_tw(twt, tid, 29 + i);
#pragma unroll
    for (int i = 0; i < 4; i++) {
        tw3[0][i] = seg_tw(twt, tid, 37 + i);
        tw3[1][i] = seg_tw(twt, tid, 41 + i);
    }

    const size_t n_cols = (size_t)n_bins * nset;
    const int omax = min(step, n_bins - c0);                       // even: step, n_bins and c0 are even
    const bool full = (NKEEP < 8) && omax == step;                 // CTA-uniform
    const int nv = max(0, min(8, (omax - 2 * tid + 255) >> 8));    // kept t3 of BOTH p = 2 tid and 2 tid + 1
    float* pbase = HAS_PLANE ? plane + (size_t)bt * n_z * n_cols + (size_t)(c0 + 2 * tid) * nset : nullptr;
    fdas_cand* clist = HAS_CANDS ? cands + (size_t)bt * cap : nullptr;
    uint32_t* ccount = HAS_CANDS ? counts + bt : nullptr;

    float4 w4[8];
    const float4* Wn = Wr + (size_t)t_begin * (8 * SEG_THREADS) + tid;      // template whose spectrum is fetched next
    if constexpr (NG == 1) {
        if (t_begin < t_end) {
#pragma unroll
            for (int j = 0; j < 8; j++) w4[j] = __ldg(Wn + j * SEG_THREADS);
        }
    }
    float* prow1 = HAS_PLANE ? pbase + (size_t)t_begin * n_cols : nullptr;  // NSET == 1: row of template t
    for (int t = t_begin; t < t_end; t++) {
        float2* buf = sm + ((t - t_begin) & 1) * SEG_BUF;
        if constexpr (NG > 1) {                                                  // slot b = use k of the ring: parity k & 1
            const int b = (t - t_begin) & 1, k = (t - t_begin) >> 1;
            if (!mbar_wait(stg.full + b, k & 1, stg.status)) return;
            const float4* ws = stg.wbuf + b * (8 * SEG_THREADS) + tid;
#pragma unroll
            for (int j = 0; j < 8; j++) w4[j] = ws[j * SEG_THREADS];
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(stg.empty + b);
        }
        float2 v[16];
        if (PK) mul_first_stage16_pk(v, X, w4);                                  // X W and stage 1
        else mul_first_stage16(v, X, w4);
        dit_const_stage<16, +1, 2, PK>(v);                                       // pass 1: k1 -> t1
        dit_const_stage<16, +1, 3, PK>(v);
        dit_const_stage<16, +1, 4, PK>(v);
#pragma unroll
        for (int t1 = 0; t1 < 16; t1++) buf[lo + 18 * t1 + SEG_PITCH3 * k3A] = v[t1];
        __syncwarp();
        {
            const float4* row = reinterpret_cast<const float4*>(buf + 18 * lo + SEG_PITCH3 * k3A);
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const float4 q = row[j];
                v[bitrev(2 * j, 4)] = make_float2(q.x, q.y);
                v[bitrev(2 * j + 1, 4)] = make_float2(q.z, q.w);
            }
        }
        dit_tw<16, PK>(v, tw2);                                                  // pass 2: k2 -> t2
        __syncwarp();
#pragma unroll
        for (int t2 = 0; t2 < 16; t2++) buf[lo + 16 * t2 + SEG_PITCH3 * k3A] = v[t2];
        if constexpr (NG == 1) {
            if (t + 1 < t_end) Wn += 8 * SEG_THREADS;                             // (the last iteration re-reads its own)
#pragma unroll
            for (int j = 0; j < 8; j++) w4[j] = __ldg(Wn + j * SEG_THREADS);
        } else if (stg.producer && t + 2 < t_end) {                               // refill this iteration's slot with template t + 2
            const int b = (t - t_begin) & 1, k = (t - t_begin) >> 1;
            // (on a time-out nothing is issued and nobody leaves alone: every thread then gives up together at the
            // next wait for this slot, so that no group is left short at its named barrier)
            if (mbar_wait(stg.empty + b, k & 1, stg.status)) {
                mbar_expect_tx(stg.full + b, 8 * SEG_THREADS * 16);
                tma_load_1d(const_cast<float4*>(stg.wbuf) + b * (8 * SEG_THREADS), Wr + (size_t)(t + 2) * (8 * SEG_THREADS),
                            8 * SEG_THREADS * 16, stg.full + b);
            }
        }
        group_barrier();
        const int zi = NSET == 1 ? t : (t >> 1), s = NSET == 1 ? 0 : (t & 1);
        float* prow = !HAS_PLANE ? nullptr : NSET == 1 ? prow1 : pbase + (size_t)zi * n_cols + s;
        if (HAS_PLANE && NSET == 1) prow1 += n_cols;
        const int col0 = (c0 + 2 * tid) * nset + s;
        if (full)                                                                // pass 3: k3 -> t3
            seg_pass3<HAS_PLANE, HAS_CANDS, NSET, NKEEP, true, PK>(buf, tw3[0], tw3[1], tid, prow, nv, clist, ccount, cap, thr, col0, zi);
        else
            seg_pass3<HAS_PLANE, HAS_CANDS, NSET, 8, false, PK>(buf, tw3[0], tw3[1], tid, prow, nv, clist, ccount, cap, thr, col0, zi);
    }
}


template <bool HAS_PLANE, bool HAS_CANDS, int NSET, int NKEEP, bool PK>
__global__ void __launch_bounds__(SEG_THREADS, 3)
k_correlate_2048(const float2* __restrict__ spec, const float4* __restrict__ Wr, const float4* __restrict__ twt,
                 float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ counts, uint32_t cap, float thr,
                 int n_bins, int n_z, int m, int step, int t_chunk)
{
    __shared__ __align__(16) float2 sm[2 * SEG_BUF];
    const int n_t = n_z * NSET;
    const int t_begin = blockIdx.y * t_chunk, t_end = min(n_t, t_begin + t_chunk);
    correlate_segment<HAS_PLANE, HAS_CANDS, NSET, NKEEP, PK, 1>(sm, threadIdx.x, blockIdx.x, blockIdx.z, t_begin, t_end, spec, Wr,
                                                                 twt, plane, cands, counts, cap, thr, n_bins, n_z, m, step, SegStage{});
}

// STAGED variant (tuning key FDAS_OPT_TUNE_STAGE_TEMPLATES; SURVEY section 7 hard part 2, "several segments per
// template load"): one CTA = SEG_GROUPS groups of 128 threads = SEG_GROUPS adjacent segments; every template
// spectrum crosses L2 -> SM ONCE per CTA, as a 16 KB bulk copy (UBLKCP) into a two-slot ring, instead of once
// per segment: 0.8 GB instead of up to 3.3 GB per DM trial at configs[2], whatever L1 does.  Groups run
// independently between ring accesses (their own exchange buffers and named barrier).  A group whose segment
// lies beyond the series (last CTA) only keeps the ring protocol going.
// dynamic shared memory: ring [2][16 KB] | exchange buffers [SEG_GROUPS][2][SEG_BUF] | 4 mbarriers.
constexpr int SEG_GROUPS = 4;
constexpr int SEG_RING_BYTES = 2 * 8 * SEG_THREADS * 16;
constexpr int SEG_STAGED_SMEM = SEG_RING_BYTES + SEG_GROUPS * 2 * SEG_BUF * 8 + 128;

template <bool HAS_PLANE, bool HAS_CANDS, int NSET, int NKEEP, bool PK>
__global__ void __launch_bounds__(SEG_GROUPS* SEG_THREADS, 1)
k_correlate_2048_staged(const float2* __restrict__ spec, const float4* __restrict__ Wr, const float4* __restrict__ twt,
                        float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ counts, uint32_t cap, float thr,
                        int n_bins, int n_z, int m, int step, int t_chunk, int n_seg, uint32_t* status)
{
    extern __shared__ __align__(128) float2 dsm[];
    float4* ring = reinterpret_cast<float4*>(dsm);
    float2* exch = dsm + SEG_RING_BYTES / 8;
    uint64_t* bars = reinterpret_cast<uint64_t*>(exch + SEG_GROUPS * 2 * SEG_BUF);
    const int group = threadIdx.x / SEG_THREADS, tid = threadIdx.x % SEG_THREADS;
    const int n_t = n_z * NSET;
    const int t_begin = blockIdx.y * t_chunk, t_end = min(n_t, t_begin + t_chunk);
    SegStage stg;
    stg.wbuf = ring; stg.full = bars; stg.empty = bars + 2; stg.status = status; stg.group = group;
    stg.producer = threadIdx.x == 0;
    if (threadIdx.x == 0) {
        for (int b = 0; b < 2; b++) {
            mbar_init(stg.full + b, 1);
            mbar_init(stg.empty + b, SEG_GROUPS * SEG_THREADS / 32);
        }
        mbar_fence_init();
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int b = 0; b < 2 && t_begin + b < t_end; b++) {
            mbar_expect_tx(stg.full + b, 8 * SEG_THREADS * 16);
            tma_load_1d(ring + b * (8 * SEG_THREADS), Wr + (size_t)(t_begin + b) * (8 * SEG_THREADS), 8 * SEG_THREADS * 16,
                        stg.full + b);
        }
    }
    const int seg = blockIdx.x * SEG_GROUPS + group;
    if (seg < n_seg) {
        correlate_segment<HAS_PLANE, HAS_CANDS, NSET, NKEEP, PK, SEG_GROUPS>(exch + group * 2 * SEG_BUF, tid, seg, blockIdx.z, t_begin,
                                                                           t_end, spec, Wr, twt, plane, cands, counts, cap, thr,
                                                                           n_bins, n_z, m, step, stg);
    } else {                                   // no segment: consume the ring so that the producer's waits complete
        for (int t = t_begin; t < t_end; t++) {
            const int b = (t - t_begin) & 1, k = (t - t_begin) >> 1;
            if (!mbar_wait(stg.full + b, k & 1, status)) return;
            __syncwarp();
            if ((tid & 31) == 0) mbar_arrive(stg.empty + b);
        }
    }
}

// Wr[(t*8 + j)*128 + tid] = (W[128(2j) + 8 k2 + k3], W[128(2j+1) + 8 k2 + k3]), tid = 16 k3 + k2.
__global__ void k_permute_templates_2048(const float2* __restrict__ W, float4* __restrict__ Wr, int n_t)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_t * 8 * SEG_THREADS) return;
    int tid = i % SEG_THREADS, j = (i / SEG_THREADS) % 8, t = i / (8 * SEG_THREADS);
    int k2 = tid & 15, k3 = tid >> 4;
    float2 a = W[(size_t)t * 2048 + 128 * (2 * j) + 8 * k2 + k3];
    float2 b = W[(size_t)t * 2048 + 128 * (2 * j + 1) + 8 * k2 + k3];
    Wr[i] = make_float4(a.x, a.y, b.x, b.y);
}

int fdas_permute_templates(fdas_plan* p, cudaStream_t st)
{
    if (p->L != 2048) return FDAS_OK;
    int n = p->n_t * 8 * SEG_THREADS;
    k_permute_templates_2048<<<(n + 255) / 256, 256, 0, st>>>(p->d_W, reinterpret_cast<float4*>(p->d_Wr), p->n_t);
    FDAS_LAUNCH_CHECK();
    k_segment_twiddles<<<1, SEG_THREADS, 0, st>>>(reinterpret_cast<float4*>(p->d_segtw));
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

int fdas_launch_correlate(fdas_plan* p, const float2* d_spec, int n_batch, float* d_plane, float thr,
                          fdas_cand* d_cands, uint32_t* d_counts, uint32_t cap, cudaStream_t st)
{
    if (d_cands) FDAS_CUDA(cudaMemsetAsync(d_counts, 0, sizeof(uint32_t) * n_batch, st));
    if (p->L == 2048) {
        // Template chunks per segment.  A single series (2341 segments at 2^23 samples) needs ~29 templates per CTA to
        // fill 148 SMs x 3 CTAs for many waves (short tail), at the price of one forward FFT per chunk (+3.5 %).  A batch
        // that gives >= 20 waves by itself (configs[3]: 64 series) lets one CTA own ALL templates of its segment: the
        // forward FFT and the twiddle set-up are done once per segment (SURVEY section 7 hard part 2).
        const long long slots = 3LL * (p->n_sms > 0 ? p->n_sms : 148);
        const bool one_chunk = (long long)p->n_seg * n_batch >= 20 * slots;
        int n_chunk = p->tune_t_chunks > 0 ? p->tune_t_chunks : one_chunk ? 1 : (p->n_t + 28) / 29;
        int t_chunk = (p->n_t + n_chunk - 1) / n_chunk;
        n_chunk = (p->n_t + t_chunk - 1) / t_chunk;
        dim3 grid(p->n_seg, n_chunk, n_batch);
#define FDAS_SEG_ARGS d_spec, reinterpret_cast<const float4*>(p->d_Wr), reinterpret_cast<const float4*>(p->d_segtw), d_plane, d_cands, d_counts, cap, thr, \
                      (int)p->n_bins, p->n_z, p->m, p->step, t_chunk
#define FDAS_SEG_LAUNCH(...)                                                                                        \
        if (d_plane && d_cands) k_correlate_2048<true, true, __VA_ARGS__><<<grid, SEG_THREADS, 0, st>>>(FDAS_SEG_ARGS); \
        else if (d_plane) k_correlate_2048<true, false, __VA_ARGS__><<<grid, SEG_THREADS, 0, st>>>(FDAS_SEG_ARGS);      \
        else k_correlate_2048<false, true, __VA_ARGS__><<<grid, SEG_THREADS, 0, st>>>(FDAS_SEG_ARGS)
        const bool scalar = p->tune_scalar != 0;                  // scalar FFMA butterflies (tuning key; bit-identical planes)
        if (p->tune_stage_templates && !scalar) {                 // several segments per template load (see k_correlate_2048_staged)
            dim3 sgrid((p->n_seg + SEG_GROUPS - 1) / SEG_GROUPS, n_chunk, n_batch);
#define FDAS_STG_LAUNCH(...)                                                                                                   \
            do {                                                                                                               \
                FDAS_CUDA(cudaFuncSetAttribute(k_correlate_2048_staged<__VA_ARGS__>, cudaFuncAttributeMaxDynamicSharedMemorySize, \
                                               SEG_STAGED_SMEM));                                                              \
                k_correlate_2048_staged<__VA_ARGS__><<<sgrid, SEG_GROUPS * SEG_THREADS, SEG_STAGED_SMEM, st>>>(                \
                    FDAS_SEG_ARGS, p->n_seg, p->d_status);                                                                     \
            } while (0)
#define FDAS_STG_LAUNCH_NS(NS, NK)                                                           \
            if (d_plane && d_cands) FDAS_STG_LAUNCH(true, true, NS, NK, true);               \
            else if (d_plane) FDAS_STG_LAUNCH(true, false, NS, NK, true);                    \
            else FDAS_STG_LAUNCH(false, true, NS, NK, true)
            const bool k7 = p->step == 7 * 256;
            if (p->nset == 1) { if (k7) { FDAS_STG_LAUNCH_NS(1, 7); } else { FDAS_STG_LAUNCH_NS(1, 8); } }
            else { if (k7) { FDAS_STG_LAUNCH_NS(2, 7); } else { FDAS_STG_LAUNCH_NS(2, 8); } }
#undef FDAS_STG_LAUNCH_NS
#undef FDAS_STG_LAUNCH
            FDAS_LAUNCH_CHECK();
            return FDAS_OK;
        }
        const bool keep7 = p->step == 7 * 256;                    // m = 256: full segments keep t3 < 7 exactly
#define FDAS_SEG_LAUNCH_NS(NS)                                                                   \
        if (keep7 && !scalar) { FDAS_SEG_LAUNCH(NS, 7, true); }                                  \
        else if (keep7) { FDAS_SEG_LAUNCH(NS, 7, false); }                                       \
        else if (!scalar) { FDAS_SEG_LAUNCH(NS, 8, true); }                                      \
        else { FDAS_SEG_LAUNCH(NS, 8, false); }
        if (p->nset == 1) {
            FDAS_SEG_LAUNCH_NS(1)
        } else {
            FDAS_SEG_LAUNCH_NS(2)
        }
#undef FDAS_SEG_LAUNCH_NS
#undef FDAS_SEG_LAUNCH
#undef FDAS_SEG_ARGS
        FDAS_LAUNCH_CHECK();
        return FDAS_OK;
    }
    size_t smem = 3 * (size_t)p->L * sizeof(float2);
    FDAS_CUDA(cudaFuncSetAttribute(k_correlate_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_correlate_smem<<<dim3(p->n_seg, n_batch), 256, smem, st>>>(d_spec, p->d_W, d_plane, d_cands, d_counts, cap, thr,
                                                                  (int)p->n_bins, p->n_z, p->nset, p->m, p->L, p->step);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

int fdas_occupancy_correlate(int which, int32_t* ctas, int32_t* regs, int32_t* smem)
{
    if (which == 0) return fdas_occupancy_of(k_correlate_2048<true, false, 1, 7, true>, SEG_THREADS, 0, ctas, regs, smem);
    if (which == 1) return fdas_occupancy_of(k_correlate_2048<false, true, 1, 7, true>, SEG_THREADS, 0, ctas, regs, smem);
    return fdas_occupancy_of(k_correlate_2048_staged<true, false, 1, 7, true>, SEG_GROUPS * SEG_THREADS, SEG_STAGED_SMEM, ctas, regs, smem);
}
