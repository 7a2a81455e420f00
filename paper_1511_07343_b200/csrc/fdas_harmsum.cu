// fdas_harmsum.cu -- incoherent harmonic summing and candidate compaction
// (BASELINE.json configs[4]; "pulse harmonics").
#include "fdas_common.cuh"
#include <stdlib.h>

struct HarmThr { float t[5]; };

// One CTA per tile of HS_COLS = 128 plane columns x all n_z rows: warp w walks rows w, w+8, ...; a lane
// owns the HS_CPT (2 or 4) cells col0 + lane + 32 j of the row.  S_1 = P; stage 2H adds the odd-h terms of
// fraction h/(2H) (the rounding rule is invariant under (h,H)->(2h,2H), so S_2H = S_H + odd terms).
//   k_h = floor((k h + H/2)/H), zeta_h = sgn(zeta) floor((|zeta| h + H/2)/H)   (include/fdas.h)
// Index arithmetic is done once per lane and row: stepping k by 32 moves k_h by exactly 32 h/H (an
// integer for H <= 16), so the other three cells reuse the first cell's source address plus a
// compile-time offset.  The 15 stretched streams of a tile touch ~4.84 x the tile's cells, each
// needed by ~1/f^2 cells of the tile; keeping whole columns of the tile in one CTA lets the L1 serve
// that reuse.  The f = 1 stream is read once (streaming load).
// grid = ceil(n_cols/(32 HS_CPT)), block = (32, 8).
constexpr int HS_ROWS_PER_PASS = 8;

__device__ __noinline__ void push_cand_hs(fdas_cand* list, uint32_t* count, uint32_t cap,
                                          int col, int zi, int nharm, float power)
{
    push_cand(list, count, cap, col, zi, nharm, power);
}

// CHECK = true: edge tiles (first tile: k_h may fall below bin0; last tile: columns beyond n_cols).
template <int NST, int HS_CPT, bool CHECK>
__device__ __forceinline__ void harmsum_tile(const float* __restrict__ plane, fdas_cand* __restrict__ cands,
                                             uint32_t* __restrict__ count, uint32_t cap, const HarmThr& thr,
                                             int n_cols, int n_z, int bin0)
{
    constexpr int HS_COLS = 32 * HS_CPT;
    const int col0 = blockIdx.x * HS_COLS + threadIdx.x;
    const int zc = (n_z - 1) / 2;
    const int k = bin0 + col0;
    constexpr int HMAX = 1 << (NST - 1);
    for (int zi = threadIdx.y; zi < n_z; zi += HS_ROWS_PER_PASS) {
        const int zeta = zi - zc, az = abs(zeta), sg = zeta < 0 ? -1 : 1;
        // issue every gather of the row's HS_CPT cells first (all independent), then sum in stage order
        float v[HS_CPT][HMAX];
        const float* prow = plane + (size_t)zi * n_cols + col0;
#pragma unroll
        for (int j = 0; j < HS_CPT; j++) v[j][0] = (!CHECK || col0 + 32 * j < n_cols) ? __ldcs(prow + 32 * j) : 0.0f;
#pragma unroll
        for (int st = 1; st < NST; st++) {
            const int H = 1 << st;
#pragma unroll
            for (int h = 1; h < H; h += 2) {
                const int kh = (k * h + (H >> 1)) >> st;              // k*h < 2^29 for n_samples <= 2^25
                const int zh = sg * ((az * h + (H >> 1)) >> st);
                const float* src = plane + (size_t)(zc + zh) * n_cols + (kh - bin0);
                const int dk = (32 * h) >> st;                         // exact: 32 h / H
#pragma unroll
                for (int j = 0; j < HS_CPT; j++) {
                    float x = 0.0f;
                    if (!CHECK || (kh + dk * j >= bin0 && col0 + 32 * j < n_cols)) x = __ldg(src + dk * j);
                    v[j][(H >> 1) + (h >> 1)] = x;                     // stage st occupies slots [H/2, H)
                }
            }
        }
#pragma unroll
        for (int j = 0; j < HS_CPT; j++) {
            float acc = v[j][0];
            const bool ok = !CHECK || col0 + 32 * j < n_cols;
            if (acc > thr.t[0] && ok) push_cand_hs(cands, count, cap, col0 + 32 * j, zi, 1, acc);
#pragma unroll
            for (int st = 1; st < NST; st++) {
                const int H = 1 << st;
#pragma unroll
                for (int i = H >> 1; i < H; i++) acc += v[j][i];
                if (acc > thr.t[st] && ok) push_cand_hs(cands, count, cap, col0 + 32 * j, zi, H, acc);
            }
        }
    }
}

template <int NST, int HS_CPT, int MINB>
__global__ void __launch_bounds__(256, MINB)
k_harmsum(const float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ count,
          uint32_t cap, HarmThr thr, int n_cols, int n_z, int bin0)
{
    constexpr int HS_COLS = 32 * HS_CPT;
    const bool edge = blockIdx.x == 0 || blockIdx.x * HS_COLS + HS_COLS > n_cols;     // CTA-uniform
    if (edge) harmsum_tile<NST, HS_CPT, true>(plane, cands, count, cap, thr, n_cols, n_z, bin0);
    else harmsum_tile<NST, HS_CPT, false>(plane, cands, count, cap, thr, n_cols, n_z, bin0);
}

// Threshold + compaction over one plane (row a8). grid-stride over float4 groups of a row.
// grid = (ceil(n_cols/1024), n_z), block 256.
__global__ void __launch_bounds__(256)
k_candidates(const float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ count,
             uint32_t cap, float thr, int n_cols)
{
    const int zi = blockIdx.y;
    const float* row = plane + (size_t)zi * n_cols;
    const int c4 = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (c4 >= n_cols) return;
    if (c4 + 3 < n_cols && ((((size_t)zi * n_cols) & 3) == 0)) {
        float4 v = __ldg(reinterpret_cast<const float4*>(row + c4));
        if (v.x > thr) push_cand(cands, count, cap, c4, zi, 1, v.x);
        if (v.y > thr) push_cand(cands, count, cap, c4 + 1, zi, 1, v.y);
        if (v.z > thr) push_cand(cands, count, cap, c4 + 2, zi, 1, v.z);
        if (v.w > thr) push_cand(cands, count, cap, c4 + 3, zi, 1, v.w);
    } else {
        for (int c = c4; c < min(c4 + 4, n_cols); c++) {
            float v = __ldg(row + c);
            if (v > thr) push_cand(cands, count, cap, c, zi, 1, v);
        }
    }
}

int fdas_launch_harmsum(fdas_plan* p, const float* d_plane, int max_harm, const float* h_thr,
                        fdas_cand* d_cands, uint32_t* d_count, uint32_t cap, cudaStream_t st)
{
    int n_stage = 0;
    for (int H = 1; H <= max_harm; H <<= 1) n_stage++;
    HarmThr thr;
    for (int i = 0; i < 5; i++) thr.t[i] = i < n_stage ? h_thr[i] : 3.0e38f;
    FDAS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));
    int n_cols = (int)p->n_cols;
    static const int variant = getenv("FDAS_HS_VARIANT") ? atoi(getenv("FDAS_HS_VARIANT")) : 0;
    dim3 block(32, HS_ROWS_PER_PASS);
#define FDAS_HS_ARGS d_plane, d_cands, d_count, cap, thr, n_cols, p->n_z, p->bin0
#define FDAS_HS_GRID(CPT) dim3((n_cols + 32 * CPT - 1) / (32 * CPT))
    switch (n_stage) {
    case 1: k_harmsum<1, 4, 2><<<FDAS_HS_GRID(4), block, 0, st>>>(FDAS_HS_ARGS); break;
    case 2: k_harmsum<2, 4, 2><<<FDAS_HS_GRID(4), block, 0, st>>>(FDAS_HS_ARGS); break;
    case 3: k_harmsum<3, 4, 2><<<FDAS_HS_GRID(4), block, 0, st>>>(FDAS_HS_ARGS); break;
    case 4: k_harmsum<4, 2, 2><<<FDAS_HS_GRID(2), block, 0, st>>>(FDAS_HS_ARGS); break;
    default:
        if (variant == 1) k_harmsum<5, 4, 2><<<FDAS_HS_GRID(4), block, 0, st>>>(FDAS_HS_ARGS);
        else k_harmsum<5, 2, 4><<<FDAS_HS_GRID(2), block, 0, st>>>(FDAS_HS_ARGS);     // measured best on B200
        break;
    }
#undef FDAS_HS_GRID
#undef FDAS_HS_ARGS
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}

int fdas_launch_candidates(fdas_plan* p, const float* d_plane, float thr, fdas_cand* d_cands,
                           uint32_t* d_count, uint32_t cap, cudaStream_t st)
{
    FDAS_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint32_t), st));
    int n_cols = (int)p->n_cols;
    k_candidates<<<dim3((n_cols + 1023) / 1024, p->n_z), 256, 0, st>>>(d_plane, d_cands, d_count, cap, thr, n_cols);
    FDAS_LAUNCH_CHECK();
    return FDAS_OK;
}
