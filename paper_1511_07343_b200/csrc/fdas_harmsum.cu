// fdas_harmsum.cu -- incoherent harmonic summing and candidate compaction
// (BASELINE.json configs[4]; "pulse harmonics").
#include "fdas_common.cuh"

struct HarmThr { float t[5]; };

// One thread per top-harmonic cell (col, zi).  S_1 = P; stage 2H adds the odd-h terms of
// fraction h/(2H) (the rounding rule is invariant under (h,H)->(2h,2H), so S_2H = S_H + odd terms).
//   k_h = floor((k h + H/2)/H), zeta_h = sgn(zeta) floor((|zeta| h + H/2)/H)   (include/fdas.h)
// grid = (ceil(n_cols/256), n_z), block 256.
__global__ void __launch_bounds__(256)
k_harmsum(const float* __restrict__ plane, fdas_cand* __restrict__ cands, uint32_t* __restrict__ count,
          uint32_t cap, HarmThr thr, int n_cols, int n_z, int bin0, int n_stage)
{
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    const int zi = blockIdx.y;
    if (col >= n_cols) return;
    const int zc = (n_z - 1) / 2;
    const int zeta = zi - zc, az = abs(zeta), sg = zeta < 0 ? -1 : 1;
    const int k = bin0 + col;
    float acc = __ldg(plane + (size_t)zi * n_cols + col);
    if (acc > thr.t[0]) push_cand(cands, count, cap, col, zi, 1, acc);
    int H = 2;
    for (int st = 1; st < n_stage; st++, H <<= 1) {
        const int sh = st;                       // H = 1 << st
        for (int h = 1; h < H; h += 2) {
            int kh = (int)(((long long)k * h + (H >> 1)) >> sh);
            int zh = sg * ((az * h + (H >> 1)) >> sh);
            if (kh >= bin0) acc += __ldg(plane + (size_t)(zc + zh) * n_cols + (kh - bin0));
        }
        if (acc > thr.t[st]) push_cand(cands, count, cap, col, zi, H, acc);
    }
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
    k_harmsum<<<dim3((n_cols + 255) / 256, p->n_z), 256, 0, st>>>(d_plane, d_cands, d_count, cap, thr,
                                                                 n_cols, p->n_z, p->bin0, n_stage);
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
