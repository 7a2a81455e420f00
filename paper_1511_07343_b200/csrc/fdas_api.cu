// fdas_api.cu -- the extern "C" boundary of libfdas.so (include/fdas.h): plan object,
// argument validation, error text, and the host-buffer convenience path.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include "fdas_common.cuh"

static thread_local char g_cuda_err[512] = "no CUDA error recorded";

void fdas_set_cuda_error(cudaError_t e, const char* where)
{
    snprintf(g_cuda_err, sizeof(g_cuda_err), "CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), where);
}

char* fdas_cuda_error_text() { return g_cuda_err; }

// Vector accesses in the kernels need these alignments (a misaligned device pointer would fault on the GPU).
static bool misaligned(const void* ptr, uintptr_t a) { return ((uintptr_t)ptr & (a - 1)) != 0; }

static bool is_pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

static void derive_sizes(fdas_plan* p)
{
    p->nset = 1 + p->interbin;
    p->n_t = p->n_z * p->nset;
    p->n_cols = p->n_bins * p->nset;
    int lg = 0;
    while ((1LL << lg) < p->M) lg++;
    p->R1 = 1 << ((lg + 1) / 2);
    p->R2 = 1 << (lg / 2);
    int c1 = 8192 / p->R1; if (c1 < 1) c1 = 1; if (c1 > p->R2) c1 = p->R2;
    int c2 = 4096 / p->R2; if (c2 < 1) c2 = 1; if (c2 > p->R1 / 2) c2 = p->R1 / 2; if (c2 < 1) c2 = 1;
    p->C1 = c1; p->C2 = c2;
    p->n_part = p->R2 / p->C1;
    fdas_spectrum_tma_plan(p);
    // partial sums: the generic kernels use n_part per series, the TMA-staged passes M/4096 and one scale per series
    size_t parts = (size_t)p->n_part;
    if (p->sp_npass && (size_t)(p->M / 4096) > parts) parts = (size_t)(p->M / 4096);
    p->ws_inter_bytes = align_up((size_t)p->max_batch * p->M * sizeof(float2), 256);
    p->ws_part_bytes = align_up((size_t)p->max_batch * (parts * 3 * sizeof(double) + sizeof(float)), 256);
    p->workspace_bytes = p->ws_inter_bytes + p->ws_part_bytes;
}

extern "C" int fdas_set_device(int32_t device)
{
    FDAS_CUDA(cudaSetDevice(device));
    return FDAS_OK;
}

extern "C" int fdas_plan_create(fdas_plan** out, int64_t n_samples, double z_max, double dz,
                                int32_t template_width, int32_t segment_len)
{
    if (!out) return FDAS_E_INVALID;
    *out = nullptr;
    const int L = segment_len, m = template_width;
    if (!(L == 256 || L == 512 || L == 1024 || L == 2048 || L == 4096)) return FDAS_E_INVALID;
    if (!is_pow2(n_samples) || n_samples < 2LL * L || n_samples > (1LL << 25)) return FDAS_E_INVALID;
    if (m < 2 || (m & 1) || m > L / 2) return FDAS_E_INVALID;
    if (!(dz > 0.0) || !(z_max >= 0.0) || !isfinite(dz) || !isfinite(z_max)) return FDAS_E_INVALID;
    double q = z_max / dz;
    if (fabs(q - nearbyint(q)) > 1e-9 * fmax(1.0, q)) return FDAS_E_INVALID;
    int64_t n_z = 2 * (int64_t)nearbyint(q) + 1;
    if (n_z > 32767) return FDAS_E_INVALID;
    fdas_plan* p = new (std::nothrow) fdas_plan;
    if (!p) return FDAS_E_NOMEM;
    memset(p, 0, sizeof(*p));
    p->n_samples = n_samples;
    p->n_bins = n_samples / 2;
    p->M = (int32_t)(n_samples / 2);
    p->bin0 = 1;
    p->n_z = (int32_t)n_z;
    p->m = m;
    p->L = L;
    p->step = L - m;
    p->n_seg = (int32_t)((p->n_bins + p->step - 1) / p->step);
    p->interbin = 0;
    p->z_max = z_max;
    p->dz = dz;
    p->max_batch = 1;
    p->quad_points = 32768;
    derive_sizes(p);
    *out = p;
    return FDAS_OK;
}

extern "C" int fdas_plan_set_option(fdas_plan* p, int32_t key, int64_t value)
{
    if (!p) return FDAS_E_INVALID;
    switch (key) {                        // tuning keys: any time, results do not depend on them
    case FDAS_OPT_TUNE_SCALAR:     if (value != 0 && value != 1) return FDAS_E_INVALID; p->tune_scalar = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_T_CHUNKS:   if (value < 0 || value > 1024) return FDAS_E_INVALID; p->tune_t_chunks = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_HS_SECTORS: if (value < 0 || value > 64) return FDAS_E_INVALID; p->tune_hs_sectors = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_HS_ROWS:    if (value < 0 || value > 8) return FDAS_E_INVALID; p->tune_hs_rows = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_HS_VARIANT: if (value < 0 || value > 1) return FDAS_E_INVALID; p->tune_hs_variant = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_STAGE_TEMPLATES: if (value < 0 || value > 1) return FDAS_E_INVALID; p->tune_stage_templates = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_SPEC_SELFTEST: if (value < 0 || value > 2 || p->built) return FDAS_E_INVALID; p->tune_spec_selftest = (int32_t)value; return FDAS_OK;
    case FDAS_OPT_TUNE_SPEC_GENERIC: if (value < 0 || value > 1) return FDAS_E_INVALID; p->tune_spec_generic = (int32_t)value; return FDAS_OK;
    default: break;
    }
    if (p->built) return FDAS_E_STATE;
    switch (key) {
    case FDAS_OPT_INTERBIN:
        if (value != 0 && value != 1) return FDAS_E_INVALID;
        p->interbin = (int32_t)value;
        break;
    case FDAS_OPT_MAX_BATCH:
        if (value < 1 || value > 4096) return FDAS_E_INVALID;
        p->max_batch = (int32_t)value;
        break;
    case FDAS_OPT_QUAD_POINTS:
        if (value < 64 || value > (1 << 24)) return FDAS_E_INVALID;
        p->quad_points = (int32_t)value;
        break;
    default:
        return FDAS_E_INVALID;
    }
    derive_sizes(p);
    return FDAS_OK;
}

extern "C" int fdas_plan_info(const fdas_plan* p, fdas_info* o)
{
    if (!p || !o) return FDAS_E_INVALID;
    o->n_samples = p->n_samples; o->n_bins = p->n_bins; o->n_cols = p->n_cols;
    o->bin0 = p->bin0; o->n_z = p->n_z; o->n_templates = p->n_t; o->width = p->m; o->seg_len = p->L;
    o->step = p->step; o->n_seg = p->n_seg; o->interbin = p->interbin;
    o->z_max = p->z_max; o->dz = p->dz; o->workspace_bytes = p->workspace_bytes;
    return FDAS_OK;
}

extern "C" int fdas_build_templates(fdas_plan* p, void* stream)
{
    if (!p) return FDAS_E_INVALID;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->built) return FDAS_OK;                                  // the bank is built once
    if (!p->d_taps && cudaMalloc(&p->d_taps, (size_t)p->n_t * p->m * sizeof(float2)) != cudaSuccess) { p->d_taps = nullptr; cudaGetLastError(); return FDAS_E_NOMEM; }
    if (!p->d_W && cudaMalloc(&p->d_W, (size_t)p->n_t * p->L * sizeof(float2)) != cudaSuccess) { p->d_W = nullptr; cudaGetLastError(); return FDAS_E_NOMEM; }
    if (!p->d_Wr && cudaMalloc(&p->d_Wr, (size_t)p->n_t * p->L * sizeof(float2)) != cudaSuccess) { p->d_Wr = nullptr; cudaGetLastError(); return FDAS_E_NOMEM; }
    if (!p->d_segtw && cudaMalloc(&p->d_segtw, 46 * 128 * sizeof(float2)) != cudaSuccess) { p->d_segtw = nullptr; cudaGetLastError(); return FDAS_E_NOMEM; }
    if (!p->d_status) {
        if (cudaMalloc(&p->d_status, sizeof(uint32_t)) != cudaSuccess) { p->d_status = nullptr; cudaGetLastError(); return FDAS_E_NOMEM; }
        FDAS_CUDA(cudaMemsetAsync(p->d_status, 0, sizeof(uint32_t), st));
    }
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
            cudaGetLastError();
            sms = 148;
        }
        p->n_sms = sms > 0 ? sms : 148;
    }
    int rc = fdas_launch_templates(p, st);
    if (rc) return rc;
    FDAS_CUDA(cudaStreamSynchronize(st));
    if (p->sp_npass && !p->tune_spec_generic && p->tune_spec_selftest != 1) {
        rc = fdas_spectrum_selftest(p, p->tune_spec_selftest, st);
        if (rc) return rc;
    }
    p->built = 1;
    return FDAS_OK;
}

extern "C" int fdas_plan_status(const fdas_plan* p, uint32_t* out)
{
    if (!p || !out) return FDAS_E_INVALID;
    *out = 0;
    if (!p->d_status) return FDAS_OK;
    FDAS_CUDA(cudaMemcpy(out, p->d_status, sizeof(uint32_t), cudaMemcpyDeviceToHost));
    return FDAS_OK;
}

extern "C" int fdas_kernel_occupancy(const char* kernel, int32_t* ctas_per_sm, int32_t* registers, int32_t* smem_bytes)
{
    if (!kernel || !ctas_per_sm || !registers || !smem_bytes) return FDAS_E_INVALID;
    if (!strcmp(kernel, "spec_pass_a")) return fdas_occupancy_spectrum(0, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "spec_pass_b")) return fdas_occupancy_spectrum(1, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "spec_pass_c")) return fdas_occupancy_spectrum(2, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "correlate")) return fdas_occupancy_correlate(0, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "correlate_fused")) return fdas_occupancy_correlate(1, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "correlate_staged")) return fdas_occupancy_correlate(2, ctas_per_sm, registers, smem_bytes);
    if (!strcmp(kernel, "harmsum")) return fdas_occupancy_harmsum(ctas_per_sm, registers, smem_bytes);
    return FDAS_E_INVALID;
}

extern "C" int fdas_get_templates(const fdas_plan* p, float* h_re_im)
{
    if (!p || !h_re_im) return FDAS_E_INVALID;
    if (!p->built) return FDAS_E_STATE;
    FDAS_CUDA(cudaMemcpy(h_re_im, p->d_taps, (size_t)p->n_t * p->m * sizeof(float2), cudaMemcpyDeviceToHost));
    return FDAS_OK;
}

extern "C" int fdas_spectrum(fdas_plan* p, const float* d_series, int32_t n_batch, float* d_spectrum,
                             float* d_meanpow, void* d_workspace, void* stream)
{
    if (!p || !d_series || !d_spectrum || n_batch < 1 || n_batch > p->max_batch) return FDAS_E_INVALID;
    if (misaligned(d_series, 8) || misaligned(d_spectrum, 8) || misaligned(d_meanpow, 4)) return FDAS_E_INVALID;
    if (!d_workspace || ((uintptr_t)d_workspace & 255)) return FDAS_E_WORKSPACE;
    return fdas_run_spectrum(p, d_series, n_batch, reinterpret_cast<float2*>(d_spectrum), d_meanpow, d_workspace,
                             (cudaStream_t)stream);
}

extern "C" int fdas_correlate(fdas_plan* p, const float* d_spectrum, int32_t n_batch, float* d_plane,
                              float threshold, fdas_cand* d_cands, uint32_t* d_counts, uint32_t capacity,
                              void* d_workspace, void* stream)
{
    (void)d_workspace;
    if (!p || !d_spectrum || n_batch < 1 || n_batch > 65535) return FDAS_E_INVALID;      // batch = gridDim.z
    if (!d_plane && !d_cands) return FDAS_E_INVALID;
    if (d_cands && !d_counts) return FDAS_E_INVALID;
    if (misaligned(d_spectrum, 8) || misaligned(d_plane, 16) || misaligned(d_cands, 4) || misaligned(d_counts, 4))
        return FDAS_E_INVALID;
    if (!p->built) return FDAS_E_STATE;
    return fdas_launch_correlate(p, reinterpret_cast<const float2*>(d_spectrum), n_batch, d_plane, threshold,
                                 d_cands, d_counts, capacity, (cudaStream_t)stream);
}

static bool valid_max_harm(int h) { return h == 1 || h == 2 || h == 4 || h == 8 || h == 16; }

extern "C" int fdas_harmsum(fdas_plan* p, const float* d_plane, int32_t max_harm, const float* h_thresholds,
                            fdas_cand* d_cands, uint32_t* d_count, uint32_t capacity, void* stream)
{
    if (!p || !d_plane || !h_thresholds || !d_cands || !d_count) return FDAS_E_INVALID;
    if (!valid_max_harm(max_harm) || p->interbin) return FDAS_E_INVALID;
    if (!p->built) return FDAS_E_STATE;
    if (misaligned(d_plane, 4) || misaligned(d_cands, 4) || misaligned(d_count, 4)) return FDAS_E_INVALID;
    return fdas_launch_harmsum(p, d_plane, max_harm, h_thresholds, d_cands, d_count, capacity, (cudaStream_t)stream);
}

extern "C" int fdas_resample(fdas_plan* p, const float* d_series, double beta, float* d_out, void* stream)
{
    if (!p || !d_series || !d_out || d_series == d_out) return FDAS_E_INVALID;
    if (!(beta > -0.5 && beta < 0.5)) return FDAS_E_INVALID;
    if (misaligned(d_series, 4) || misaligned(d_out, 16)) return FDAS_E_INVALID;
    return fdas_launch_resample(p, d_series, beta, d_out, (cudaStream_t)stream);
}

extern "C" int fdas_candidates(fdas_plan* p, const float* d_plane, float threshold, fdas_cand* d_cands,
                               uint32_t* d_count, uint32_t capacity, void* stream)
{
    if (!p || !d_plane || !d_cands || !d_count) return FDAS_E_INVALID;
    if (misaligned(d_plane, 4) || misaligned(d_cands, 4) || misaligned(d_count, 4)) return FDAS_E_INVALID;
    return fdas_launch_candidates(p, d_plane, threshold, d_cands, d_count, capacity, (cudaStream_t)stream);
}
