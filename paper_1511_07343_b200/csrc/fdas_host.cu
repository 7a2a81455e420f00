// fdas_host.cu -- host-buffer convenience path (fdas_search_host), thresholds, teardown,
// error text.  Part of the extern "C" boundary declared in include/fdas.h.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include "fdas_common.cuh"

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// Scratch of fdas_search_host (all owned by the plan, built lazily): a device arena with TWO
// series buffers (so the copy of chunk c+1 overlaps the kernels of chunk c: PAPER.md:49 step 1,
// "asynchronous copy of the time series"), one spectrum, the FFT workspace, one plane
// (harmonic-sum mode), candidate lists for the whole batch; two copy streams and a few events.
struct Arena {
    float* series[2]; float* spec; void* ws; float* plane; fdas_cand* cands; uint32_t* counts;
};

static int arena_prepare(fdas_plan* p, int n_batch, int cb, bool need_plane, uint32_t cap, Arena* a)
{
    const size_t series_b = align_up((size_t)cb * p->n_samples * sizeof(float), 256);
    size_t o_series = 0;
    size_t o_spec = o_series + 2 * series_b;
    size_t o_ws = o_spec + align_up((size_t)cb * p->n_bins * sizeof(float2), 256);
    size_t o_plane = o_ws + align_up(p->workspace_bytes, 256);
    size_t o_cands = o_plane + (need_plane ? align_up((size_t)p->n_z * p->n_cols * sizeof(float), 256) : 0);
    size_t o_counts = o_cands + align_up((size_t)n_batch * cap * sizeof(fdas_cand), 256);
    size_t total = o_counts + align_up((size_t)n_batch * sizeof(uint32_t), 256);
    if (total > p->arena_bytes) {
        if (p->arena) cudaFree(p->arena);
        p->arena = nullptr; p->arena_bytes = 0;
        if (cudaMalloc(&p->arena, total) != cudaSuccess) { cudaGetLastError(); return FDAS_E_NOMEM; }
        p->arena_bytes = total;
    }
    if ((size_t)n_batch > p->pinned_counts_n) {
        if (p->pinned_counts) cudaFreeHost(p->pinned_counts);
        p->pinned_counts = nullptr; p->pinned_counts_n = 0;
        if (cudaMallocHost(&p->pinned_counts, (size_t)n_batch * sizeof(uint32_t)) != cudaSuccess) { cudaGetLastError(); return FDAS_E_NOMEM; }
        p->pinned_counts_n = (size_t)n_batch;
    }
    if (!p->pipe_ready) {
        FDAS_CUDA(cudaStreamCreateWithFlags(&p->st_h2d, cudaStreamNonBlocking));
        FDAS_CUDA(cudaStreamCreateWithFlags(&p->st_d2h, cudaStreamNonBlocking));
        for (int i = 0; i < 2; i++) {
            FDAS_CUDA(cudaEventCreateWithFlags(&p->ev_in[i], cudaEventDisableTiming));
            FDAS_CUDA(cudaEventCreateWithFlags(&p->ev_free[i], cudaEventDisableTiming));
            FDAS_CUDA(cudaEventCreateWithFlags(&p->ev_done[i], cudaEventDisableTiming));
        }
        p->pipe_ready = 1;
    }
    char* b = reinterpret_cast<char*>(p->arena);
    a->series[0] = reinterpret_cast<float*>(b + o_series);
    a->series[1] = reinterpret_cast<float*>(b + o_series + series_b);
    a->spec = reinterpret_cast<float*>(b + o_spec);
    a->ws = b + o_ws;
    a->plane = need_plane ? reinterpret_cast<float*>(b + o_plane) : nullptr;
    a->cands = reinterpret_cast<fdas_cand*>(b + o_cands);
    a->counts = reinterpret_cast<uint32_t*>(b + o_counts);
    return FDAS_OK;
}

// Copy the candidate lists of series [b0, b0 + nb) back: their counts are already in pinned host memory.
static int fetch_cands(fdas_plan* p, const Arena& a, int b0, int nb, uint32_t capacity, fdas_cand* h_cands,
                       uint32_t* h_counts)
{
    for (int b = b0; b < b0 + nb; b++) {
        h_counts[b] = p->pinned_counts[b];
        uint32_t n = h_counts[b] < capacity ? h_counts[b] : capacity;
        if (n)
            FDAS_CUDA(cudaMemcpyAsync(h_cands + (size_t)b * capacity, a.cands + (size_t)b * capacity,
                                      (size_t)n * sizeof(fdas_cand), cudaMemcpyDeviceToHost, p->st_d2h));
    }
    return FDAS_OK;
}

extern "C" int fdas_search_host(fdas_plan* p, const float* h_series, int32_t n_batch, int32_t max_harm,
                                const float* h_thresholds, fdas_cand* h_cands, uint32_t* h_counts,
                                uint32_t capacity, void* stream)
{
    if (!p || !h_series || !h_thresholds || !h_cands || !h_counts || n_batch < 1 || capacity < 1) return FDAS_E_INVALID;
    if (!(max_harm == 0 || max_harm == 1 || max_harm == 2 || max_harm == 4 || max_harm == 8 || max_harm == 16)) return FDAS_E_INVALID;
    if (max_harm > 0 && p->interbin) return FDAS_E_INVALID;
    if (!p->built) return FDAS_E_STATE;
    cudaStream_t st = (cudaStream_t)stream;
    const bool fused = (max_harm == 0);
    const int cb = fused ? (n_batch < p->max_batch ? n_batch : p->max_batch) : 1;      // series per chunk
    const int n_chunk = (n_batch + cb - 1) / cb;
    Arena a;
    int rc = arena_prepare(p, n_batch, cb, !fused, capacity, &a);
    if (rc) return rc;
    auto chunk_nb = [&](int c) { int b0 = c * cb; return n_batch - b0 < cb ? n_batch - b0 : cb; };
    auto enqueue_h2d = [&](int c) -> int {       // on the copy stream, after the buffer's previous reader
        if (c >= 2) FDAS_CUDA(cudaStreamWaitEvent(p->st_h2d, p->ev_free[c & 1], 0));
        FDAS_CUDA(cudaMemcpyAsync(a.series[c & 1], h_series + (size_t)c * cb * p->n_samples,
                                  (size_t)chunk_nb(c) * p->n_samples * sizeof(float), cudaMemcpyHostToDevice, p->st_h2d));
        FDAS_CUDA(cudaEventRecord(p->ev_in[c & 1], p->st_h2d));
        return FDAS_OK;
    };
    // the arena may still be in use by work the caller enqueued on `st` before this call
    FDAS_CUDA(cudaEventRecord(p->ev_done[0], st));
    FDAS_CUDA(cudaStreamWaitEvent(p->st_h2d, p->ev_done[0], 0));
    rc = enqueue_h2d(0);
    if (rc) return rc;
    for (int c = 0; c < n_chunk; c++) {
        const int b0 = c * cb, nb = chunk_nb(c);
        if (c + 1 < n_chunk) { rc = enqueue_h2d(c + 1); if (rc) return rc; }
        FDAS_CUDA(cudaStreamWaitEvent(st, p->ev_in[c & 1], 0));
        rc = fdas_run_spectrum(p, a.series[c & 1], nb, reinterpret_cast<float2*>(a.spec), nullptr, a.ws, st);
        if (rc) return rc;
        FDAS_CUDA(cudaEventRecord(p->ev_free[c & 1], st));
        if (fused) {
            rc = fdas_launch_correlate(p, reinterpret_cast<const float2*>(a.spec), nb, nullptr, h_thresholds[0],
                                       a.cands + (size_t)b0 * capacity, a.counts + b0, capacity, st);
            if (rc) return rc;
        } else {
            rc = fdas_launch_correlate(p, reinterpret_cast<const float2*>(a.spec), 1, a.plane, 0.f, nullptr, nullptr, 0, st);
            if (rc) return rc;
            rc = fdas_launch_harmsum(p, a.plane, max_harm, h_thresholds, a.cands + (size_t)b0 * capacity,
                                     a.counts + b0, capacity, st);
            if (rc) return rc;
        }
        FDAS_CUDA(cudaMemcpyAsync(p->pinned_counts + b0, a.counts + b0, (size_t)nb * sizeof(uint32_t),
                                  cudaMemcpyDeviceToHost, st));
        FDAS_CUDA(cudaEventRecord(p->ev_done[c & 1], st));
        if (c >= 1) {                             // one chunk behind: its lists come back while chunk c computes
            FDAS_CUDA(cudaEventSynchronize(p->ev_done[(c - 1) & 1]));
            rc = fetch_cands(p, a, (c - 1) * cb, chunk_nb(c - 1), capacity, h_cands, h_counts);
            if (rc) return rc;
        }
    }
    FDAS_CUDA(cudaEventSynchronize(p->ev_done[(n_chunk - 1) & 1]));
    rc = fetch_cands(p, a, (n_chunk - 1) * cb, chunk_nb(n_chunk - 1), capacity, h_cands, h_counts);
    if (rc) return rc;
    FDAS_CUDA(cudaStreamSynchronize(p->st_d2h));
    FDAS_CUDA(cudaStreamSynchronize(st));
    return FDAS_OK;
}

// Q(H, T) = exp(-T) sum_{j<H} T^j / j!  evaluated in log space for robustness.
static double surv(int H, double T)
{
    double term = 1.0, sum = 1.0;
    for (int j = 1; j < H; j++) { term *= T / (double)j; sum += term; }
    return exp(-T + log(sum));
}

extern "C" double fdas_threshold(int32_t n_harm, double pfa)
{
    if (n_harm < 1 || !(pfa > 0.0) || !(pfa < 1.0)) return NAN;
    double lo = 0.0, hi = 8.0;
    while (surv(n_harm, hi) > pfa) hi *= 2.0;
    for (int i = 0; i < 100; i++) {
        double mid = 0.5 * (lo + hi);
        if (surv(n_harm, mid) > pfa) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

extern "C" int fdas_plan_destroy(fdas_plan* p)
{
    if (!p) return FDAS_E_INVALID;
    if (p->d_taps) cudaFree(p->d_taps);
    if (p->d_W) cudaFree(p->d_W);
    if (p->d_Wr) cudaFree(p->d_Wr);
    if (p->d_status) cudaFree(p->d_status);
    if (p->d_segtw) cudaFree(p->d_segtw);
    if (p->arena) cudaFree(p->arena);
    if (p->pinned_counts) cudaFreeHost(p->pinned_counts);
    if (p->pipe_ready) {
        cudaStreamDestroy(p->st_h2d);
        cudaStreamDestroy(p->st_d2h);
        for (int i = 0; i < 2; i++) { cudaEventDestroy(p->ev_in[i]); cudaEventDestroy(p->ev_free[i]); cudaEventDestroy(p->ev_done[i]); }
    }
    delete p;
    return FDAS_OK;
}

extern char* fdas_cuda_error_text();

extern "C" const char* fdas_strerror(int code)
{
    switch (code) {
    case FDAS_OK: return "ok";
    case FDAS_E_INVALID: return "invalid argument";
    case FDAS_E_STATE: return "wrong plan state (templates not built, or option set after build)";
    case FDAS_E_WORKSPACE: return "workspace missing or not 256-byte aligned";
    case FDAS_E_CUDA: return fdas_cuda_error_text();
    case FDAS_E_NOMEM: return "allocation failed";
    default: return "unknown error code";
    }
}
