// Self-test of the emulator's model of the asynchronous copies (emu_tma.h): small kernels, written straight
// against the emulator API, that use the copies correctly and INCORRECTLY.  The tests in
// tests/test_emulated_kernels.py prove nothing about the product's TMA code unless the misuses below are
// caught (tests/test_emulated_kernels.py::test_the_emulator_models_the_asynchronous_copies).
#include "emu_tma.h"

// mode 0: correct use (box load, in-place change, box store): returns 0 if the output is right
// mode 1: the destination is read BEFORE the mbarrier wait: returns 1 if the reader saw NaN poison
// mode 2: fewer bytes announced than copied: the wait can never be satisfied -> the emulator aborts (deadlock)
// mode 3: a store that is never committed / waited for -> abort at CTA exit
// mode 4: a box destination that is not 128-byte aligned -> abort
// mode 5: the store's source buffer is overwritten before tma_store_wait_read: returns 1 if the output is corrupted
extern "C" int emu_selftest_tma(int mode)
{
    const int R = 4, C = 8;                                        // tensor [2][R][C] of 8-byte elements, box (C, R, 1)
    double* g = nullptr; double* o = nullptr;
    cudaMalloc(&g, 2 * R * C * sizeof(double));
    cudaMalloc(&o, 2 * R * C * sizeof(double));
    for (int i = 0; i < 2 * R * C; i++) { g[i] = i; o[i] = -1.0; }
    CUtensorMap mi, mo;
    const uint64_t dims[3] = {C, R, 2}, str[2] = {C * 8, R * C * 8};
    const uint32_t box[3] = {C, R, 1};
    if (!fdas_encode_tensor_map(&mi, g, 3, dims, str, box) || !fdas_encode_tensor_map(&mo, o, 3, dims, str, box)) return -1;
    int saw_nan = 0;
    emu_launch(dim3(2), dim3(32), 1024, "selftest_tma", [&] {
        double* sm = (double*)emu_dyn_smem();
        static thread_local uint64_t bar;
        const int tid = threadIdx.x, b = blockIdx.x;
        if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
        __syncthreads();
        if (tid == 0) {
            mbar_expect_tx(&bar, mode == 2 ? R * C * 8 - 16 : R * C * 8);
            tma_load_3d(mode == 4 ? (void*)(sm + 2) : (void*)sm, &mi, 0, 0, b, &bar);
        }
        if (mode == 1 && tid == 1 && sm[5] != sm[5]) saw_nan = 1;   // (tid 0 has issued the copy: forward order)
        if (!mbar_wait(&bar, 0, nullptr)) return;
        sm[tid] += 100.0;
        fence_proxy_async();
        __syncthreads();
        if (tid == 0) {
            tma_store_3d(&mo, sm, 0, 0, b);
            if (mode != 3) tma_store_commit();
            if (mode == 5) sm[3] = -7.0;                            // too early: the store has not read the buffer yet
            if (mode != 3) tma_store_wait_all();
        }
    });
    int bad = 0;
    for (int i = 0; i < 2 * R * C; i++) bad += o[i] != g[i] + 100.0;
    cudaFree(g); cudaFree(o);
    if (mode == 1) return saw_nan;
    if (mode == 5) return bad != 0;
    return bad;
}
