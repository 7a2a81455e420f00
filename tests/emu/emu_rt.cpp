// Host emulation runtime: guard-paged "device" memory + coroutine CTA scheduler (test infrastructure, tests/emu/README.md).
#include "cuda_runtime.h"
#include <signal.h>
#include <sys/mman.h>
#include <ucontext.h>
#include <unistd.h>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>
#include <vector>

thread_local uint3 threadIdx, blockIdx;
thread_local dim3 blockDim, gridDim;

// ------------------------------------------------------------------ memory
struct Alloc { char* map; size_t map_len; char* user; size_t n; };
static std::map<uintptr_t, Alloc> g_allocs;      // keyed by user pointer
static std::mutex g_mu;
static const size_t PG = 4096;
static bool align_end() { const char* e = getenv("EMU_ALIGN"); return !(e && !strcmp(e, "start")); }

static void* guarded_alloc(size_t n, bool poison = true)
{
    size_t body = (n + PG - 1) / PG * PG;
    if (body == 0) body = PG;
    size_t len = body + 2 * PG;
    char* m = (char*)mmap(nullptr, len, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
    if (m == MAP_FAILED) return nullptr;
    mprotect(m, PG, PROT_NONE);
    mprotect(m + PG + body, PG, PROT_NONE);
    char* user = m + PG;
    if (align_end()) user = m + PG + body - ((n + 15) / 16 * 16);
    if (poison) memset(m + PG, 0xFF, body);                  // poison: an uninitialised float reads as NaN and shows up in parity
    std::lock_guard<std::mutex> lk(g_mu);
    g_allocs[(uintptr_t)user] = Alloc{m, len, user, n};
    return user;
}
static void guarded_free(void* p)
{
    std::lock_guard<std::mutex> lk(g_mu);
    auto it = g_allocs.find((uintptr_t)p);
    if (it == g_allocs.end()) { fprintf(stderr, "EMU: free of unknown pointer %p\n", p); abort(); }
    munmap(it->second.map, it->second.map_len);
    g_allocs.erase(it);
}
cudaError_t cudaMalloc(void** p, size_t n) { *p = guarded_alloc(n); return *p ? cudaSuccess : cudaErrorMemoryAllocation; }
cudaError_t cudaFree(void* p) { if (p) guarded_free(p); return cudaSuccess; }
cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind) { memcpy(d, s, n); return cudaSuccess; }
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t) { memcpy(d, s, n); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t) { memset(d, v, n); return cudaSuccess; }
extern "C" void* emu_malloc(size_t n) { return guarded_alloc(n); }
extern "C" void emu_free(void* p) { guarded_free(p); }

static thread_local const char* t_kernel = "(host)";
static void describe(const void* p)
{
    std::lock_guard<std::mutex> lk(g_mu);
    uintptr_t a = (uintptr_t)p;
    for (auto& kv : g_allocs) {
        const Alloc& al = kv.second;
        if (a >= (uintptr_t)al.map && a < (uintptr_t)al.map + al.map_len)
            fprintf(stderr, "     address is %+lld bytes from the start of a %zu-byte allocation (end %+lld)\n",
                    (long long)(a - (uintptr_t)al.user), al.n, (long long)(a - (uintptr_t)al.user - al.n));
    }
}
void emu_check_ptr(const void* p, size_t n, const char* what)
{
    if ((uintptr_t)p % n) {
        fprintf(stderr, "EMU: misaligned %s of %zu bytes at %p in %s block (%u,%u,%u) thread (%u,%u)\n", what, n, p,
                t_kernel, blockIdx.x, blockIdx.y, blockIdx.z, threadIdx.x, threadIdx.y);
        abort();
    }
}
static void on_segv(int, siginfo_t* si, void*)
{
    fprintf(stderr, "EMU: illegal access at %p in %s block (%u,%u,%u) thread (%u,%u,%u)\n", si->si_addr, t_kernel,
            blockIdx.x, blockIdx.y, blockIdx.z, threadIdx.x, threadIdx.y, threadIdx.z);
    describe(si->si_addr);
    _exit(99);
}
__attribute__((constructor)) static void install()
{
    static char altstack[1 << 16];
    stack_t ss; ss.ss_sp = altstack; ss.ss_size = sizeof(altstack); ss.ss_flags = 0;
    sigaltstack(&ss, nullptr);
    struct sigaction sa; memset(&sa, 0, sizeof(sa));
    sa.sa_sigaction = on_segv; sa.sa_flags = SA_SIGINFO | SA_ONSTACK;
    sigaction(SIGSEGV, &sa, nullptr);
    sigaction(SIGBUS, &sa, nullptr);
}

// ------------------------------------------------------------------ CTA scheduler
enum { ST_RUN = 0, ST_BLOCK_BAR = 1, ST_WARP_BAR = 2, ST_DONE = 3 };
#if defined(__x86_64__)
// Minimal user-level context switch (callee-saved registers + stack pointer): swapcontext makes a
// signal-mask system call per switch, which dominates the run time of barrier-heavy kernels.
extern "C" void emu_switch(void** save_sp, void* load_sp);
asm(".text\n.globl emu_switch\n.type emu_switch,@function\nemu_switch:\n"
    "  pushq %rbp\n  pushq %rbx\n  pushq %r12\n  pushq %r13\n  pushq %r14\n  pushq %r15\n"
    "  movq %rsp, (%rdi)\n  movq %rsi, %rsp\n"
    "  popq %r15\n  popq %r14\n  popq %r13\n  popq %r12\n  popq %rbx\n  popq %rbp\n  ret\n"
    ".size emu_switch, .-emu_switch\n");
struct Ctx { void* sp; };
static void ctx_switch(Ctx* from, Ctx* to) { emu_switch(&from->sp, to->sp); }
static void ctx_make(Ctx* c, char* stack, size_t size, void (*fn)(), Ctx*)
{
    uintptr_t top = ((uintptr_t)stack + size) & ~(uintptr_t)15;
    void** sp = (void**)(top - 16);              // return address slot, 16-byte aligned: fn enters with rsp % 16 == 8
    *sp = (void*)fn;
    for (int i = 0; i < 6; i++) *--sp = nullptr; // rbp rbx r12 r13 r14 r15
    c->sp = sp;
}
#else
struct Ctx { ucontext_t uc; };
static void ctx_switch(Ctx* from, Ctx* to) { swapcontext(&from->uc, &to->uc); }
static void ctx_make(Ctx* c, char* stack, size_t size, void (*fn)(), Ctx* link)
{
    getcontext(&c->uc);
    c->uc.uc_stack.ss_sp = stack;
    c->uc.uc_stack.ss_size = size;
    c->uc.uc_link = &link->uc;
    makecontext(&c->uc, fn, 0);
}
#endif
struct Fiber { Ctx ctx; char* stack; int state; uint3 tid; unsigned n_ballot; };
struct Worker {
    std::vector<Fiber> fibers;
    std::vector<unsigned> ballot;            // [warp][2]: alternating accumulators of __ballot_sync
    std::vector<unsigned> shfl;              // [thread]: the value each lane offers to __shfl_sync
    Ctx sched;
    int cur;
    const std::function<void()>* body;
    void* dyn_smem;
};
static thread_local Worker* t_w = nullptr;
static const size_t STACK = 256 << 10;

static void tramp()
{
    Worker* w = t_w;
    (*w->body)();
    w = t_w;
    w->fibers[w->cur].state = ST_DONE;
    ctx_switch(&w->fibers[w->cur].ctx, &w->sched);
    abort();                                     // a finished fibre is never resumed
}
static void yield_with(int st)
{
    Worker* w = t_w;
    w->fibers[w->cur].state = st;
    ctx_switch(&w->fibers[w->cur].ctx, &w->sched);
}
void emu_syncthreads() { yield_with(ST_BLOCK_BAR); }
void emu_syncwarp() { yield_with(ST_WARP_BAR); }
void* emu_dyn_smem() { return t_w->dyn_smem; }

// __ballot_sync over the full warp: OR this lane's bit into the warp's accumulator, meet at a warp barrier,
// read; the other accumulator is cleared for the next ballot between the two barriers (nobody uses it then).
unsigned emu_ballot(int pred)
{
    Worker* w = t_w;
    const int i = w->cur, warp = i / 32, lane = i % 32;
    const unsigned cur = w->fibers[i].n_ballot++ & 1u;
    if (pred) w->ballot[2 * warp + cur] |= 1u << lane;
    yield_with(ST_WARP_BAR);
    w = t_w;
    const unsigned r = w->ballot[2 * warp + cur];
    w->ballot[2 * warp + (cur ^ 1u)] = 0;
    yield_with(ST_WARP_BAR);
    return r;
}

// __shfl_sync over the full warp: every lane publishes its value, warp barrier, read the source lane's,
// warp barrier (so that nobody overwrites a slot that is still being read).
unsigned emu_shfl(unsigned v, int src_lane)
{
    Worker* w = t_w;
    const int i = w->cur, warp = i / 32;
    w->shfl[i] = v;
    yield_with(ST_WARP_BAR);
    w = t_w;
    const unsigned r = w->shfl[32 * warp + (src_lane & 31)];
    yield_with(ST_WARP_BAR);
    return r;
}

int emu_env_int(const char* name, int dflt)
{
    const char* e = getenv(name);
    const int v = e ? atoi(e) : dflt;
    return v > 0 ? v : dflt;
}

static void run_block(Worker* w, dim3 block, int order)      // order: 0 forward, 1 reversed, >= 2 pseudo-random (seed)
{
    const bool rev = order == 1;
    uint64_t rng = 0x9E3779B97F4A7C15ull * (uint64_t)(order + 1) + blockIdx.x * 0x632BE59BD9B4E019ull + blockIdx.y * 977 + blockIdx.z;
    std::vector<int> perm;
    const int nt = block.x * block.y * block.z;
    if ((int)w->fibers.size() < nt) {
        size_t old = w->fibers.size();
        w->fibers.resize(nt);
        for (size_t i = old; i < (size_t)nt; i++) w->fibers[i].stack = (char*)guarded_alloc(STACK, false);
    }
    for (int i = 0; i < nt; i++) {
        Fiber& f = w->fibers[i];
        ctx_make(&f.ctx, f.stack, STACK, tramp, &w->sched);
        f.state = ST_RUN;
        f.n_ballot = 0;
        f.tid = uint3{(unsigned)i % block.x, ((unsigned)i / block.x) % block.y, (unsigned)i / (block.x * block.y)};
    }
    w->ballot.assign(2 * ((nt + 31) / 32), 0u);
    w->shfl.assign(32 * ((nt + 31) / 32), 0u);
    int done = 0;
    while (done < nt) {
        bool progress = false;
        if (order >= 2) {                        // a fresh random order of the threads for every scheduling round
            perm.resize(nt);
            for (int q = 0; q < nt; q++) perm[q] = q;
            for (int q = nt - 1; q > 0; q--) {
                rng ^= rng << 13; rng ^= rng >> 7; rng ^= rng << 17;
                std::swap(perm[q], perm[(int)(rng % (uint64_t)(q + 1))]);
            }
        }
        for (int q = 0; q < nt; q++) {
            int i = order >= 2 ? perm[q] : (rev ? nt - 1 - q : q);
            Fiber& f = w->fibers[i];
            if (f.state != ST_RUN) continue;
            w->cur = i;
            threadIdx = f.tid;
            ctx_switch(&w->sched, &f.ctx);
            progress = true;
            if (f.state == ST_DONE) done++;
        }
        // release warp barriers
        for (int w0 = 0; w0 < nt; w0 += 32) {
            int at = 0, live = 0;
            for (int i = w0; i < w0 + 32 && i < nt; i++) {
                if (w->fibers[i].state != ST_DONE) live++;
                if (w->fibers[i].state == ST_WARP_BAR) at++;
            }
            if (live && at == live) {
                for (int i = w0; i < w0 + 32 && i < nt; i++)
                    if (w->fibers[i].state == ST_WARP_BAR) w->fibers[i].state = ST_RUN;
                progress = true;
            }
        }
        int at = 0;
        for (int i = 0; i < nt; i++) at += w->fibers[i].state == ST_BLOCK_BAR;
        if (at && at == nt - done) {
            for (int i = 0; i < nt; i++) if (w->fibers[i].state == ST_BLOCK_BAR) w->fibers[i].state = ST_RUN;
            progress = true;
        } else if (at && done && !progress) {
            fprintf(stderr, "EMU: %s block (%u,%u,%u): __syncthreads reached by %d of %d threads after %d exited\n",
                    t_kernel, blockIdx.x, blockIdx.y, blockIdx.z, at, nt, done);
            abort();
        }
        if (!progress) {
            fprintf(stderr, "EMU: deadlock in %s block (%u,%u,%u)\n", t_kernel, blockIdx.x, blockIdx.y, blockIdx.z);
            abort();
        }
    }
}

static std::atomic<long> g_launches{0};
extern "C" long emu_launch_count() { return g_launches.load(); }

void emu_launch(dim3 grid, dim3 block, size_t smem, const char* name, const std::function<void()>& body)
{
    g_launches++;
    if (getenv("EMU_TRACE"))
        fprintf(stderr, "EMU launch %s grid (%u,%u,%u) block (%u,%u,%u) smem %zu\n", name, grid.x, grid.y, grid.z,
                block.x, block.y, block.z, smem);
    if ((size_t)block.x * block.y * block.z > 1024 || smem > 227 * 1024 || grid.y > 65535 || grid.z > 65535) {
        fprintf(stderr, "EMU: invalid launch configuration for %s\n", name);
        abort();
    }
    const long nblocks = (long)grid.x * grid.y * grid.z;
    std::atomic<long> next{0};
    const char* eo = getenv("EMU_ORDER");
    const int rev = !eo ? 0 : !strcmp(eo, "rev") ? 1 : !strncmp(eo, "rand", 4) ? 2 + atoi(eo + 4) : 0;
    int nthr = getenv("EMU_THREADS") ? atoi(getenv("EMU_THREADS")) : (int)std::thread::hardware_concurrency();
    if (nthr > nblocks) nthr = (int)nblocks;
    if (nthr < 1) nthr = 1;
    auto work = [&]() {
        Worker* w = new Worker();
        t_w = w;
        t_kernel = name;
        w->body = &body;
        w->dyn_smem = smem ? guarded_alloc(smem) : nullptr;
        gridDim = grid;
        blockDim = block;
        for (;;) {
            long b = next.fetch_add(1);
            if (b >= nblocks) break;
            blockIdx = uint3{(unsigned)(b % grid.x), (unsigned)((b / grid.x) % grid.y), (unsigned)(b / ((long)grid.x * grid.y))};
            run_block(w, block, rev);
        }
        if (w->dyn_smem) guarded_free(w->dyn_smem);
        for (auto& f : w->fibers) guarded_free(f.stack);
        delete w;
        t_w = nullptr;
        t_kernel = "(host)";
    };
    std::vector<std::thread> pool;
    for (int i = 0; i < nthr; i++) pool.emplace_back(work);
    for (auto& t : pool) t.join();
}
