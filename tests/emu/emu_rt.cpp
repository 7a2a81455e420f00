// Host emulation runtime: guard-paged "device" memory + coroutine CTA scheduler (test infrastructure, tests/emu/README.md).
#include "cuda_runtime.h"
#include "emu_tma.h"
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
// ---- stream / event trace: "op stream a b n" per line, in host issue order
static std::atomic<uintptr_t> g_ids{0};
uintptr_t emu_new_id() { return ++g_ids; }
void emu_trace(const char* op, const void* a, const void* b, const void* c, size_t n)
{
    const char* path = getenv("EMU_STREAM_TRACE");
    if (!path) return;
    static std::mutex mu;
    std::lock_guard<std::mutex> lk(mu);
    FILE* f = fopen(path, "a");
    if (!f) return;
    if (!strcmp(op, "launch")) fprintf(f, "launch %p %s\n", a, (const char*)b);
    else fprintf(f, "%s %p %p %p %zu\n", op, a, b, c, n);
    fclose(f);
}
cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t st) { emu_trace("memcpy", st, d, s, n); memcpy(d, s, n); return cudaSuccess; }
cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t st) { emu_trace("memset", st, d, 0, n); memset(d, v, n); return cudaSuccess; }
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
enum { ST_RUN = 0, ST_BLOCK_BAR = 1, ST_WARP_BAR = 2, ST_DONE = 3, ST_SPIN = 4, ST_NAMED_BAR = 5 };   // ST_SPIN: a failed mbarrier wait, to be retried
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
// a box of a tensor map (or a contiguous run) to be copied when its mbarrier is waited on / its store group is waited for
struct EmuCopy { bool tensor; void* smem; const void* gmem; uint32_t bytes; CUtensorMap map; int c[3]; };
struct EmuMbar { uint32_t init; int64_t pending; int64_t tx; uint32_t phase; std::vector<EmuCopy> loads; };
struct Fiber { Ctx ctx; char* stack; int state; uint3 tid; unsigned n_ballot; int bar_id, bar_n;
               std::vector<EmuCopy> store_open, store_committed; };
struct Worker {
    std::vector<Fiber> fibers;
    std::vector<unsigned> ballot;            // [warp][2]: alternating accumulators of __ballot_sync
    std::vector<unsigned> shfl;              // [thread]: the value each lane offers to __shfl_sync
    std::map<uintptr_t, EmuMbar> mbars;      // the CTA's mbarrier objects, by shared-memory address
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
    if (!w->fibers[w->cur].store_open.empty() || !w->fibers[w->cur].store_committed.empty()) {
        fprintf(stderr, "EMU: %s block (%u,%u,%u) thread %d exits with bulk stores that were not committed and waited for\n",
                t_kernel, blockIdx.x, blockIdx.y, blockIdx.z, w->cur);
        abort();
    }
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


// ------------------------------------------------------------------ mbarrier + bulk / tensor-map copies (emu_tma.h)
struct EmuMap { uint64_t magic; const char* base; int rank; int elem; uint64_t dims[3]; uint64_t strides[2]; uint32_t box[3]; };
static const uint64_t EMU_MAP_MAGIC = 0x544d41454d55ull;
static void tma_fail(const char* what)
{
    fprintf(stderr, "EMU: %s in %s block (%u,%u,%u) thread (%u,%u)\n", what, t_kernel, blockIdx.x, blockIdx.y, blockIdx.z,
            threadIdx.x, threadIdx.y);
    abort();
}
static CUresult emu_cuTensorMapEncodeTiled(CUtensorMap* out, CUtensorMapDataType type, cuuint32_t rank, void* base,
                                           const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box,
                                           const cuuint32_t* estr, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                           CUtensorMapFloatOOBfill)
{
    if (!out || rank < 1 || rank > 3 || ((uintptr_t)base & 15)) return CUDA_ERROR_INVALID_VALUE;
    EmuMap m; memset(&m, 0, sizeof(m));
    m.magic = EMU_MAP_MAGIC; m.base = (const char*)base; m.rank = (int)rank; m.elem = (int)type;
    for (cuuint32_t i = 0; i < rank; i++) {
        if (dims[i] == 0 || box[i] == 0 || box[i] > 256 || estr[i] != 1) return CUDA_ERROR_INVALID_VALUE;
        m.dims[i] = dims[i]; m.box[i] = box[i];
    }
    if (((uint64_t)box[0] * m.elem) & 15) return CUDA_ERROR_INVALID_VALUE;        // inner box extent: a multiple of 16 bytes
    for (cuuint32_t i = 0; i + 1 < rank; i++) {
        if (strides[i] & 15) return CUDA_ERROR_INVALID_VALUE;
        m.strides[i] = strides[i];
    }
    static_assert(sizeof(EmuMap) <= sizeof(CUtensorMap), "EmuMap must fit");
    memcpy(out, &m, sizeof(m));
    return CUDA_SUCCESS;
}
cudaError_t cudaGetDriverEntryPoint(const char* symbol, void** fn, unsigned long long, cudaDriverEntryPointQueryResult* q)
{
    const bool ok = !strcmp(symbol, "cuTensorMapEncodeTiled");
    *fn = ok ? (void*)emu_cuTensorMapEncodeTiled : nullptr;
    if (q) *q = ok ? cudaDriverEntryPointSuccess : cudaDriverEntryPointSymbolNotFound;
    return cudaSuccess;
}
static uint64_t box_bytes(const EmuMap& m)
{
    uint64_t n = m.elem;
    for (int i = 0; i < m.rank; i++) n *= m.box[i];
    return n;
}
// move one box between shared memory (dense, innermost first) and the tensor; outside the tensor: zeros / skipped
static void run_copy(const EmuCopy& c, bool to_smem)
{
    if (!c.tensor) {
        if (to_smem) memcpy(c.smem, c.gmem, c.bytes); else memcpy(const_cast<void*>(c.gmem), c.smem, c.bytes);
        return;
    }
    EmuMap m; memcpy(&m, &c.map, sizeof(m));
    char* sp = (char*)c.smem;
    const uint32_t b1 = m.rank > 1 ? m.box[1] : 1, b2 = m.rank > 2 ? m.box[2] : 1;
    for (uint32_t i2 = 0; i2 < b2; i2++)
        for (uint32_t i1 = 0; i1 < b1; i1++)
            for (uint32_t i0 = 0; i0 < m.box[0]; i0++, sp += m.elem) {
                const long long x0 = (long long)c.c[0] + i0, x1 = (long long)c.c[1] + i1, x2 = (long long)c.c[2] + i2;
                const bool in = x0 >= 0 && x0 < (long long)m.dims[0] && (m.rank < 2 || (x1 >= 0 && x1 < (long long)m.dims[1])) &&
                                (m.rank < 3 || (x2 >= 0 && x2 < (long long)m.dims[2]));
                char* gp = const_cast<char*>(m.base) + x0 * m.elem + (m.rank > 1 ? x1 * (long long)m.strides[0] : 0) +
                           (m.rank > 2 ? x2 * (long long)m.strides[1] : 0);
                if (to_smem) { if (in) memcpy(sp, gp, m.elem); else memset(sp, 0, m.elem); }
                else if (in) memcpy(gp, sp, m.elem);
            }
}
static EmuMbar& mbar_of(uint64_t* bar, bool must_exist = true)
{
    if ((uintptr_t)bar & 7) tma_fail("misaligned mbarrier");
    auto& tab = t_w->mbars;
    auto it = tab.find((uintptr_t)bar);
    if (it == tab.end()) {
        if (must_exist) tma_fail("use of an mbarrier that was not initialised in this CTA");
        it = tab.emplace((uintptr_t)bar, EmuMbar{0, 0, 0, 0, {}}).first;
    }
    return it->second;
}
static void mbar_check(EmuMbar& b)
{
    if (b.pending < 0) tma_fail("more arrivals on an mbarrier than its count");
    if (b.pending == 0 && b.tx == 0) { b.phase++; b.pending = b.init; }
}
void mbar_init(uint64_t* bar, uint32_t arrivals)
{
    EmuMbar& b = mbar_of(bar, false);
    b.init = arrivals; b.pending = arrivals; b.tx = 0; b.phase = 0; b.loads.clear();
}
void mbar_expect_tx(uint64_t* bar, uint32_t bytes) { EmuMbar& b = mbar_of(bar); b.tx += bytes; b.pending--; mbar_check(b); }
void mbar_arrive(uint64_t* bar) { EmuMbar& b = mbar_of(bar); b.pending--; mbar_check(b); }
bool mbar_try_wait(uint64_t* bar, uint32_t parity)
{
    return (mbar_of(bar).phase & 1u) != (parity & 1u);
}
// The copy engines: the bytes of every issued load land at the END of a scheduling round, i.e. after every runnable
// thread has had its turn -- not at issue -- so that a read of the destination that is not ordered after the
// mbarrier wait sees poison.  Returns whether anything moved.
static bool land_loads(Worker* w)
{
    bool any = false;
    for (auto& kv : w->mbars) {
        EmuMbar& b = kv.second;
        std::vector<EmuCopy> q;
        q.swap(b.loads);
        for (const EmuCopy& c : q) {
            run_copy(c, true);
            b.tx -= c.bytes;
            mbar_check(b);
            any = true;
        }
    }
    return any;
}
bool mbar_wait(uint64_t* bar, uint32_t parity, uint32_t*)
{
    for (;;) {
        if (mbar_try_wait(bar, parity)) return true;
        yield_with(ST_SPIN);
        t_w->fibers[t_w->cur].state = ST_RUN;
    }
}
static void queue_load(EmuCopy c, uint64_t* bar, size_t smem_align)
{
    if ((uintptr_t)c.smem & (smem_align - 1)) tma_fail("bulk copy: shared-memory address not aligned");
    if (c.bytes == 0 || (c.bytes & 15)) tma_fail("bulk copy: size is not a positive multiple of 16 bytes");
    memset(c.smem, 0xFF, c.bytes);                          // until the wait, the destination holds poison
    mbar_of(bar).loads.push_back(c);
}
void tma_load_1d(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar)
{
    if ((uintptr_t)gmem_src & 15) tma_fail("bulk copy: global address not 16-byte aligned");
    emu_check_ptr(gmem_src, 1, "bulk copy source");
    queue_load(EmuCopy{false, smem_dst, gmem_src, bytes, {}, {0, 0, 0}}, bar, 16);
}
static EmuCopy tensor_copy(void* smem, const CUtensorMap* map, int rank, int c0, int c1, int c2)
{
    EmuMap m; memcpy(&m, map, sizeof(m));
    if (m.magic != EMU_MAP_MAGIC) tma_fail("tensor copy through a map that was never encoded");
    if (m.rank != rank) tma_fail("tensor copy: rank of the instruction differs from the map's");
    EmuCopy c{true, smem, nullptr, (uint32_t)box_bytes(m), *map, {c0, c1, c2}};
    return c;
}
void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) { queue_load(tensor_copy(smem_dst, map, 2, c0, c1, 0), bar, 128); }
void tma_load_3d(void* smem_dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) { queue_load(tensor_copy(smem_dst, map, 3, c0, c1, c2), bar, 128); }
void tma_store_3d(const CUtensorMap* map, const void* smem_src, int c0, int c1, int c2)
{
    if ((uintptr_t)smem_src & 127) tma_fail("tensor store: shared-memory address not 128-byte aligned");
    t_w->fibers[t_w->cur].store_open.push_back(tensor_copy(const_cast<void*>(smem_src), map, 3, c0, c1, c2));
}
void tma_store_commit()
{
    Fiber& f = t_w->fibers[t_w->cur];
    for (auto& c : f.store_open) f.store_committed.push_back(c);
    f.store_open.clear();
}
void tma_store_wait_read()
{
    Fiber& f = t_w->fibers[t_w->cur];
    for (const EmuCopy& c : f.store_committed) run_copy(c, false);        // shared memory is read NOW
    f.store_committed.clear();
}
void tma_store_wait_all() { tma_store_wait_read(); }
// bar.sync id, n: released when n threads of the CTA wait on barrier `id` (they must agree on n)
void named_bar_sync(int id, int n_threads)
{
    if (id < 1 || id > 15 || n_threads < 32 || (n_threads & 31)) tma_fail("named barrier: id not in 1..15 or thread count not whole warps");
    Fiber& f = t_w->fibers[t_w->cur];
    f.bar_id = id; f.bar_n = n_threads;
    yield_with(ST_NAMED_BAR);
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
        f.store_open.clear(); f.store_committed.clear();
        f.tid = uint3{(unsigned)i % block.x, ((unsigned)i / block.x) % block.y, (unsigned)i / (block.x * block.y)};
    }
    w->ballot.assign(2 * ((nt + 31) / 32), 0u);
    w->shfl.assign(32 * ((nt + 31) / 32), 0u);
    w->mbars.clear();
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
            if (f.state != ST_RUN && f.state != ST_SPIN) continue;
            w->cur = i;
            threadIdx = f.tid;
            ctx_switch(&w->sched, &f.ctx);
            if (f.state != ST_SPIN) progress = true;     // a fibre that only re-tried a failed mbarrier wait made no progress
            if (f.state == ST_DONE) done++;
        }
        if (land_loads(w)) progress = true;
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
        for (int id = 1; id <= 15; id++) {                       // named barriers
            int n_at = 0, want = 0;
            for (int i = 0; i < nt; i++)
                if (w->fibers[i].state == ST_NAMED_BAR && w->fibers[i].bar_id == id) {
                    if (want && want != w->fibers[i].bar_n) {
                        fprintf(stderr, "EMU: %s: threads disagree on the size of named barrier %d\n", t_kernel, id);
                        abort();
                    }
                    want = w->fibers[i].bar_n;
                    n_at++;
                }
            if (want && n_at > want) { fprintf(stderr, "EMU: %s: %d threads at named barrier %d of %d\n", t_kernel, n_at, id, want); abort(); }
            if (want && n_at == want) {
                for (int i = 0; i < nt; i++)
                    if (w->fibers[i].state == ST_NAMED_BAR && w->fibers[i].bar_id == id) w->fibers[i].state = ST_RUN;
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
            int spin = 0;
            for (int i = 0; i < nt; i++) spin += w->fibers[i].state == ST_SPIN;
            fprintf(stderr, "EMU: deadlock in %s block (%u,%u,%u)%s\n", t_kernel, blockIdx.x, blockIdx.y, blockIdx.z,
                    spin ? ": an mbarrier wait can never be satisfied (arrivals or announced bytes do not match)" : "");
            abort();
        }
    }
}

static std::atomic<long> g_launches{0};
extern "C" long emu_launch_count() { return g_launches.load(); }

void emu_launch(dim3 grid, dim3 block, size_t smem, const char* name, const std::function<void()>& body, cudaStream_t st)
{
    g_launches++;
    emu_trace("launch", st, name, 0, 0);
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
