// cuda_emu.cpp -- fibers, CTA scheduler, warp collectives and guarded allocations of the host CUDA model (see cuda_emu.h).
// TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.
#include "cuda_emu.h"

#include <sys/mman.h>
#include <unistd.h>

#include <algorithm>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>
#include <vector>

// Context switch (x86-64 System V): callee-saved registers go on the old stack, stack pointers are swapped.
extern "C" void emu_switch(void** save_sp, void* load_sp);
asm(R"(
.text
.globl emu_switch
.type emu_switch,@function
emu_switch:
    pushq %rbp
    pushq %rbx
    pushq %r12
    pushq %r13
    pushq %r14
    pushq %r15
    movq %rsp, (%rdi)
    movq %rsi, %rsp
    popq %r15
    popq %r14
    popq %r13
    popq %r12
    popq %rbx
    popq %rbp
    ret
.size emu_switch,.-emu_switch
)");

// Race-detector build (-DHOUGH_EMU_TSAN, g++ -fsanitize=thread; tests/emu/build_emu.py --tsan): every CUDA thread is a
// ThreadSanitizer fiber of its own, switched WITHOUT synchronisation, so that two CUDA threads of a CTA are concurrent for the
// detector exactly where CUDA says they are: the only happens-before edges inside a CTA are __syncthreads (all threads),
// __syncwarp (the lanes of the mask) and program order.  ballot / shuffle / match exchange registers and order no memory.
// Atomics are relaxed (cuda_emu.h), as CUDA's are.  Kernel launches and the CTAs that follow one another on one worker are
// ordered through the scheduler (they reuse the same host memory as "shared memory").
#ifdef HOUGH_EMU_TSAN
extern "C" {
void* __tsan_get_current_fiber(void);
void* __tsan_create_fiber(unsigned flags);
void __tsan_destroy_fiber(void* fiber);
void __tsan_switch_to_fiber(void* fiber, unsigned flags);  // flags 1: no synchronisation on the switch
void __tsan_acquire(void* addr);
void __tsan_release(void* addr);
}
#define TSAN_ONLY(...) __VA_ARGS__
#else
#define TSAN_ONLY(...)
#endif

namespace cuda_emu {

enum State { RUNNABLE, AT_BARRIER, AT_WARP, DONE };

struct Fiber {
    void* sp;
    int tid;
    State state;
};

struct Pending {  // one warp collective in flight
    unsigned mask, arrived;
    WarpOp op;
    unsigned long long val[32];
    int arg[32];
};

struct Warp {
    Pending pend[8];
    char sync_token[8];  // race-detector build: what the lanes of a __syncwarp release and acquire, one per slot of pend
    unsigned long long res[32];
    unsigned gen[32];  // per lane: bumped when the collective the lane waits in completes
};

// Per OS thread ("worker"): the CTA it is running.  With one worker (the default) the CTAs of a grid run one after another;
// with several (cuda_emu_set_workers) each worker takes the next CTA of the grid, so that persistent CTAs really share the
// work counter, the deferred list and their per-CTA scratch slabs, and global atomics are real atomics.
thread_local Fiber* g_cur = nullptr;
thread_local unsigned char* g_smem = nullptr;
thread_local unsigned g_smem_bytes = 0;
unsigned g_smem_window = 1024;
dim3 g_block_dim, g_grid_dim;
long long g_violations = 0;

static thread_local uint3 g_block_idx;
static thread_local void* g_sched_sp = nullptr;
static const std::function<void()>* g_body = nullptr;
static thread_local std::vector<Fiber> g_fibers;
static thread_local std::vector<Warp> g_warps;
static thread_local std::vector<unsigned char*> g_stacks;
static thread_local std::vector<int> g_ready;  // runnable fibers that are not running
static thread_local int g_n_barrier = 0, g_n_done = 0;
static const size_t kStackBytes = 256 * 1024;
static unsigned long long g_seed = 0x9E3779B97F4A7C15ull;
static thread_local unsigned long long g_rng = 0x9E3779B97F4A7C15ull;
static int g_preempt_per_1024 = 0;  // chance (in 1/1024) that an atomic / cache-bypassing access yields first
static int g_workers = 1;
static char g_first_violation[256] = "";
static std::mutex g_mutex;
#ifdef HOUGH_EMU_TSAN
static thread_local std::vector<void*> g_tsan_fibers;  // one detector context per CUDA thread slot of this worker
static thread_local void* g_tsan_sched = nullptr;
static thread_local char g_barrier_token, g_start_token, g_done_token;  // addresses only: what release / acquire name
#endif

static unsigned rnd()
{
    g_rng ^= g_rng << 13; g_rng ^= g_rng >> 7; g_rng ^= g_rng << 17;
    return (unsigned)(g_rng >> 32);
}

uint3 cur_thread_idx() { return uint3{(unsigned)g_cur->tid, 0, 0}; }
uint3 cur_block_idx() { return g_block_idx; }

void violation(const char* what, unsigned long long a, unsigned long long lim)
{
    std::lock_guard<std::mutex> lock(g_mutex);
    if (g_violations == 0) {
        snprintf(g_first_violation, sizeof g_first_violation, "%s (value %llu, limit %llu; block %u thread %d)", what, a, lim,
                 g_block_idx.x, g_cur ? g_cur->tid : -1);
        fprintf(stderr, "cuda_emu: VIOLATION: %s\n", g_first_violation);
    }
    ++g_violations;
}

static void yield_to_scheduler()
{
    TSAN_ONLY(__tsan_switch_to_fiber(g_tsan_sched, 1);)
    emu_switch(&g_cur->sp, g_sched_sp);
}

void maybe_yield()
{
    if (g_preempt_per_1024 && g_cur && (int)(rnd() & 1023u) < g_preempt_per_1024) {  // stays RUNNABLE
        g_ready.push_back(g_cur->tid);
        yield_to_scheduler();
    }
}

void sync_threads()
{
    g_cur->state = AT_BARRIER;
    ++g_n_barrier;
    TSAN_ONLY(__tsan_release(&g_barrier_token);)  // every thread releases before the first one leaves ...
    yield_to_scheduler();
    TSAN_ONLY(__tsan_acquire(&g_barrier_token);)  // ... and acquires all of them
}

static void complete(Warp& w, Pending& p)
{
    for (int l = 0; l < 32; ++l) {
        if (!((p.mask >> l) & 1u)) continue;
        unsigned long long r = 0;
        switch (p.op) {
            case W_BALLOT: for (int j = 0; j < 32; ++j) if (((p.mask >> j) & 1u) && p.val[j]) r |= 1ull << j; break;
            case W_SHFL: { const int s = p.arg[l] & 31; r = ((p.mask >> s) & 1u) ? p.val[s] : p.val[l]; break; }
            case W_SHFL_UP: { const int s = l - p.arg[l]; r = (s >= 0 && ((p.mask >> s) & 1u)) ? p.val[s] : p.val[l]; break; }
            case W_SHFL_DOWN: { const int s = l + p.arg[l]; r = (s < 32 && ((p.mask >> s) & 1u)) ? p.val[s] : p.val[l]; break; }
            case W_SHFL_XOR: { const int s = (l ^ p.arg[l]) & 31; r = ((p.mask >> s) & 1u) ? p.val[s] : p.val[l]; break; }
            case W_MATCH_ANY: for (int j = 0; j < 32; ++j) if (((p.mask >> j) & 1u) && p.val[j] == p.val[l]) r |= 1ull << j; break;
            case W_SYNC: break;
        }
        w.res[l] = r;
        ++w.gen[l];
    }
    p.mask = 0;
    p.arrived = 0;
}

unsigned long long warp_collective(WarpOp op, unsigned mask, unsigned long long val, int arg)
{
    Fiber* f = g_cur;
    const int lane = f->tid & 31;
    Warp& w = g_warps[f->tid >> 5];
    // lanes of a partial last warp do not exist
    const int nthr = (int)g_block_dim.x, first = f->tid & ~31;
    unsigned exist = 0xffffffffu;
    if (first + 32 > nthr) exist = (1u << (nthr - first)) - 1u;
    mask &= exist;
    if (!((mask >> lane) & 1u)) { violation("warp collective called by a lane that is not in its mask", mask, lane); return 0; }
    // A lane joins the collective in flight that names the same lanes and operation and that it has not joined yet; lanes
    // that skipped a sub-mask collective may already wait in a later one, so collectives in flight may share lanes.
    Pending* p = nullptr;
    for (Pending& q : w.pend)
        if (q.mask == mask && q.op == op && !((q.arrived >> lane) & 1u)) { p = &q; break; }
    if (!p) {
        for (Pending& q : w.pend)
            if (!q.mask) { p = &q; break; }
        if (!p) { violation("more than 8 warp collectives in flight in one warp", mask, 8); return 0; }
        p->mask = mask; p->arrived = 0; p->op = op;
    }
    p->val[lane] = val;
    p->arg[lane] = arg;
    p->arrived |= 1u << lane;
    TSAN_ONLY(char* const token = &w.sync_token[p - w.pend]; if (op == W_SYNC) __tsan_release(token);)
    if (p->arrived == p->mask) {
        const unsigned m = p->mask;
        complete(w, *p);
        for (int l = 0; l < 32; ++l)
            if (((m >> l) & 1u) && l != lane) { g_fibers[first + l].state = RUNNABLE; g_ready.push_back(first + l); }
    } else {
        const unsigned my_gen = w.gen[lane];
        f->state = AT_WARP;
        while (w.gen[lane] == my_gen) yield_to_scheduler();
    }
    TSAN_ONLY(if (op == W_SYNC) __tsan_acquire(token);)
    return w.res[lane];
}

static void fiber_main()
{
    TSAN_ONLY(__tsan_acquire(&g_start_token);)  // after the scheduler's set-up of this CTA (and whatever ran before it)
    (*g_body)();
    TSAN_ONLY(__tsan_release(&g_done_token);)
    g_cur->state = DONE;
    ++g_n_done;
    for (;;) yield_to_scheduler();
}

static void* guarded(size_t bytes, size_t* map_bytes, void** map_base)
{
    const size_t page = 4096, need = (bytes + 15) & ~(size_t)15;
    const size_t body = (need + page - 1) / page * page;
    unsigned char* m = static_cast<unsigned char*>(mmap(nullptr, body + 2 * page, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0));
    if (m == MAP_FAILED) return nullptr;
    mprotect(m, page, PROT_NONE);                // an underrun of more than the alignment slack faults
    mprotect(m + page + body, page, PROT_NONE);  // an overrun faults at once
    *map_bytes = body + 2 * page;
    *map_base = m;
    return m + page + body - need;
}

static std::map<void*, std::pair<void*, size_t>> g_allocs;

void* dev_alloc(size_t bytes)
{
    size_t mb; void* base;
    void* p = guarded(bytes ? bytes : 16, &mb, &base);
    if (p) { memset(p, 0xCD, bytes); g_allocs[p] = {base, mb}; }  // device memory is not zero-initialised
    return p;
}

void dev_free(void* p)
{
    if (!p) return;
    auto it = g_allocs.find(p);
    if (it == g_allocs.end()) { violation("cudaFree of an unknown pointer", (unsigned long long)(uintptr_t)p, 0); return; }
    munmap(it->second.first, it->second.second);
    g_allocs.erase(it);
}

static void run_cta(unsigned b, int nthr, unsigned char* smem, size_t smem_bytes)
{
    while ((int)g_stacks.size() < nthr) {
        unsigned char* st = static_cast<unsigned char*>(mmap(nullptr, kStackBytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0));
        if (st == MAP_FAILED) { fprintf(stderr, "cuda_emu: out of memory for fiber stacks\n"); abort(); }
        mprotect(st, 4096, PROT_NONE);
        g_stacks.push_back(st);
    }
    g_block_idx = uint3{b, 0, 0};
    g_smem = smem;
    g_smem_bytes = (unsigned)smem_bytes;
    memset(smem, 0xA5, smem_bytes);  // shared memory is not zero-initialised
#ifdef HOUGH_EMU_TSAN
    if (!g_tsan_sched) g_tsan_sched = __tsan_get_current_fiber();
    while ((int)g_tsan_fibers.size() < nthr) g_tsan_fibers.push_back(__tsan_create_fiber(0));
    __tsan_release(&g_start_token);
#endif
    g_fibers.assign(nthr, Fiber{});
    g_warps.assign((nthr + 31) / 32, Warp{});
    g_ready.clear();
    g_n_barrier = 0;
    g_n_done = 0;
    for (int t = 0; t < nthr; ++t) {
        Fiber& f = g_fibers[t];
        f.tid = t;
        f.state = RUNNABLE;
        void** top = reinterpret_cast<void**>(g_stacks[t] + kStackBytes);  // 16-byte aligned
        void** sp = top - 8;
        for (int i = 0; i < 8; ++i) sp[i] = nullptr;
        sp[6] = reinterpret_cast<void*>(&fiber_main);  // "return address" of the first switch into the fiber
        f.sp = sp;
        g_ready.push_back(t);
    }
    while (g_n_done < nthr) {
        if (!g_ready.empty()) {  // resume a runnable fiber picked at random
            const size_t i = rnd() % g_ready.size();
            const int t = g_ready[i];
            g_ready[i] = g_ready.back();
            g_ready.pop_back();
            g_cur = &g_fibers[t];
            TSAN_ONLY(__tsan_switch_to_fiber(g_tsan_fibers[t], 1);)
            emu_switch(&g_sched_sp, g_cur->sp);
            continue;
        }
        if (g_n_barrier && g_n_barrier == nthr - g_n_done) {  // every live thread has arrived
            for (Fiber& f : g_fibers) if (f.state == AT_BARRIER) { f.state = RUNNABLE; g_ready.push_back(f.tid); }
            g_n_barrier = 0;
            continue;
        }
        int nb = 0, nw = 0;
        for (Fiber& f : g_fibers) { nb += f.state == AT_BARRIER; nw += f.state == AT_WARP; }
        fprintf(stderr, "cuda_emu: DEADLOCK in block %u: %d threads at __syncthreads, %d in warp collectives, %d done of %d\n",
                b, nb, nw, g_n_done, nthr);
        abort();
    }
    TSAN_ONLY(__tsan_acquire(&g_done_token);)  // the CTA's accesses happen before whatever this worker does next
    g_cur = nullptr;
    g_smem = nullptr;
}

void launch(dim3 grid, dim3 block, size_t smem_bytes, const std::function<void()>& body)
{
    const int nthr = (int)block.x;
    g_block_dim = block;
    g_grid_dim = grid;
    g_body = &body;
    const int workers = (int)std::min<unsigned>((unsigned)std::max(g_workers, 1), grid.x);
    std::atomic<unsigned> next{0};
    auto worker = [&](int wid) {
        g_rng = g_seed ^ (0x9E3779B97F4A7C15ull * (unsigned long long)(wid + 1));
        if (!g_rng) g_rng = 1;
        size_t smem_map = 0; void* smem_base = nullptr;
        unsigned char* smem = static_cast<unsigned char*>(guarded(smem_bytes ? smem_bytes : 16, &smem_map, &smem_base));
        for (unsigned b = next.fetch_add(1); b < grid.x; b = next.fetch_add(1)) run_cta(b, nthr, smem, smem_bytes);
        munmap(smem_base, smem_map);
        if (workers > 1) {  // a worker thread ends with the launch: give its fiber stacks back
            for (unsigned char* st : g_stacks) munmap(st, kStackBytes);
            g_stacks.clear();
#ifdef HOUGH_EMU_TSAN
            for (void* f : g_tsan_fibers) __tsan_destroy_fiber(f);
            g_tsan_fibers.clear();
            g_tsan_sched = nullptr;
#endif
        }
    };
    if (workers <= 1) {
        worker(0);
    } else {
        std::vector<std::thread> th;
        for (int w = 0; w < workers; ++w) th.emplace_back(worker, w);
        for (auto& t : th) t.join();
    }
}

}  // namespace cuda_emu

extern "C" long long cuda_emu_violations(void) { return cuda_emu::g_violations; }
extern "C" const char* cuda_emu_first_violation(void) { return cuda_emu::g_first_violation; }
extern "C" void cuda_emu_reset_violations(void) { cuda_emu::g_violations = 0; cuda_emu::g_first_violation[0] = 0; }
extern "C" void cuda_emu_configure(unsigned long long seed, int preempt_per_1024, unsigned smem_window)
{
    cuda_emu::g_seed = 0x9E3779B97F4A7C15ull ^ (seed * 0xD1342543DE82EF95ull);
    cuda_emu::g_preempt_per_1024 = preempt_per_1024;
    cuda_emu::g_smem_window = smem_window;
}
// CTAs of a grid that run at the same time, each on its own OS thread (1 = one after another)
extern "C" void cuda_emu_set_workers(int n) { cuda_emu::g_workers = n < 1 ? 1 : n; }
