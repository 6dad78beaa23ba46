// simt_runtime.cpp — TEST INFRASTRUCTURE (see simt_shim.h): the fibre scheduler that executes a CUDA grid on one host
// thread, and the handful of CUDA runtime calls the library's host side makes (memory is host memory, a stream is
// in-order and synchronous, a captured graph is the list of recorded operations replayed in issue order).
#include "simt_shim.h"

#include <chrono>

// Context switch.  swapcontext() makes a system call (signal mask) per switch and a kernel launch here is millions of
// switches, so x86-64 gets the dozen instructions that do the same job; anything else falls back to ucontext.
#if defined(__x86_64__)
extern "C" void simt_switch(void** save_sp, void* next_sp);
asm(R"(
.text
.globl simt_switch
.type simt_switch,@function
simt_switch:
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
.size simt_switch,.-simt_switch
)");
struct Context { void* sp = nullptr; };
static void context_make(Context* c, char* stack, size_t bytes, void (*entry)()) {
  void** top = (void**)(((uintptr_t)stack + bytes) & ~(uintptr_t)15);
  *--top = nullptr;                 // where entry() would return to: it never does
  *--top = (void*)entry;            // popped by simt_switch's ret
  for (int k = 0; k < 6; ++k) *--top = nullptr;
  c->sp = top;
}
static inline void context_switch(Context* from, Context* to) { simt_switch(&from->sp, to->sp); }
#else
#include <ucontext.h>
struct Context { ucontext_t uc; };
static void context_make(Context* c, char* stack, size_t bytes, void (*entry)()) {
  getcontext(&c->uc);
  c->uc.uc_stack.ss_sp = stack; c->uc.uc_stack.ss_size = bytes; c->uc.uc_link = nullptr;
  makecontext(&c->uc, entry, 0);
}
static inline void context_switch(Context* from, Context* to) { swapcontext(&from->uc, &to->uc); }
#endif

#if defined(__SANITIZE_ADDRESS__)
extern "C" void __sanitizer_start_switch_fiber(void** fake_stack_save, const void* bottom, size_t size);
extern "C" void __sanitizer_finish_switch_fiber(void* fake_stack_save, const void** bottom_old, size_t* size_old);
#define SIMT_ASAN 1
#else
#define SIMT_ASAN 0
#endif

// ThreadSanitizer (build mode "tsan": kernels instrumented, this file not): every CUDA thread index is a TSan fibre, switches
// carry NO synchronisation, and the happens-before edges are exactly the ones CUDA gives: launch boundaries, __syncthreads,
// __syncwarp, mbarrier arrive -> wait, __threadfence.  A conflicting pair of plain accesses that none of these orders is
// reported as a data race.
#if defined(SIMT_TSAN)
extern "C" {
void* __tsan_get_current_fiber(void);
void* __tsan_create_fiber(unsigned flags);
void __tsan_destroy_fiber(void* fiber);
void __tsan_switch_to_fiber(void* fiber, unsigned flags);
void __tsan_acquire(void* addr);
void __tsan_release(void* addr);
}
#define TSAN_SWITCH(f) __tsan_switch_to_fiber((f), 1u /* no synchronisation */)
#define TSAN_ACQUIRE(a) __tsan_acquire((void*)(a))
#define TSAN_RELEASE(a) __tsan_release((void*)(a))
#else
#define TSAN_SWITCH(f) ((void)0)
#define TSAN_ACQUIRE(a) ((void)0)
#define TSAN_RELEASE(a) ((void)0)
#endif

struct SimtStream { int dummy; };
struct SimtEvent { std::chrono::steady_clock::time_point at; };
struct SimtGraph { std::vector<std::function<void()>> ops; };

namespace simt {

Builtins g;

namespace {

constexpr size_t kStackBytes = 256 * 1024;
constexpr unsigned kMaxThreads = 1024;

struct Fibre {
  Context ctx;
  char* stack = nullptr;
  void* fake = nullptr;          // ASan fake-stack handle while the fibre is switched out
  void* tsan = nullptr;          // TSan fibre of this thread index (kept across blocks and launches)
  bool done = true;
};
struct WarpSync {
  unsigned arrived = 0, releasing = 0, part = 0, live = 0;
  char hb = 0;                   // happens-before token of __syncwarp
  unsigned long long val[32], snap[32];
};
struct Block {
  unsigned n = 0, alive = 0;
  unsigned bar_arrived = 0, bar_gen = 0;
  WarpSync warp[kMaxThreads / 32];
  Fibre fib[kMaxThreads];
  Context main;
  const void* main_bottom = nullptr;
  size_t main_size = 0;
  unsigned cur = 0;
  const std::function<void()>* body = nullptr;
  void* dyn = nullptr;
  unsigned long long progress = 0;
  void* tsan_main = nullptr;
  char hb_bar = 0, hb_launch_start = 0, hb_launch_end = 0, hb_fence = 0;
};
Block B;
SimtGraph* g_capture = nullptr;
unsigned long long g_switches = 0, g_launches = 0;

// Adversarial mode (SIMT_SCHED_SEED != 0): blocks run in a random order, every scheduler pass visits a random subset of
// the live fibres in a random order, and deferred work (bulk copies) lands as late as it legally can.  Whatever the
// schedule, the results must not change: that is the race / ordering check (a missing barrier, a queue shared between
// warps, a result that depends on which atomic wins, a stage read before its copy landed all show as a mismatch).
unsigned long long g_rng = 0;
bool g_adversarial = false;
unsigned rnd() { g_rng ^= g_rng << 13; g_rng ^= g_rng >> 7; g_rng ^= g_rng << 17; return (unsigned)(g_rng >> 32); }
struct Deferred { const void* key; std::function<void()> fn; };
std::vector<Deferred> g_deferred;

void fibre_entry() {
#if SIMT_ASAN
  __sanitizer_finish_switch_fiber(nullptr, &B.main_bottom, &B.main_size);
#endif
  TSAN_ACQUIRE(&B.hb_launch_start);            // everything before the launch happens-before every thread of it
  (*B.body)();
  TSAN_RELEASE(&B.hb_launch_end);
  const unsigned t = B.cur;
  B.fib[t].done = true;
  B.alive--;
  B.warp[t >> 5].live &= ~(1u << (t & 31u));
  B.progress++;
#if SIMT_ASAN
  __sanitizer_start_switch_fiber(nullptr, B.main_bottom, B.main_size);     // this fibre never runs again
#endif
  TSAN_SWITCH(B.tsan_main);
  context_switch(&B.fib[t].ctx, &B.main);
}

void die(const char* what) {
  std::fprintf(stderr, "simt: %s (block %u of %u, %u threads, %u alive)\n", what, g.bid.x, g.gdim.x, B.n, B.alive);
  std::abort();
}

void run_block(unsigned n) {
  B.n = n; B.alive = n; B.bar_arrived = 0; B.bar_gen = 0;
  for (unsigned w = 0; w < (n + 31u) / 32u; ++w) {
    WarpSync& W = B.warp[w];
    W.arrived = W.releasing = W.part = 0;
    const unsigned lanes = std::min(32u, n - w * 32u);
    W.live = lanes == 32u ? 0xFFFFFFFFu : ((1u << lanes) - 1u);
  }
  for (unsigned t = 0; t < n; ++t) {
    Fibre& f = B.fib[t];
    if (!f.stack) f.stack = (char*)std::malloc(kStackBytes);
    context_make(&f.ctx, f.stack, kStackBytes, fibre_entry);
#if defined(SIMT_TSAN)
    if (!f.tsan) f.tsan = __tsan_create_fiber(0);
#endif
    f.done = false; f.fake = nullptr;
  }
  unsigned idle = 0;
  static unsigned order[kMaxThreads];
  for (unsigned t = 0; t < n; ++t) order[t] = t;
  while (B.alive) {
    const unsigned long long before = B.progress;
    if (g_adversarial) for (unsigned t = n - 1; t > 0; --t) std::swap(order[t], order[rnd() % (t + 1u)]);
    for (unsigned k = 0; k < n; ++k) {
      const unsigned t = order[k];
      Fibre& f = B.fib[t];
      if (f.done) continue;
      if (g_adversarial && (rnd() & 3u) == 0u) continue;          // this fibre sits the pass out
      B.cur = t; g.tid.x = t;
      ++g_switches;
#if SIMT_ASAN
      void* fake_main = nullptr;
      __sanitizer_start_switch_fiber(&fake_main, f.stack, kStackBytes);
#endif
      TSAN_SWITCH(f.tsan);
      context_switch(&B.main, &f.ctx);
#if SIMT_ASAN
      __sanitizer_finish_switch_fiber(fake_main, nullptr, nullptr);
#endif
    }
    if (B.progress == before) { if (++idle > 100000u) die("deadlock: no fibre can make progress"); }
    else idle = 0;
  }
}

void execute_grid(unsigned grid, unsigned block, size_t smem, const std::function<void()>& body) {
  if (block == 0 || block > kMaxThreads) die("bad block size");
  ++g_launches;
  B.body = &body;
  B.dyn = smem ? std::malloc(smem) : nullptr;      // its own allocation: ASan sees an overrun of the dynamic shared memory
  g.bdim = uint3{block, 1, 1}; g.gdim = uint3{grid, 1, 1};
  const char* seed = std::getenv("SIMT_SCHED_SEED");
  g_adversarial = seed && std::atoll(seed) != 0;
  if (g_adversarial) { g_rng = (unsigned long long)std::atoll(seed) * 0x9E3779B97F4A7C15ull + g_launches; rnd(); rnd(); }
#if defined(SIMT_TSAN)
  B.tsan_main = __tsan_get_current_fiber();
#endif
  TSAN_RELEASE(&B.hb_launch_start);
  std::vector<unsigned> blocks(grid);
  for (unsigned b = 0; b < grid; ++b) blocks[b] = b;
  if (g_adversarial) for (unsigned b = grid; b > 1; --b) std::swap(blocks[b - 1], blocks[rnd() % b]);
  for (unsigned b : blocks) {
    g.bid = uint3{b, 0, 0};
    if (B.dyn) std::memset(B.dyn, 0xCD, smem);     // shared memory starts as garbage in every block
    TSAN_RELEASE(&B.hb_launch_start);              // again: the fill above is the host's, and so is what it learnt from the block before
    run_block(block);
    // Shared memory (statics, the dynamic buffer) is reused by the next block, which on the GPU has its own: for
    // ThreadSanitizer the blocks of a launch are therefore ordered one after the other; a conflict BETWEEN blocks is
    // what the seeded block orders of the adversarial schedules are for.
    TSAN_ACQUIRE(&B.hb_launch_end);
    if (!g_deferred.empty()) die("a bulk copy was still in flight when its block ended");
  }
  TSAN_ACQUIRE(&B.hb_launch_end);               // the launch happens-before whatever the host does next
  std::free(B.dyn); B.dyn = nullptr; B.body = nullptr;
}

}  // namespace

void yield() {
  Fibre& f = B.fib[B.cur];
#if SIMT_ASAN
  __sanitizer_start_switch_fiber(&f.fake, B.main_bottom, B.main_size);
#endif
  TSAN_SWITCH(B.tsan_main);
  context_switch(&f.ctx, &B.main);
#if SIMT_ASAN
  __sanitizer_finish_switch_fiber(f.fake, &B.main_bottom, &B.main_size);
#endif
}
void note_progress() { B.progress++; }
void hb_release(const void* token) { TSAN_RELEASE(token); (void)token; }
void hb_acquire(const void* token) { TSAN_ACQUIRE(token); (void)token; }
void hb_fence() { TSAN_RELEASE(&B.hb_fence); TSAN_ACQUIRE(&B.hb_fence); }
bool defer(const void* key, std::function<void()> fn) {
  if (!g_adversarial) return false;                // the caller does the work now
  g_deferred.push_back(Deferred{key, std::move(fn)});
  TSAN_RELEASE(key);                                // whoever runs it later comes after the issue (and its allocation)
  return true;
}
void run_deferred(const void* key) {
  TSAN_ACQUIRE(key);
  for (size_t k = 0; k < g_deferred.size();) {
    if (g_deferred[k].key == key) { auto fn = std::move(g_deferred[k].fn); g_deferred.erase(g_deferred.begin() + k); fn(); }
    else ++k;
  }
}
void* dyn_smem() { return B.dyn; }

void syncthreads() {
  const unsigned gen = B.bar_gen;
  TSAN_RELEASE(&B.hb_bar);
  B.bar_arrived++; B.progress++;
  for (;;) {
    if (B.bar_gen != gen) break;
    if (B.bar_arrived >= B.alive) { B.bar_arrived = 0; B.bar_gen++; B.progress++; break; }   // exited threads count as arrived
    yield();
  }
  TSAN_ACQUIRE(&B.hb_bar);
}

void warp_exchange(unsigned mask, unsigned long long v, unsigned long long out[32], unsigned* participants, bool fence) {
  const unsigned t = B.cur, lane = t & 31u, bit = 1u << lane;
  WarpSync& W = B.warp[t >> 5];
  if (!(mask & bit)) die("warp collective called by a lane that is not in its mask");
  while (W.releasing) yield();                     // the previous collective is still being picked up
  if (fence) TSAN_RELEASE(&W.hb);
  W.val[lane] = v; W.arrived |= bit; B.progress++;
  for (;;) {
    if (W.releasing & bit) break;                  // completed by another lane
    const unsigned need = mask & W.live;
    if (!W.releasing && (W.arrived & need) == need) {
      std::memcpy(W.snap, W.val, sizeof(W.snap));
      W.part = W.arrived; W.releasing = W.arrived; B.progress++;
      break;
    }
    yield();
  }
  std::memcpy(out, W.snap, sizeof(W.snap));
  *participants = W.part;
  W.releasing &= ~bit; W.arrived &= ~bit;
  if (!W.releasing) B.progress++;
  if (fence) TSAN_ACQUIRE(&W.hb);
}

void run_grid(unsigned grid, unsigned block, size_t smem, std::function<void()> body) {
  if (g_capture) { g_capture->ops.push_back([=]() { execute_grid(grid, block, smem, body); }); return; }
  execute_grid(grid, block, smem, body);
}

int blocks_per_sm() { const char* e = std::getenv("SIMT_BLOCKS_PER_SM"); return e ? std::atoi(e) : 2; }

}  // namespace simt

// ---------------------------------------------------------------------------------------------- runtime calls
using simt::g_capture;

const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : "simt: error"; }
cudaError_t cudaGetLastError() { return cudaSuccess; }
cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
cudaError_t cudaGetDevice(int* d) { *d = 0; return cudaSuccess; }
cudaError_t cudaDeviceGetAttribute(int* v, int attr, int) {
  const char* e = std::getenv("SIMT_SMS");
  *v = attr == cudaDevAttrMultiProcessorCount ? (e ? std::atoi(e) : 3) : 0;
  return cudaSuccess;
}
cudaError_t cudaMemcpyAsync(void* dst, const void* src, size_t n, cudaMemcpyKind, cudaStream_t) {
  if (g_capture) { g_capture->ops.push_back([=]() { std::memmove(dst, src, n); }); return cudaSuccess; }
  std::memmove(dst, src, n);
  return cudaSuccess;
}
cudaError_t cudaMemcpy(void* dst, const void* src, size_t n, cudaMemcpyKind k) { return cudaMemcpyAsync(dst, src, n, k, nullptr); }
cudaError_t cudaMemsetAsync(void* dst, int v, size_t n, cudaStream_t) {
  if (g_capture) { g_capture->ops.push_back([=]() { std::memset(dst, v, n); }); return cudaSuccess; }
  std::memset(dst, v, n);
  return cudaSuccess;
}
cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = new SimtStream(); return cudaSuccess; }
cudaError_t cudaStreamDestroy(cudaStream_t s) { delete s; return cudaSuccess; }
cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
cudaError_t cudaStreamBeginCapture(cudaStream_t, int) {
  if (g_capture || std::getenv("SIMT_NO_GRAPHS")) return cudaErrorUnknown;
  g_capture = new SimtGraph();
  return cudaSuccess;
}
cudaError_t cudaStreamEndCapture(cudaStream_t, cudaGraph_t* out) {
  *out = g_capture; g_capture = nullptr;
  return *out ? cudaSuccess : cudaErrorUnknown;
}
cudaError_t cudaGraphInstantiate(cudaGraphExec_t* out, cudaGraph_t gph, unsigned long long) { *out = new SimtGraph(*gph); return cudaSuccess; }
cudaError_t cudaGraphDestroy(cudaGraph_t gph) { delete gph; return cudaSuccess; }
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t gph) { delete gph; return cudaSuccess; }
cudaError_t cudaGraphLaunch(cudaGraphExec_t gph, cudaStream_t) {
  for (auto& op : gph->ops) op();
  return cudaSuccess;
}
cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = new SimtEvent(); return cudaSuccess; }
cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned) { return cudaEventCreate(e); }
cudaError_t cudaEventDestroy(cudaEvent_t e) { delete e; return cudaSuccess; }
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t) { e->at = std::chrono::steady_clock::now(); return cudaSuccess; }
cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t a, cudaEvent_t b) {
  *ms = std::chrono::duration<float, std::milli>(b->at - a->at).count();
  return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------- for the harness
extern "C" {
// "Device" memory for the workspace: its own heap block (ASan red zones on both sides), filled with garbage.
void* simt_alloc(size_t bytes) {
  void* p = nullptr;
  if (posix_memalign(&p, 256, bytes)) return nullptr;
  unsigned long long x = 0x9E3779B97F4A7C15ull;
  unsigned long long* q = (unsigned long long*)p;
  for (size_t i = 0; i < bytes / 8; ++i) { x ^= x << 13; x ^= x >> 7; x ^= x << 17; q[i] = x; }
  for (size_t i = bytes & ~(size_t)7; i < bytes; ++i) ((unsigned char*)p)[i] = 0xA5;
  return p;
}
void simt_free(void* p) { std::free(p); }
unsigned long long simt_switches() { return simt::g_switches; }
unsigned long long simt_launches() { return simt::g_launches; }
}

// Self-test of the memcheck: one lane of a two-warp block reads the byte right behind a `bytes`-long block.  Under the
// sanitizer build this must end the process with an AddressSanitizer report (tests/test_simt_kernels.py checks that it does).
extern "C" int simt_selftest_overrun(const unsigned char* p, size_t bytes) {
  int seen = 0;
  simt::run_grid(1, 64, 0, [&]() {
    __syncthreads();
    if (threadIdx.x == 37u) seen = p[bytes];
    __syncwarp();
  });
  return seen;
}
