// simt_shim.h — TEST INFRASTRUCTURE, not product code.  A host-side stand-in for the CUDA language and runtime, just
// large enough to compile paper_2606_14603_b200/csrc/*.cu{,h} UNCHANGED (apart from the mechanical rewrites of
// tests/simt/build.py) with g++ and to execute the kernels on the CPU the way the GPU would: every CUDA thread of a block
// is a fibre (ucontext) with its own stack and threadIdx, warps synchronise through __shfl / __ballot / __syncwarp
// rendezvous, blocks through __syncthreads, blocks of a grid run one after the other (no kernel of the product waits on
// another block).  What it is for (tests/test_simt_kernels.py):
//   * the kernels' logic is checked against the oracle by `pytest -m "not gpu"`, on a machine without a GPU;
//   * the same build under -fsanitize=address,undefined is a memcheck of every kernel access against the exact
//     workspace allocation (compute-sanitizer is closed on the GPU pool, profiles/r2_sanitizers.md);
//   * the workspace is filled with garbage before use, so reliance on zero-initialised memory shows up as a mismatch;
//   * seeded adversarial schedules (SIMT_SCHED_SEED) and a ThreadSanitizer build (one TSan fibre per CUDA thread,
//     happens-before only where CUDA gives it) are the race check.
// What it is NOT: a CPU fallback.  The package (paper_2606_14603_b200/) never builds, loads or mentions it; the
// product path fails loudly without the CUDA library (binding.load_library).  It says nothing about performance.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <string>
#include <utility>
#include <vector>

// ---------------------------------------------------------------------------------------------- language
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __noinline__ __attribute__((noinline))
#define __grid_constant__
#define __launch_bounds__(...)
#define __align__(n) __attribute__((aligned(n)))
#define __shared__ static          /* one block at a time, one OS thread: a static IS block-shared */

struct alignas(16) int4 { int x, y, z, w; };
struct alignas(16) uint4 { unsigned x, y, z, w; };
struct alignas(8) uint2 { unsigned x, y; };
struct alignas(4) uchar4 { unsigned char x, y, z, w; };
struct uint3 { unsigned x, y, z; };
static inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }
static inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }
static inline uint2 make_uint2(unsigned x, unsigned y) { return uint2{x, y}; }
static inline uchar4 make_uchar4(unsigned char x, unsigned char y, unsigned char z, unsigned char w) { return uchar4{x, y, z, w}; }

namespace simt {
struct Builtins { uint3 tid, bid, bdim, gdim; };
extern Builtins g;
void yield();                                  // back to the block scheduler; resumed later
void note_progress();                          // something another fibre may be waiting for has happened
void* dyn_smem();                              // the launch's dynamic shared memory
bool defer(const void* key, std::function<void()> fn);   // adversarial mode: queue fn under key, true; else false
void run_deferred(const void* key);            // run (and forget) everything queued under key
void syncthreads();
// Warp rendezvous: every live lane named in `mask` deposits v; each gets all deposits and who took part.
// `fence`: the rendezvous also orders the lanes' memory accesses (__syncwarp does, shuffles and ballots do not).
void warp_exchange(unsigned mask, unsigned long long v, unsigned long long out[32], unsigned* participants, bool fence = false);
// ThreadSanitizer build (tests/simt/build.py mode "tsan"): happens-before edges; no-ops otherwise.
void hb_release(const void* token);
void hb_acquire(const void* token);
void hb_fence();                               // __threadfence: ordered against every other fibre that fences
template <class T> inline void relaxed_store(T* p, T v) { __atomic_store_n(p, v, __ATOMIC_RELAXED); }
template <class T> inline T relaxed_load(const T* p) { return __atomic_load_n(p, __ATOMIC_RELAXED); }
}  // namespace simt
#define threadIdx (simt::g.tid)
#define blockIdx (simt::g.bid)
#define blockDim (simt::g.bdim)
#define gridDim (simt::g.gdim)

// ---------------------------------------------------------------------------------------------- intrinsics
static inline int min(int a, int b) { return a < b ? a : b; }
static inline int max(int a, int b) { return a > b ? a : b; }
static inline unsigned min(unsigned a, unsigned b) { return a < b ? a : b; }
static inline unsigned max(unsigned a, unsigned b) { return a > b ? a : b; }
static inline long long min(long long a, long long b) { return a < b ? a : b; }
static inline long long max(long long a, long long b) { return a > b ? a : b; }
static inline unsigned long long min(unsigned long long a, unsigned long long b) { return a < b ? a : b; }
static inline unsigned long long max(unsigned long long a, unsigned long long b) { return a > b ? a : b; }

static inline unsigned __umulhi(unsigned a, unsigned b) { return (unsigned)(((unsigned long long)a * b) >> 32); }
static inline int __popc(unsigned v) { return __builtin_popcount(v); }
static inline int __ffs(unsigned v) { return __builtin_ffs((int)v); }
static inline int __clz(int v) { return v ? __builtin_clz((unsigned)v) : 32; }
template <class T> static inline T __ldg(const T* p) { return *p; }
template <class T> static inline T __ldcg(const T* p) { return *p; }
static inline void __threadfence() { simt::hb_fence(); }
static inline void __nanosleep(unsigned) { simt::yield(); }
static inline void __syncthreads() { simt::syncthreads(); }

namespace simt {
template <class T> inline unsigned long long to_bits(T v) {
  static_assert(sizeof(T) <= 8, "warp collectives move at most 64 bits");
  unsigned long long b = 0; std::memcpy(&b, &v, sizeof(T)); return b;
}
template <class T> inline T from_bits(unsigned long long b) { T v; std::memcpy(&v, &b, sizeof(T)); return v; }
inline unsigned lane_id() { return g.tid.x & 31u; }
}  // namespace simt

static inline void __syncwarp(unsigned mask = 0xFFFFFFFFu) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, 0, o, &part, true);
}
template <class T> static inline T __shfl_sync(unsigned mask, T v, int src) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, simt::to_bits(v), o, &part);
  const unsigned s = (unsigned)src & 31u;
  return (part >> s & 1u) ? simt::from_bits<T>(o[s]) : v;
}
template <class T> static inline T __shfl_up_sync(unsigned mask, T v, unsigned d) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, simt::to_bits(v), o, &part);
  const unsigned l = simt::lane_id();
  return (l >= d && (part >> (l - d) & 1u)) ? simt::from_bits<T>(o[l - d]) : v;
}
template <class T> static inline T __shfl_xor_sync(unsigned mask, T v, int d) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, simt::to_bits(v), o, &part);
  const unsigned s = (simt::lane_id() ^ (unsigned)d) & 31u;
  return (part >> s & 1u) ? simt::from_bits<T>(o[s]) : v;
}
static inline unsigned __ballot_sync(unsigned mask, bool pred) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, pred ? 1ull : 0ull, o, &part);
  unsigned r = 0;
  for (unsigned l = 0; l < 32u; ++l) if ((part >> l & 1u) && o[l]) r |= 1u << l;
  return r;
}
static inline unsigned __reduce_add_sync(unsigned mask, unsigned v) {
  unsigned long long o[32]; unsigned part; simt::warp_exchange(mask, v, o, &part);
  unsigned r = 0;
  for (unsigned l = 0; l < 32u; ++l) if (part >> l & 1u) r += (unsigned)o[l];
  return r;
}

// Atomics.  One OS thread runs every fibre and a fibre is only ever switched at a synchronisation point, so plain
// read-modify-write would do; the builtins make them atomics in the eyes of ThreadSanitizer too (relaxed, as CUDA's are).
static inline unsigned atomicAdd(unsigned* p, unsigned v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline int atomicAdd(int* p, int v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned long long atomicAdd(unsigned long long* p, unsigned long long v) { return __atomic_fetch_add(p, v, __ATOMIC_RELAXED); }
static inline unsigned atomicSub(unsigned* p, unsigned v) { return __atomic_fetch_sub(p, v, __ATOMIC_RELAXED); }
static inline int atomicSub(int* p, int v) { return __atomic_fetch_sub(p, v, __ATOMIC_RELAXED); }
static inline unsigned atomicOr(unsigned* p, unsigned v) { return __atomic_fetch_or(p, v, __ATOMIC_RELAXED); }
template <class T> static inline T simt_atomic_min(T* p, T v) {
  T o = __atomic_load_n(p, __ATOMIC_RELAXED);
  while (v < o && !__atomic_compare_exchange_n(p, &o, v, false, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
  return o;
}
static inline unsigned atomicMin(unsigned* p, unsigned v) { return simt_atomic_min(p, v); }
static inline unsigned long long atomicMin(unsigned long long* p, unsigned long long v) { return simt_atomic_min(p, v); }

// ---------------------------------------------------------------------------------------------- runtime
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorUnknown = 999 };
struct SimtStream;
typedef SimtStream* cudaStream_t;
struct SimtEvent;
typedef SimtEvent* cudaEvent_t;
struct SimtGraph;
typedef SimtGraph* cudaGraph_t;
typedef SimtGraph* cudaGraphExec_t;
enum cudaMemcpyKind { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2, cudaMemcpyDeviceToDevice = 3 };
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2, cudaStreamCaptureModeThreadLocal = 1,
       cudaDevAttrMultiProcessorCount = 16, cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };

const char* cudaGetErrorString(cudaError_t);
cudaError_t cudaGetLastError();
cudaError_t cudaGetDeviceCount(int*);
cudaError_t cudaGetDevice(int*);
cudaError_t cudaDeviceGetAttribute(int*, int, int);
cudaError_t cudaMemcpyAsync(void*, const void*, size_t, cudaMemcpyKind, cudaStream_t);
cudaError_t cudaMemcpy(void*, const void*, size_t, cudaMemcpyKind);
cudaError_t cudaMemsetAsync(void*, int, size_t, cudaStream_t);
cudaError_t cudaStreamSynchronize(cudaStream_t);
cudaError_t cudaStreamCreateWithFlags(cudaStream_t*, unsigned);
cudaError_t cudaStreamDestroy(cudaStream_t);
cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned);
cudaError_t cudaStreamBeginCapture(cudaStream_t, int);
cudaError_t cudaStreamEndCapture(cudaStream_t, cudaGraph_t*);
cudaError_t cudaGraphInstantiate(cudaGraphExec_t*, cudaGraph_t, unsigned long long);
cudaError_t cudaGraphDestroy(cudaGraph_t);
cudaError_t cudaGraphExecDestroy(cudaGraphExec_t);
cudaError_t cudaGraphLaunch(cudaGraphExec_t, cudaStream_t);
cudaError_t cudaEventCreate(cudaEvent_t*);
cudaError_t cudaEventCreateWithFlags(cudaEvent_t*, unsigned);
cudaError_t cudaEventDestroy(cudaEvent_t);
cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t);
cudaError_t cudaEventSynchronize(cudaEvent_t);
cudaError_t cudaEventElapsedTime(float*, cudaEvent_t, cudaEvent_t);
template <class F> inline cudaError_t cudaFuncSetAttribute(F, int, int) { return cudaSuccess; }
namespace simt { int blocks_per_sm(); }
template <class F> inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int* n, F, int, size_t) {
  *n = simt::blocks_per_sm(); return cudaSuccess;
}

// ---------------------------------------------------------------------------------------------- launches
// build.py rewrites `kernel<<<grid, block, smem, stream>>>(args)` into `simt::cfg(grid, block, smem, stream).call(kernel)(args)`.
namespace simt {
void run_grid(unsigned grid, unsigned block, size_t smem, std::function<void()> thread_body);   // or records it (capture)
struct cfg {
  unsigned grid, block; size_t smem; cudaStream_t stream;
  cfg(unsigned g_, unsigned b_, size_t s_, cudaStream_t st_) : grid(g_), block(b_), smem(s_), stream(st_) {}
  template <class... A> auto call(void (*kernel)(A...)) const {
    const cfg c = *this;
    return [c, kernel](A... args) {                         // arguments are copied at launch time, as on the GPU
      run_grid(c.grid, c.block, c.smem, [=]() { kernel(args...); });
    };
  }
};
}  // namespace simt
