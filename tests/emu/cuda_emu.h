// cuda_emu.h -- a small CUDA execution model on the host, for tests only.
//
// TEST INFRASTRUCTURE -- NOT PART OF THE PRODUCT.  tests/emu/build_emu.py compiles the kernel sources of
// paper_2511_02742_b200/csrc with g++ and -DHOUGH_EMU against this header (only the PTX one-liners, the dynamic shared-memory
// declaration and the <<< >>> launch syntax have host spellings there); the result (tests/emu/libhough_emu.so) exports
// the same C ABI as libhough.so and is called by tests/test_emulated_kernels.py with host pointers.  It lets the kernels'
// logic (indices, list capacities, barrier placement against the data flow, the hand-over between kernels) be checked
// against the oracle on a machine without a GPU, with every shared- and global-memory access bounds-checked.  It proves
// nothing about timing, the hardware memory model or PTX semantics: the GPU parity tests (-m gpu) remain the proof.
//
// Model: one OS thread; a CTA runs as blockDim.x fibers (one per CUDA thread) that switch only at __syncthreads and at
// warp collectives (ballot / shuffle / match / syncwarp), where a lane waits until every lane named in the mask has arrived.
// CTAs of a grid run one after another (the kernels here never wait on another CTA).  The order in which runnable fibers
// are resumed is a seeded permutation (cuda_emu_configure), so that results that depend on the schedule show up as failures.
// Shared memory is one allocation per CTA whose end sits against an inaccessible page; "device" allocations likewise.
#pragma once
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <functional>

// ------------------------------------------------------------------ vector types and qualifiers
struct uint3 { unsigned x, y, z; };
struct dim3 { unsigned x, y, z; dim3(unsigned a = 1, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {} };
struct int2 { int x, y; };
struct uint2 { unsigned x, y; };
struct alignas(16) int4 { int x, y, z, w; };
struct alignas(16) uint4 { unsigned x, y, z, w; };
struct alignas(16) float4 { float x, y, z, w; };
static inline int2 make_int2(int x, int y) { return int2{x, y}; }
static inline uint2 make_uint2(unsigned x, unsigned y) { return uint2{x, y}; }
static inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }
static inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }

#define __global__
#define __device__
#define __host__
#ifdef HOUGH_EMU_TSAN  // race-detector build: device functions keep their frames, so that a suppression can name one
#define __forceinline__ inline __attribute__((noinline))
#define EMU_ATOMIC_ORDER __ATOMIC_RELAXED  // CUDA's atomics order nothing; a stronger order here would hide races from the detector
#else
#define __forceinline__ inline __attribute__((always_inline))
#define EMU_ATOMIC_ORDER __ATOMIC_SEQ_CST
#endif
#define __noinline__ __attribute__((noinline))
#define __launch_bounds__(...)
#define __align__(n) alignas(n)
#define __shared__ static thread_local /* one CTA at a time per OS thread: a function-local static is per-CTA state */

namespace cuda_emu {

struct Fiber;
extern thread_local Fiber* g_cur;           // the fiber that is running (per OS thread: one CTA at a time on each)
extern thread_local unsigned char* g_smem;  // dynamic shared memory of the running CTA
extern thread_local unsigned g_smem_bytes;
extern unsigned g_smem_window; // shared-window address of g_smem[0] (what cvta.to.shared returns for it)
extern dim3 g_block_dim, g_grid_dim;
extern long long g_violations; // failed address checks (never performed)

uint3 cur_thread_idx();
uint3 cur_block_idx();
void violation(const char* what, unsigned long long a, unsigned long long lim);

void sync_threads();
enum WarpOp { W_BALLOT, W_SHFL, W_SHFL_UP, W_SHFL_DOWN, W_SHFL_XOR, W_MATCH_ANY, W_SYNC };
unsigned long long warp_collective(WarpOp op, unsigned mask, unsigned long long val, int arg);

void launch(dim3 grid, dim3 block, size_t smem_bytes, const std::function<void()>& body);
void maybe_yield();  // a preemption point (atomics, volatile traffic) when HOUGH_EMU_PREEMPT is set

}  // namespace cuda_emu

#define threadIdx (cuda_emu::cur_thread_idx())
#define blockIdx (cuda_emu::cur_block_idx())
#define blockDim (cuda_emu::g_block_dim)
#define gridDim (cuda_emu::g_grid_dim)

// ------------------------------------------------------------------ synchronisation and warp collectives
static inline void __syncthreads() { cuda_emu::sync_threads(); }
static inline void __syncwarp(unsigned mask = 0xffffffffu) { cuda_emu::warp_collective(cuda_emu::W_SYNC, mask, 0, 0); }
static inline void __threadfence() {}
static inline unsigned __ballot_sync(unsigned mask, int pred) { return (unsigned)cuda_emu::warp_collective(cuda_emu::W_BALLOT, mask, pred ? 1 : 0, 0); }
template <typename T> static inline T emu_shfl(cuda_emu::WarpOp op, unsigned mask, T v, int arg)
{
    static_assert(sizeof(T) <= 8, "shuffle of at most 64 bits");
    unsigned long long bits = 0;
    memcpy(&bits, &v, sizeof(T));
    bits = cuda_emu::warp_collective(op, mask, bits, arg);
    T out;
    memcpy(&out, &bits, sizeof(T));
    return out;
}
template <typename T> static inline T __shfl_sync(unsigned mask, T v, int src) { return emu_shfl(cuda_emu::W_SHFL, mask, v, src); }
template <typename T> static inline T __shfl_up_sync(unsigned mask, T v, unsigned d) { return emu_shfl(cuda_emu::W_SHFL_UP, mask, v, (int)d); }
template <typename T> static inline T __shfl_down_sync(unsigned mask, T v, unsigned d) { return emu_shfl(cuda_emu::W_SHFL_DOWN, mask, v, (int)d); }
template <typename T> static inline T __shfl_xor_sync(unsigned mask, T v, int m) { return emu_shfl(cuda_emu::W_SHFL_XOR, mask, v, m); }
static inline unsigned __match_any_sync(unsigned mask, unsigned v) { return (unsigned)cuda_emu::warp_collective(cuda_emu::W_MATCH_ANY, mask, v, 0); }

// ------------------------------------------------------------------ atomics (real ones: CTAs may run on several OS threads)
template <typename T, typename U> static inline T atomicAdd(T* p, U v) { cuda_emu::maybe_yield(); return __atomic_fetch_add(p, (T)v, EMU_ATOMIC_ORDER); }
template <typename T, typename U> static inline T atomicOr(T* p, U v) { cuda_emu::maybe_yield(); return __atomic_fetch_or(p, (T)v, EMU_ATOMIC_ORDER); }
template <typename T, typename U, typename V> static inline T atomicCAS(T* p, U cmp, V val)
{
    cuda_emu::maybe_yield();
    T expected = (T)cmp;
    __atomic_compare_exchange_n(p, &expected, (T)val, false, EMU_ATOMIC_ORDER, EMU_ATOMIC_ORDER);
    return expected;  // the value that was there
}
template <typename T, typename U> static inline T atomicMax(T* p, U v)
{
    cuda_emu::maybe_yield();
    T old = __atomic_load_n(p, EMU_ATOMIC_ORDER);
    while ((T)v > old && !__atomic_compare_exchange_n(p, &old, (T)v, false, EMU_ATOMIC_ORDER, EMU_ATOMIC_ORDER)) {}
    return old;
}
template <typename T, typename U> static inline T atomicMin(T* p, U v)
{
    cuda_emu::maybe_yield();
    T old = __atomic_load_n(p, EMU_ATOMIC_ORDER);
    while ((T)v < old && !__atomic_compare_exchange_n(p, &old, (T)v, false, EMU_ATOMIC_ORDER, EMU_ATOMIC_ORDER)) {}
    return old;
}
template <typename T, typename U> static inline T atomicExch(T* p, U v) { cuda_emu::maybe_yield(); return __atomic_exchange_n(p, (T)v, EMU_ATOMIC_ORDER); }

// ------------------------------------------------------------------ memory and arithmetic intrinsics
template <typename T> static inline T __ldg(const T* p) { return *p; }
template <typename T> static inline T __ldcg(const T* p) { cuda_emu::maybe_yield(); return *p; }
template <typename T, typename U> static inline void __stcg(T* p, U v) { cuda_emu::maybe_yield(); *p = (T)v; }
static inline size_t __cvta_generic_to_shared(const void* p)
{
    const size_t off = (size_t)((const unsigned char*)p - cuda_emu::g_smem);
    if (off > cuda_emu::g_smem_bytes) cuda_emu::violation("cvta.to.shared of a pointer outside the CTA's shared memory", off, cuda_emu::g_smem_bytes);
    return off + cuda_emu::g_smem_window;
}
// pointer of a shared-window address, checked: the access of `bytes` bytes must lie inside the CTA's dynamic shared memory
static inline void* emu_shared_ptr(unsigned addr, unsigned bytes, const char* what)
{
    const unsigned off = addr - cuda_emu::g_smem_window;
    if (addr < cuda_emu::g_smem_window || (unsigned long long)off + bytes > cuda_emu::g_smem_bytes || (addr % bytes) != 0) {
        cuda_emu::violation(what, addr, cuda_emu::g_smem_bytes);
        return nullptr;
    }
    return cuda_emu::g_smem + off;
}
static inline int __float2int_rn(float x)  // cvt.rni.s32.f32: ties to even, NaN -> 0, out of range saturates
{
    if (x != x) return 0;
    if (x >= 2147483648.0f) return 2147483647;
    if (x <= -2147483648.0f) return -2147483647 - 1;
    return (int)nearbyintf(x);
}
static inline int __float_as_int(float x) { int i; memcpy(&i, &x, 4); return i; }
static inline double __dmul_rn(double a, double b) { return a * b; }  // compiled with -ffp-contract=off
static inline double __ddiv_rn(double a, double b) { return a / b; }
static inline double __dadd_rn(double a, double b) { return a + b; }
static inline int __popc(unsigned x) { return __builtin_popcount(x); }
static inline int __ffs(unsigned x) { return __builtin_ffs((int)x); }
static inline int __ffsll(long long x) { return __builtin_ffsll(x); }
static inline int __clz(unsigned x) { return x ? __builtin_clz(x) : 32; }
static inline long long clock64() { return 0; }
static inline unsigned __vmaxu2(unsigned a, unsigned b)
{
    const unsigned lo = (a & 0xffffu) > (b & 0xffffu) ? (a & 0xffffu) : (b & 0xffffu);
    const unsigned hi = (a >> 16) > (b >> 16) ? (a >> 16) : (b >> 16);
    return lo | (hi << 16);
}
static inline unsigned __vcmpgeu2(unsigned a, unsigned b)
{
    return ((a & 0xffffu) >= (b & 0xffffu) ? 0xffffu : 0u) | ((a >> 16) >= (b >> 16) ? 0xffff0000u : 0u);
}
static inline unsigned __byte_perm(unsigned a, unsigned b, unsigned sel)
{
    const unsigned long long src = ((unsigned long long)b << 32) | a;
    unsigned out = 0;
    for (int i = 0; i < 4; ++i) {
        const unsigned s = (sel >> (4 * i)) & 0xfu;
        unsigned byte = (unsigned)((src >> (8 * (s & 7u))) & 0xffu);
        if (s & 8u) byte = (byte & 0x80u) ? 0xffu : 0u;  // sign-replication mode
        out |= byte << (8 * i);
    }
    return out;
}
template <typename T> static inline T emu_min(T a, T b) { return b < a ? b : a; }
template <typename T> static inline T emu_max(T a, T b) { return a < b ? b : a; }
static inline int min(int a, int b) { return emu_min(a, b); }
static inline int max(int a, int b) { return emu_max(a, b); }
static inline unsigned min(unsigned a, unsigned b) { return emu_min(a, b); }
static inline unsigned max(unsigned a, unsigned b) { return emu_max(a, b); }
static inline long long min(long long a, long long b) { return emu_min(a, b); }
static inline long long max(long long a, long long b) { return emu_max(a, b); }
static inline unsigned long long min(unsigned long long a, unsigned long long b) { return emu_min(a, b); }
static inline unsigned long long max(unsigned long long a, unsigned long long b) { return emu_max(a, b); }
// mixed signed / unsigned calls follow CUDA's overloads: the unsigned version
static inline unsigned min(unsigned a, int b) { return emu_min(a, (unsigned)b); }
static inline unsigned min(int a, unsigned b) { return emu_min((unsigned)a, b); }
static inline unsigned max(unsigned a, int b) { return emu_max(a, (unsigned)b); }
static inline unsigned max(int a, unsigned b) { return emu_max((unsigned)a, b); }
static inline long long min(long long a, int b) { return emu_min(a, (long long)b); }
static inline long long max(long long a, int b) { return emu_max(a, (long long)b); }

// ------------------------------------------------------------------ the part of the CUDA runtime API that hough_lib.cu uses
// Everything is synchronous: streams and events are tokens.  "Device" memory is host memory whose end sits against an
// inaccessible page (an overrun faults at once).  The device properties are those of a B200.
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorInvalidValue = 1, cudaErrorMemoryAllocation = 2 };
typedef struct emu_stream_t* cudaStream_t;
typedef struct emu_event_t* cudaEvent_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost, cudaMemcpyHostToDevice, cudaMemcpyDeviceToHost, cudaMemcpyDeviceToDevice };
enum { cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize, cudaFuncAttributePreferredSharedMemoryCarveout };
enum { cudaSharedmemCarveoutMaxShared = 100 };
struct cudaDeviceProp {
    int multiProcessorCount;
    size_t sharedMemPerBlockOptin, sharedMemPerMultiprocessor, reservedSharedMemPerBlock;
    int regsPerMultiprocessor;
};
namespace cuda_emu {
void* dev_alloc(size_t bytes);
void dev_free(void* p);
}
static inline const char* cudaGetErrorString(cudaError_t e) { return e == cudaSuccess ? "no error" : (e == cudaErrorMemoryAllocation ? "out of memory" : "invalid value"); }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaGetDeviceCount(int* n) { *n = 1; return cudaSuccess; }
static inline cudaError_t cudaSetDevice(int) { return cudaSuccess; }
static inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
static inline cudaError_t cudaGetDeviceProperties(cudaDeviceProp* p, int)
{
    p->multiProcessorCount = 148;
    p->sharedMemPerBlockOptin = 227 * 1024;
    p->sharedMemPerMultiprocessor = 228 * 1024;
    p->reservedSharedMemPerBlock = 1024;
    p->regsPerMultiprocessor = 65536;
    return cudaSuccess;
}
template <typename T> static inline cudaError_t cudaMalloc(T** p, size_t bytes)
{
    *p = static_cast<T*>(cuda_emu::dev_alloc(bytes));
    return *p ? cudaSuccess : cudaErrorMemoryAllocation;
}
static inline cudaError_t cudaFree(void* p) { cuda_emu::dev_free(p); return cudaSuccess; }
static inline cudaError_t cudaMemcpy(void* d, const void* s, size_t n, cudaMemcpyKind) { if (n) memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemcpyAsync(void* d, const void* s, size_t n, cudaMemcpyKind, cudaStream_t = nullptr) { if (n) memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemset(void* d, int v, size_t n) { if (n) memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaMemsetAsync(void* d, int v, size_t n, cudaStream_t = nullptr) { if (n) memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t* s, unsigned) { *s = reinterpret_cast<cudaStream_t>(malloc(1)); return cudaSuccess; }
static inline cudaError_t cudaStreamDestroy(cudaStream_t s) { free(s); return cudaSuccess; }
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaStreamWaitEvent(cudaStream_t, cudaEvent_t, unsigned) { return cudaSuccess; }
static inline cudaError_t cudaEventCreate(cudaEvent_t* e) { *e = reinterpret_cast<cudaEvent_t>(malloc(1)); return cudaSuccess; }
static inline cudaError_t cudaEventCreateWithFlags(cudaEvent_t* e, unsigned) { return cudaEventCreate(e); }
static inline cudaError_t cudaEventDestroy(cudaEvent_t e) { free(e); return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t = nullptr) { return cudaSuccess; }
static inline cudaError_t cudaEventSynchronize(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaEventElapsedTime(float* ms, cudaEvent_t, cudaEvent_t) { *ms = 1.0f; return cudaSuccess; }
template <typename F> static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute a, int v)
{
    if (a == cudaFuncAttributeMaxDynamicSharedMemorySize && v > 227 * 1024) return cudaErrorInvalidValue;
    return cudaSuccess;
}
