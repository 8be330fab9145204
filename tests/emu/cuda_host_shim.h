// cuda_host_shim.h — TEST INFRASTRUCTURE (tests/emu): compiles the CUDA sources of the sampling path for the HOST so
// that their index arithmetic and memory layout can be checked on a CPU under AddressSanitizer / UBSan and compared
// with the oracle without a GPU.  Single-lane emulation: every block runs ONE thread, blocks run one after the other,
// warp collectives degenerate to the identity; every "device" allocation and every launch's dynamic shared memory is
// a heap block of exactly the requested size (shared memory: rounded up to 16 for alignment, the tail poisoned under
// ASan), so an out-of-bounds index trips the sanitizer.  Kernels are entered through a function-pointer cast to a
// by-value dummy struct (see cudaLaunchKernel below): that call is itself outside the C++ standard, so UBSan vouches
// for the kernels' arithmetic and indexing, not for the launch shim.  Only valid for kernels
// without block-wide cooperation beyond "copy the image, barrier" (lgx_decode_cut, lgx_walk_finish); the Algorithm-1
// kernels are not emulated (cooperative launches fail here).  This is NOT a CPU fallback of the product: nothing in
// the package builds, loads or links it; it checks what compute-sanitizer's memcheck would, not races.
#pragma once
#include <cstdint>
#include <cstring>
#include <cstdlib>
#include <cmath>
#include <algorithm>
#include <cstdio>
#define LGX_EMU 1
#if defined(__SANITIZE_ADDRESS__)
#include <sanitizer/asan_interface.h>
#define LGX_EMU_POISON(p, n)   do { if ((n) != 0) __asan_poison_memory_region((p), (n)); } while (0)
#define LGX_EMU_UNPOISON(p, n) do { if ((n) != 0) __asan_unpoison_memory_region((p), (n)); } while (0)
#else
#define LGX_EMU_POISON(p, n)   do { } while (0)
#define LGX_EMU_UNPOISON(p, n) do { } while (0)
#endif
#define LGX_LANES 1u
#define LGX_BLOCK_THREADS(t) 1u       /* one thread per block: shared memory sized for one candidate */
#define LGX_DYN_SMEM(name) uint8_t *name = lgx_emu::g_smem
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline __attribute__((always_inline))
#define __noinline__ inline
#define __launch_bounds__(...)
#define __grid_constant__
#define __shared__ static
#define __align__(n) alignas(n)
struct dim3 { unsigned x, y, z; dim3(unsigned a = 1, unsigned b = 1, unsigned c = 1) : x(a), y(b), z(c) {} };
struct alignas(8)  uint2 { uint32_t x, y; };
struct alignas(16) uint4 { uint32_t x, y, z, w; };
struct alignas(16) double2 { double x, y; };
static inline uint2 make_uint2(uint32_t x, uint32_t y) { return uint2{x, y}; }
static inline uint4 make_uint4(uint32_t x, uint32_t y, uint32_t z, uint32_t w) { return uint4{x, y, z, w}; }
static inline double2 make_double2(double x, double y) { return double2{x, y}; }
namespace lgx_emu {
  inline dim3 threadIdx, blockIdx, blockDim, gridDim;
  inline uint8_t *g_smem = nullptr;      // this launch's dynamic shared memory: a heap block of the launch's size
}
using lgx_emu::threadIdx; using lgx_emu::blockIdx; using lgx_emu::blockDim; using lgx_emu::gridDim;
using std::min; using std::max;
static inline uint32_t __umulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * b) >> 32); }
static inline uint32_t __vsub4(uint32_t a, uint32_t b) { uint32_t r = 0; for (int i = 0; i < 4; ++i) r |= (uint32_t)(uint8_t)((a >> (8 * i)) - (b >> (8 * i))) << (8 * i); return r; }
static inline int __popc(uint32_t v) { return __builtin_popcount(v); }
static inline int __popcll(uint64_t v) { return __builtin_popcountll(v); }
static inline int __clzll(long long v) { return v == 0 ? 64 : __builtin_clzll((unsigned long long)v); }
static inline int __ffsll(long long v) { return __builtin_ffsll(v); }
static inline double __dadd_rn(double a, double b) { volatile double r = a + b; return r; }
static inline double __dsub_rn(double a, double b) { volatile double r = a - b; return r; }
static inline double __dmul_rn(double a, double b) { volatile double r = a * b; return r; }
static inline double __ddiv_rn(double a, double b) { volatile double r = a / b; return r; }
static inline double __dsqrt_rn(double a) { return std::sqrt(a); }
static inline double __fma_rn(double a, double b, double c) { return std::fma(a, b, c); }
static inline long long __double_as_longlong(double d) { long long v; std::memcpy(&v, &d, 8); return v; }
static inline double __longlong_as_double(long long v) { double d; std::memcpy(&d, &v, 8); return d; }
static inline double __hiloint2double(int hi, int lo) { uint64_t v = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo; double d; std::memcpy(&d, &v, 8); return d; }
static inline int __double2hiint(double d) { uint64_t v; std::memcpy(&v, &d, 8); return (int)(v >> 32); }
static inline unsigned __ballot_sync(unsigned, bool p) { return p ? 1u : 0u; }
template <class T> static inline T __shfl_sync(unsigned, T v, int) { return v; }
template <class T> static inline T __shfl_down_sync(unsigned, T v, int) { return v; }
template <class T> static inline T __shfl_up_sync(unsigned, T v, int) { return v; }
template <class T> static inline T __shfl_xor_sync(unsigned, T v, int) { return v; }
static inline void __syncthreads() {}
static inline void __syncwarp() {}
static inline void __threadfence() {}
template <class T, class U> static inline T atomicAdd(T *p, U v) { T o = *p; *p = (T)(o + (T)v); return o; }
template <class T> static inline T __ldcg(const T *p) { return *p; }

// ---- runtime
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorNoDevice = 100, cudaErrorEmu = 999 };
typedef void *cudaStream_t; typedef void *cudaEvent_t; typedef void *cudaMemPool_t;
enum { cudaMemcpyHostToDevice = 1, cudaMemcpyDeviceToHost = 2 };
enum { cudaDevAttrMultiProcessorCount = 16, cudaDevAttrMaxSharedMemoryPerBlockOptin = 97, cudaDevAttrCooperativeLaunch = 95 };
enum { cudaFuncAttributeMaxDynamicSharedMemorySize = 8 };
enum { cudaMemAllocationTypePinned = 1, cudaMemHandleTypeNone = 0, cudaMemLocationTypeDevice = 1, cudaMemPoolAttrReleaseThreshold = 4 };
struct cudaMemPoolProps { int allocType, handleTypes; struct { int type, id; } location; };
static inline const char *cudaGetErrorString(cudaError_t) { return "emu"; }
static inline cudaError_t cudaGetLastError() { return cudaSuccess; }
static inline cudaError_t cudaGetDeviceCount(int *n) { *n = 1; return cudaSuccess; }
static inline cudaError_t cudaGetDevice(int *d) { *d = 0; return cudaSuccess; }
static inline cudaError_t cudaDeviceGetAttribute(int *v, int a, int) {
  if (a == cudaDevAttrMultiProcessorCount) { const char *e = getenv("LGX_EMU_SMS"); *v = e ? atoi(e) : 3; }
  else if (a == cudaDevAttrMaxSharedMemoryPerBlockOptin) *v = 227 * 1024; else *v = 1;
  return cudaSuccess; }
static inline cudaError_t cudaMalloc(void **p, size_t n) { *p = calloc(n ? n : 1, 1); return cudaSuccess; }
static inline cudaError_t cudaFree(void *p) { free(p); return cudaSuccess; }
static inline cudaError_t cudaMemcpy(void *d, const void *s, size_t n, int) { memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t n, int, cudaStream_t) { memcpy(d, s, n); return cudaSuccess; }
static inline cudaError_t cudaMemsetAsync(void *d, int v, size_t n, cudaStream_t) { memset(d, v, n); return cudaSuccess; }
static inline cudaError_t cudaMallocAsync(void **p, size_t n, cudaStream_t) { return cudaMalloc(p, n); }
static inline cudaError_t cudaMallocFromPoolAsync(void **p, size_t n, cudaMemPool_t, cudaStream_t) { return cudaMalloc(p, n); }
static inline cudaError_t cudaFreeAsync(void *p, cudaStream_t) { free(p); return cudaSuccess; }
static inline cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned) { *s = nullptr; return cudaSuccess; }
static inline cudaError_t cudaStreamDestroy(cudaStream_t) { return cudaSuccess; }
enum { cudaStreamNonBlocking = 1 };
static inline cudaError_t cudaMemPoolCreate(cudaMemPool_t *p, const cudaMemPoolProps *) { *p = (void *)1; return cudaSuccess; }
static inline cudaError_t cudaMemPoolDestroy(cudaMemPool_t) { return cudaSuccess; }
static inline cudaError_t cudaMemPoolTrimTo(cudaMemPool_t, size_t) { return cudaSuccess; }
static inline cudaError_t cudaMemPoolSetAttribute(cudaMemPool_t, int, void *) { return cudaSuccess; }
static inline cudaError_t cudaStreamSynchronize(cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaDeviceSynchronize() { return cudaSuccess; }
static inline cudaError_t cudaEventCreate(cudaEvent_t *e) { *e = nullptr; return cudaSuccess; }
static inline cudaError_t cudaEventRecord(cudaEvent_t, cudaStream_t) { return cudaSuccess; }
static inline cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t, cudaEvent_t) { *ms = 1.f; return cudaSuccess; }
static inline cudaError_t cudaEventDestroy(cudaEvent_t) { return cudaSuccess; }
static inline cudaError_t cudaFuncSetAttribute(const void *, int, int) { return cudaSuccess; }
struct cudaFuncAttributes { size_t sharedSizeBytes; };
static inline cudaError_t cudaFuncGetAttributes(cudaFuncAttributes *a, const void *) { a->sharedSizeBytes = 0; return cudaSuccess; }
template <class F> static inline cudaError_t cudaOccupancyMaxActiveBlocksPerMultiprocessor(int *n, F, int, size_t) { *n = 1; return cudaSuccess; }
// by-value kernel parameter structs travel in memory on x86-64 SysV: call through a dummy of the maximum size
// (sizeof(lgx::KParams) comes from tests/emu/emu_params.cu: only the kernels that take a KParams are emulated)
struct EmuBig { uint8_t b[4096]; };
size_t lgx_emu_param_bytes();
static inline cudaError_t cudaLaunchKernel(const void *fn, dim3 grid, dim3 block, void **args, size_t smem, cudaStream_t) {
  if (block.x != 1u) return cudaErrorEmu;                       // the host code must size launches with LGX_BLOCK_THREADS
  EmuBig big; memset(&big, 0, sizeof big); memcpy(&big, args[0], lgx_emu_param_bytes());
  lgx_emu::gridDim = grid; lgx_emu::blockDim = dim3(1); lgx_emu::threadIdx = dim3(0);
  for (unsigned b = 0; b < grid.x; ++b) {
    // exactly `smem` addressable bytes: aligned_alloc wants a multiple of the alignment, so the block is rounded up to 16
    // and, under AddressSanitizer, the 0..15 bytes behind the launch's size are poisoned (byte-exact: ASan's shadow encodes
    // "first k bytes of a granule addressable"); an index one past the last state row or sentinel cell is reported.
    // Without ASan the tail is ordinary heap slack.
    const size_t rounded = (std::max<size_t>(smem, 1) + 15) / 16 * 16;
    lgx_emu::g_smem = (uint8_t *)aligned_alloc(16, rounded);
    LGX_EMU_POISON(lgx_emu::g_smem + smem, rounded - smem);
    lgx_emu::blockIdx = dim3(b); ((void (*)(EmuBig))fn)(big);
    LGX_EMU_UNPOISON(lgx_emu::g_smem + smem, rounded - smem);
    free(lgx_emu::g_smem); lgx_emu::g_smem = nullptr;
  }
  return cudaSuccess; }
static inline cudaError_t cudaLaunchCooperativeKernel(const void *, dim3, dim3, void **, size_t, cudaStream_t) { return cudaErrorEmu; }
static inline cudaError_t cudaMemset(void *d, int v, size_t n) { memset(d, v, n); return cudaSuccess; }
