// TEST INFRASTRUCTURE ONLY -- a host-side stand-in for <cuda_runtime.h> that lets g++ compile the product's
// .cu files (paper_2308_10868_b200/csrc) as plain C++ so that their kernel LOGIC (indexing, layouts, barriers,
// reductions, tie rules) can be exercised without a GPU by tests/test_emul_parity.py.  Every CUDA thread of a
// CTA runs as a cooperative fiber (ucontext); __syncthreads, warp collectives, mbarrier and TMA are emulated in
// emul.cpp.  The product library (libnrr_bm.so) never sees this header: it is on the include path only when
// tests/cuda_emul/build_emul.py builds libnrr_bm_emul.so, and nothing under the package imports or loads that.
#pragma once
#define NRR_EMUL 1

#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <functional>

// ------------------------------------------------------------------------------------------ qualifiers
#define __global__
#define __device__
#define __host__
#define __forceinline__ inline
#define __restrict__
#define __launch_bounds__(...)
#define __grid_constant__
#define __align__(n) __attribute__((aligned(n)))
#define __shared__ static
#define __constant__ static const

// ------------------------------------------------------------------------------------------ vector types
struct uint3 { unsigned int x, y, z; };
struct dim3 {
    unsigned int x, y, z;
    dim3(unsigned int a = 1, unsigned int b = 1, unsigned int c = 1) : x(a), y(b), z(c) {}
};
struct float2 { float x, y; };
struct __attribute__((aligned(16))) float4 { float x, y, z, w; };
struct __attribute__((aligned(16))) int4 { int x, y, z, w; };
struct __attribute__((aligned(16))) double2 { double x, y; };
struct __attribute__((aligned(16))) ulonglong2 { unsigned long long x, y; };
struct __attribute__((aligned(8))) uint2 { unsigned int x, y; };
struct __attribute__((aligned(16))) uint4 { unsigned int x, y, z, w; };
static inline float2 make_float2(float x, float y) { return float2{x, y}; }
static inline float4 make_float4(float x, float y, float z, float w) { return float4{x, y, z, w}; }
static inline int4 make_int4(int x, int y, int z, int w) { return int4{x, y, z, w}; }
static inline double2 make_double2(double x, double y) { return double2{x, y}; }
static inline uint2 make_uint2(unsigned x, unsigned y) { return uint2{x, y}; }
static inline uint4 make_uint4(unsigned x, unsigned y, unsigned z, unsigned w) { return uint4{x, y, z, w}; }

// ------------------------------------------------------------------------------------------ runtime API
typedef int cudaError_t;
enum { cudaSuccess = 0, cudaErrorEmul = 999 };
typedef struct emulStream_st *cudaStream_t;
struct emulEvent_st { double t_ms; };
typedef emulEvent_st *cudaEvent_t;
typedef struct emulPool_st *cudaMemPool_t;
enum cudaMemcpyKind { cudaMemcpyHostToHost, cudaMemcpyHostToDevice, cudaMemcpyDeviceToHost, cudaMemcpyDeviceToDevice };
enum cudaFuncAttribute { cudaFuncAttributeMaxDynamicSharedMemorySize = 8, cudaFuncAttributePreferredSharedMemoryCarveout = 9 };
enum { cudaSharedmemCarveoutMaxShared = 100 };
enum cudaMemPoolAttr { cudaMemPoolAttrReleaseThreshold = 4 };
enum cudaDeviceAttr { cudaDevAttrMultiProcessorCount = 16 };
enum cudaDriverEntryPointQueryResult { cudaDriverEntryPointSuccess = 0, cudaDriverEntryPointSymbolNotFound = 1 };
enum { cudaEnableDefault = 0, cudaStreamNonBlocking = 1, cudaEventDisableTiming = 2 };

cudaError_t cudaGetDevice(int *dev);
cudaError_t cudaDeviceGetAttribute(int *v, cudaDeviceAttr a, int dev);
cudaError_t cudaDeviceGetDefaultMemPool(cudaMemPool_t *pool, int dev);
cudaError_t cudaMemPoolSetAttribute(cudaMemPool_t pool, cudaMemPoolAttr a, void *v);
cudaError_t cudaMalloc(void **p, size_t bytes);
cudaError_t cudaFree(void *p);
cudaError_t cudaMallocHost(void **p, size_t bytes);
cudaError_t cudaMallocAsync(void **p, size_t bytes, cudaStream_t s);
enum { cudaMemAllocationTypePinned = 1, cudaMemHandleTypeNone = 0, cudaMemLocationTypeDevice = 1 };
struct cudaMemLocation { int type, id; };
struct cudaMemPoolProps { int allocType, handleTypes; cudaMemLocation location; };
cudaError_t cudaMemPoolCreate(cudaMemPool_t *pool, const cudaMemPoolProps *props);
cudaError_t cudaMallocFromPoolAsync(void **p, size_t bytes, cudaMemPool_t pool, cudaStream_t s);
cudaError_t cudaFreeAsync(void *p, cudaStream_t s);
cudaError_t cudaMemset(void *p, int v, size_t bytes);
cudaError_t cudaMemsetAsync(void *p, int v, size_t bytes, cudaStream_t s);
cudaError_t cudaMemcpyAsync(void *d, const void *s, size_t bytes, cudaMemcpyKind k, cudaStream_t st);
cudaError_t cudaStreamSynchronize(cudaStream_t s);
cudaError_t cudaDeviceSynchronize(void);
cudaError_t cudaStreamDestroy(cudaStream_t s);
cudaError_t cudaStreamCreateWithFlags(cudaStream_t *s, unsigned flags);
cudaError_t cudaEventCreate(cudaEvent_t *e);
cudaError_t cudaEventCreateWithFlags(cudaEvent_t *e, unsigned flags);
cudaError_t cudaStreamWaitEvent(cudaStream_t s, cudaEvent_t e, unsigned flags);
cudaError_t cudaEventDestroy(cudaEvent_t e);
cudaError_t cudaEventRecord(cudaEvent_t e, cudaStream_t s);
cudaError_t cudaEventSynchronize(cudaEvent_t e);
cudaError_t cudaEventQuery(cudaEvent_t e);
cudaError_t cudaEventElapsedTime(float *ms, cudaEvent_t a, cudaEvent_t b);
cudaError_t cudaGetLastError(void);
const char *cudaGetErrorString(cudaError_t e);
cudaError_t cudaGetDriverEntryPoint(const char *name, void **fn, unsigned long long flags, cudaDriverEntryPointQueryResult *q);
template <class F>
static inline cudaError_t cudaFuncSetAttribute(F, cudaFuncAttribute, int) { return cudaSuccess; }

// ------------------------------------------------------------------------------------------ execution model
namespace emul {
extern uint3 g_threadIdx, g_blockIdx;
extern dim3 g_blockDim, g_gridDim;
void launch(dim3 grid, dim3 block, size_t smem, const std::function<void()> &body);
unsigned char *dyn_smem();
void syncthreads();
int syncthreads_count(int pred);
void syncwarp(unsigned mask);
// all-gather of one 64-bit value per lane over the lanes of `mask`; out[l] valid for participating lanes
void warp_gather(unsigned mask, unsigned long long v, unsigned long long out[32], unsigned *present);
[[noreturn]] void trap(const char *why);
// mbarrier / TMA (keyed by the barrier's address)
void mbar_init(void *bar, unsigned count);
void mbar_arrive_expect_tx(void *bar, unsigned bytes);
bool mbar_try_wait(void *bar, unsigned parity);
void mbar_timeout();      // the kernel's bounded wait gave up (counts as progress: the thread moves on)
void tma_load_3d(void *dst, const void *map, int x, int y, int z, void *bar);
void bulk_load(void *dst, const void *src, unsigned bytes, void *bar);
}  // namespace emul

#define threadIdx ::emul::g_threadIdx
#define blockIdx ::emul::g_blockIdx
#define blockDim ::emul::g_blockDim
#define gridDim ::emul::g_gridDim

#define NRR_LAUNCH(kern, grid, block, smem, stream, ...) \
    ::emul::launch(dim3(grid), dim3(block), (size_t)(smem), [=]() { (kern)(__VA_ARGS__); })
#define NRR_DYN_SMEM(name) unsigned char *name = ::emul::dyn_smem()

static inline void __syncthreads() { emul::syncthreads(); }
static inline int __syncthreads_count(int p) { return emul::syncthreads_count(p); }
static inline void __syncwarp(unsigned mask = 0xffffffffu) { emul::syncwarp(mask); }
static inline void __threadfence() {}
static inline void __trap() { emul::trap("__trap()"); }

template <class T> static inline T __ldg(const T *p) { return *p; }
template <class T> static inline T __ldcg(const T *p) { return *p; }

static inline int emul_lane() { return (int)(threadIdx.x + blockDim.x * (threadIdx.y + blockDim.y * threadIdx.z)) & 31; }

template <class T>
static inline T __shfl_xor_sync(unsigned mask, T v, int lanemask)
{
    static_assert(sizeof(T) <= 8, "shuffle of up to 64 bits");
    unsigned long long in = 0, out[32];
    unsigned present;
    memcpy(&in, &v, sizeof(T));
    emul::warp_gather(mask, in, out, &present);
    const int src = emul_lane() ^ lanemask;
    if (src < 0 || src > 31 || !((present >> src) & 1)) return v;
    T r;
    memcpy(&r, &out[src], sizeof(T));
    return r;
}
template <class T>
static inline T __shfl_up_sync(unsigned mask, T v, unsigned delta)
{
    unsigned long long in = 0, out[32];
    unsigned present;
    memcpy(&in, &v, sizeof(T));
    emul::warp_gather(mask, in, out, &present);
    const int src = emul_lane() - (int)delta;
    if (src < 0 || !((present >> src) & 1)) return v;
    T r;
    memcpy(&r, &out[src], sizeof(T));
    return r;
}
template <class T>
static inline T __shfl_sync(unsigned mask, T v, int src_lane)
{
    static_assert(sizeof(T) <= 8, "shuffle of up to 64 bits");
    unsigned long long in = 0, out[32];
    unsigned present;
    memcpy(&in, &v, sizeof(T));
    emul::warp_gather(mask, in, out, &present);
    const int src = src_lane & 31;
    if (!((present >> src) & 1)) return v;
    T r;
    memcpy(&r, &out[src], sizeof(T));
    return r;
}
static inline unsigned __ballot_sync(unsigned mask, int pred)
{
    unsigned long long out[32];
    unsigned present, r = 0;
    emul::warp_gather(mask, pred ? 1ull : 0ull, out, &present);
    for (int l = 0; l < 32; ++l)
        if (((present >> l) & 1) && out[l]) r |= 1u << l;
    return r;
}
static inline unsigned __reduce_max_sync(unsigned mask, unsigned v)
{
    unsigned long long out[32];
    unsigned present, r = 0;
    emul::warp_gather(mask, v, out, &present);
    for (int l = 0; l < 32; ++l)
        if ((present >> l) & 1) r = std::max(r, (unsigned)out[l]);
    return r;
}
static inline int __reduce_max_sync(unsigned mask, int v)
{
    unsigned long long out[32];
    unsigned present;
    int r = INT32_MIN;
    emul::warp_gather(mask, (unsigned long long)(long long)v, out, &present);
    for (int l = 0; l < 32; ++l)
        if ((present >> l) & 1) r = std::max(r, (int)(long long)out[l]);
    return r;
}
static inline int __reduce_min_sync(unsigned mask, int v)
{
    unsigned long long out[32];
    unsigned present;
    int r = INT32_MAX;
    emul::warp_gather(mask, (unsigned long long)(long long)v, out, &present);
    for (int l = 0; l < 32; ++l)
        if ((present >> l) & 1) r = std::min(r, (int)(long long)out[l]);
    return r;
}
static inline unsigned __reduce_min_sync(unsigned mask, unsigned v)
{
    unsigned long long out[32];
    unsigned present, r = 0xffffffffu;
    emul::warp_gather(mask, v, out, &present);
    for (int l = 0; l < 32; ++l)
        if ((present >> l) & 1) r = std::min(r, (unsigned)out[l]);
    return r;
}

// atomics: fibers of one CTA run on one OS thread and CTAs run one after another, so plain operations do
template <class T> static inline T atomicAdd(T *p, T v) { T o = *p; *p = o + v; return o; }
template <class T> static inline T atomicSub(T *p, T v) { T o = *p; *p = o - v; return o; }
template <class T> static inline T atomicMax(T *p, T v) { T o = *p; if (v > o) *p = v; return o; }
template <class T> static inline T atomicMin(T *p, T v) { T o = *p; if (v < o) *p = v; return o; }
template <class T> static inline T atomicOr(T *p, T v) { T o = *p; *p = o | v; return o; }
template <class T> static inline T atomicExch(T *p, T v) { T o = *p; *p = v; return o; }

static inline int __popc(unsigned v) { return __builtin_popcount(v); }
static inline int __popcll(unsigned long long v) { return __builtin_popcountll(v); }
static inline int __clz(int v) { return v ? __builtin_clz((unsigned)v) : 32; }
static inline unsigned __float_as_uint(float f) { unsigned u; memcpy(&u, &f, 4); return u; }
static inline float __uint_as_float(unsigned u) { float f; memcpy(&f, &u, 4); return f; }
static inline float __int_as_float(int i) { float f; memcpy(&f, &i, 4); return f; }
static inline int __float_as_int(float f) { int i; memcpy(&i, &f, 4); return i; }
static inline long long __double_as_longlong(double d) { long long l; memcpy(&l, &d, 8); return l; }
static inline double __longlong_as_double(long long l) { double d; memcpy(&d, &l, 8); return d; }
// explicitly rounded double operations (the emulation is built with -ffp-contract=off)
static inline double __dadd_rn(double a, double b) { return a + b; }
static inline double __dsub_rn(double a, double b) { return a - b; }
static inline double __dmul_rn(double a, double b) { return a * b; }
static inline double __ddiv_rn(double a, double b) { return a / b; }
static inline size_t __cvta_generic_to_shared(const void *p) { return (size_t)p; }
using std::max;
using std::min;
static inline float rsqrtf(float x) { return 1.0f / sqrtf(x); }
